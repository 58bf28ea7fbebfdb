// f32 ks instantiations, radius 6, of the field-split 3D lattice kernel (lat3s_kernel.cuh).
#include "lat3_host.cuh"

namespace oscnet {
int32_t lattice_v3_entry_f32_ks6(net* h, int stage, double dt, void* rhs_out) {
    return l3_entry_p<float, NET_MODEL_KS, 6>(h, stage, dt, rhs_out);
}
}  // namespace oscnet
