// f32 ks instantiations of the third-generation 3D lattice kernels (lat3_kernel.cuh).
#include "lat3_host.cuh"

namespace oscnet {
int32_t lattice_v3_entry_f32_ks(net* h, int stage, double dt, void* rhs_out) {
    return l3_entry<float, NET_MODEL_KS>(h, stage, dt, rhs_out);
}
}  // namespace oscnet
