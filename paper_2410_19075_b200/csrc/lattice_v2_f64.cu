// f64 instantiations of the second-generation 3D lattice kernels (lattice_v2.cuh).
#include "lattice_v2_host.cuh"

namespace oscnet {
int32_t lattice_v2_entry_f64(net* h, const Lat2Args* a, int nops, int which_map) {
    return l2_entry<double>(h, a, nops, which_map);
}
}  // namespace oscnet
