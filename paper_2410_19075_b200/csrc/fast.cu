// Dispatch of the FAST kernel families (exact-in-mathematics rewrites of the coupling sum).
#include "oscnet_internal.cuh"

namespace oscnet {

int32_t csr_warp_stage(net* h, const StageArgs& a);

int32_t fast_select(const net_desc* d) {
    const net_topology& t = d->topo;
    if (t.kind == NET_TOPO_CSR || t.kind == NET_TOPO_RANDOM_INDEGREE) return FAST_CSR_WARP;
    return FAST_NONE;
}

size_t fast_scratch_bytes(const net_desc* d, int32_t fast_kind) {
    (void)d; (void)fast_kind;
    return 0;
}

int32_t fast_stage(net* h, const StageArgs& a) {
    switch (h->fast_kind) {
        case FAST_CSR_WARP: return csr_warp_stage(h, a);
        default: return set_err(h, NET_ERR_UNSUPPORTED, "fast kernel family %d has no stage kernel", h->fast_kind);
    }
}

int32_t fast_integrate(net* h, int64_t n_steps, double dt, bool* handled) {
    (void)h; (void)n_steps; (void)dt;
    *handled = false;
    return NET_OK;
}

}  // namespace oscnet
