// Dispatch of the FAST kernel families (exact-in-mathematics rewrites of the coupling sum).
#include "oscnet_internal.cuh"

namespace oscnet {

int32_t csr_warp_stage(net* h, const StageArgs& a);
bool csr_blocked_supported(const net_desc* d);
size_t csr_blocked_scratch_bytes(const net_desc* d);
int32_t csr_blocked_prepare(net* h);
int32_t csr_blocked_stage(net* h, const StageArgs& a);
bool lattice3d_supported(const net_desc* d);
int32_t lattice3d_prepare(net* h);
int32_t lattice3d_stage(net* h, const StageArgs& a);
bool lattice_v2_supported(const net_desc* d);
size_t lattice_v2_scratch_bytes(const net_desc* d);
size_t lattice_v2_state_bytes(const net_desc* d);
int32_t lattice_v2_prepare(net* h);
int32_t lattice_v2_stage(net* h, const StageArgs& a);
int32_t lattice_v2_refresh_exchange(net* h, const void* state);
bool lattice_v3_supported(const net_desc* d);
int32_t lattice_v3_prepare(net* h);
int32_t lattice_v3_stage(net* h, const StageArgs& a);
bool ring_supported(const net_desc* d);
size_t ring_scratch_bytes(const net_desc* d);
int32_t ring_run(net* h, const void* y_in, void* y_out, int64_t n_steps, double dt, int rhs_only);

int32_t fast_select(const net_desc* d) {
    const net_topology& t = d->topo;
    if (d->model == NET_MODEL_FHN2) return FAST_NONE;                  // eq. (2) with delay: per-link kernels (delay.cu)
    if (d->batch > 1 && t.kind != NET_TOPO_RING) return FAST_NONE;   // batches of lattices / graphs: block-diagonal DIRECT form
    const bool graph = t.kind == NET_TOPO_CSR || t.kind == NET_TOPO_RANDOM_INDEGREE;
    if (d->model == NET_MODEL_HHS) return graph ? FAST_CSR_WARP : FAST_NONE;     // gate s_j gathered per link
    // KS with inertia: the persistent ring kernel (same fields as KS), the field-split lattice kernels,
    // warp-per-row gathers on graphs (psi is a local variable); DIRECT elsewhere
    if (d->model == NET_MODEL_KSI)
        return ring_supported(d) ? FAST_RING_KS : lattice_v3_supported(d) ? FAST_LATTICE3D_V3 : graph ? FAST_CSR_WARP : FAST_NONE;
    if (t.kind == NET_TOPO_CSR || t.kind == NET_TOPO_RANDOM_INDEGREE)
        return csr_blocked_supported(d) ? FAST_CSR_BLOCKED : FAST_CSR_WARP;
    if (lattice_v3_supported(d)) return FAST_LATTICE3D_V3;
    if (lattice_v2_supported(d)) return FAST_LATTICE3D_V2;
    if (lattice3d_supported(d)) return FAST_LATTICE3D;
    if (ring_supported(d)) return d->model == NET_MODEL_KS ? FAST_RING_KS : FAST_RING_FHN;
    return FAST_NONE;
}

size_t fast_scratch_bytes(const net_desc* d, int32_t fast_kind) {
    if (fast_kind == FAST_RING_KS || fast_kind == FAST_RING_FHN) return ring_scratch_bytes(d);
    if (fast_kind == FAST_LATTICE3D_V2 || fast_kind == FAST_LATTICE3D_V3) return lattice_v2_scratch_bytes(d);
    if (fast_kind == FAST_CSR_BLOCKED) return csr_blocked_scratch_bytes(d);
    return 0;
}

size_t fast_state_bytes(const net_desc* d, int32_t fast_kind) {
    return fast_kind == FAST_LATTICE3D_V2 || fast_kind == FAST_LATTICE3D_V3 ? lattice_v2_state_bytes(d) : 0;
}

// Launch geometry, shared-memory opt-in and occupancy of the selected family.  A family that
// cannot take this shape (NET_ERR_UNSUPPORTED) falls back to DIRECT unless FAST was demanded.
int32_t fast_prepare(net* h) {
    int32_t rc = NET_OK;
    if (h->fast_kind == FAST_CSR_BLOCKED) {
        rc = csr_blocked_prepare(h);
        if (rc == NET_ERR_UNSUPPORTED) {     // a segment the 16-bit offsets cannot take: warp-per-row gathers
            h->fast_kind = FAST_CSR_WARP;
            rc = NET_OK;
        }
    }
    if (h->fast_kind == FAST_LATTICE3D_V3) {
        rc = lattice_v3_prepare(h);
        if (rc == NET_ERR_UNSUPPORTED && h->desc.model != NET_MODEL_KSI) {     // same layout, second-generation kernels
            h->fast_kind = FAST_LATTICE3D_V2;
            rc = NET_OK;
        }
    }
    if (h->fast_kind == FAST_LATTICE3D_V2) {
        rc = lattice_v2_prepare(h);
        if (rc == NET_ERR_UNSUPPORTED) {     // shape the bulk-copy kernels cannot take: first generation
            h->fast_kind = FAST_LATTICE3D;
            rc = NET_OK;
        }
    }
    if (h->fast_kind == FAST_LATTICE3D) rc = lattice3d_prepare(h);
    if (rc == NET_ERR_UNSUPPORTED && h->desc.method != NET_METHOD_FAST) {
        h->fast_kind = FAST_NONE;
        h->method = NET_METHOD_DIRECT;
        rc = NET_OK;
    } else if (rc == NET_ERR_UNSUPPORTED) {
        set_err(h, rc, "the FAST kernel family does not support this shape");
    }
    return rc;
}

int32_t fast_stage(net* h, const StageArgs& a) {
    switch (h->fast_kind) {
        case FAST_CSR_WARP: return csr_warp_stage(h, a);
        case FAST_CSR_BLOCKED: return csr_blocked_stage(h, a);
        case FAST_LATTICE3D: return lattice3d_stage(h, a);
        case FAST_LATTICE3D_V2: return lattice_v2_stage(h, a);
        case FAST_LATTICE3D_V3: return lattice_v3_stage(h, a);
        case FAST_RING_KS:
        case FAST_RING_FHN:
            // the ring family integrates whole runs (fast_integrate); as a stage it only serves
            // the RHS hook
            if (a.stage != STAGE_RHS_ONLY) break;
            return ring_run(h, a.in, a.out, 0, 0.0, 1);
        default: break;
    }
    return set_err(h, NET_ERR_UNSUPPORTED, "fast kernel family %d has no stage kernel", h->fast_kind);
}

int32_t fast_refresh_exchange(net* h, const void* state) {
    if (h->fast_kind == FAST_LATTICE3D_V2 || h->fast_kind == FAST_LATTICE3D_V3) return lattice_v2_refresh_exchange(h, state);
    return NET_OK;
}

int32_t fast_integrate(net* h, int64_t n_steps, double dt, bool* handled) {
    *handled = false;
    if (h->fast_kind != FAST_RING_KS && h->fast_kind != FAST_RING_FHN) return NET_OK;
    // one persistent launch per <= 2^20 steps (the grid-barrier counter is 32 bits wide)
    for (int64_t left = n_steps; left > 0;) {
        const int64_t now = left < (1 << 20) ? left : (1 << 20);
        int32_t rc = ring_run(h, h->b.y, h->b.y, now, dt, 0);
        if (rc) return rc;
        left -= now;
    }
    *handled = true;
    return NET_OK;
}

}  // namespace oscnet
