// C ABI of liboscnet.so (include/oscnet.h): validation, workspace layout, state I/O,
// the CUDA-graph step driver and the observable entry points.
#include <math.h>
#include <stdarg.h>
#include <stdlib.h>

#include <new>

#include "oscnet_internal.cuh"

namespace oscnet {

static thread_local char g_err[512] = "";

int32_t set_err(net* h, int32_t code, const char* fmt, ...) {
    char* dst = h ? h->err : g_err;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 512, fmt, ap);
    va_end(ap);
    return code;
}

int32_t cuda_err(net* h, cudaError_t e, const char* what) {
    return set_err(h, NET_ERR_CUDA, "CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
}

static int model_nvar(int model) {
    return model == NET_MODEL_KS ? 1 : model == NET_MODEL_FHN ? 2 : model == NET_MODEL_HH ? 4 : model == NET_MODEL_KSI ? 2 :
           model == NET_MODEL_FHN2 ? 2 : model == NET_MODEL_HHS ? 5 : -1;
}

static int32_t validate(net* h, const net_desc* d) {
    if (!d) return set_err(h, NET_ERR_INVALID, "desc is NULL");
    if (model_nvar(d->model) < 0) return set_err(h, NET_ERR_INVALID, "unknown model %d", d->model);
    if (d->dtype != NET_F32 && d->dtype != NET_F64) return set_err(h, NET_ERR_INVALID, "unknown dtype %d", d->dtype);
    if (d->n < 1 || d->n > 2147483647LL) return set_err(h, NET_ERR_INVALID, "n = %lld outside [1, 2^31-1] (col_idx is int32)", (long long)d->n);
    if (d->batch < 1) return set_err(h, NET_ERR_INVALID, "batch = %d < 1", d->batch);
    if (d->batch > 1 && d->topo.kind == NET_TOPO_COMPRESSED)
        return set_err(h, NET_ERR_UNSUPPORTED, "batch = %d: compressed matrices are not batched in this build", d->batch);
    if (d->n * (int64_t)d->batch > 2147483647LL) return set_err(h, NET_ERR_INVALID, "n * batch exceeds 2^31-1");
    if (d->method < NET_METHOD_AUTO || d->method > NET_METHOD_FAST) return set_err(h, NET_ERR_INVALID, "unknown method %d", d->method);
    if (d->delay_steps < 0 || d->delay_steps > (1 << 20) || (d->delay_steps > 0 && d->model != NET_MODEL_FHN2))
        return set_err(h, NET_ERR_INVALID, "delay_steps = %d: need 0 <= delay_steps <= 2^20, and only NET_MODEL_FHN2 has a delay", d->delay_steps);
    const net_topology& t = d->topo;
    switch (t.kind) {
        case NET_TOPO_RING:
            if (t.radius < 0 || 2 * (int64_t)t.radius >= d->n)
                return set_err(h, NET_ERR_INVALID, "ring: need 0 <= 2*radius < n (radius %d, n %lld)", t.radius, (long long)d->n);
            break;
        case NET_TOPO_LATTICE: {
            if (t.ndim < 1 || t.ndim > 3) return set_err(h, NET_ERR_INVALID, "lattice: ndim %d outside 1..3", t.ndim);
            int64_t prod = 1;
            for (int q = 0; q < t.ndim; ++q) {
                if (t.extent[q] < 1 || t.extent[q] > 2147483647LL) return set_err(h, NET_ERR_INVALID, "lattice: bad extent[%d]", q);
                if (t.radius < 0 || 2 * (int64_t)t.radius >= t.extent[q])
                    return set_err(h, NET_ERR_INVALID, "lattice: need 2*radius < extent (radius %d, extent[%d] %lld)", t.radius, q, (long long)t.extent[q]);
                prod *= t.extent[q];
            }
            if (prod != d->n) return set_err(h, NET_ERR_INVALID, "lattice: product of extents %lld != n %lld", (long long)prod, (long long)d->n);
            if (t.radius > 64) return set_err(h, NET_ERR_UNSUPPORTED, "lattice: radius %d > 64", t.radius);
            break;
        }
        case NET_TOPO_CSR:
            if (!t.row_ptr || (t.nnz > 0 && !t.col_idx)) return set_err(h, NET_ERR_INVALID, "csr: row_ptr / col_idx is NULL");
            if (t.nnz < 0) return set_err(h, NET_ERR_INVALID, "csr: nnz < 0");
            break;
        case NET_TOPO_RANDOM_INDEGREE:
            if (d->n < 2 || t.in_degree < 0 || (int64_t)t.in_degree > d->n - 1)
                return set_err(h, NET_ERR_INVALID, "random graph: need n >= 2 and 0 <= in_degree <= n-1");
            break;
        case NET_TOPO_COMPRESSED: {
            const net_compressed* c = t.compressed;
            if (!c || !c->c || !c->d_ptr || (c->v_len > 0 && !c->v_pos)) return set_err(h, NET_ERR_INVALID, "compressed matrix: NULL struct or arrays");
            if (c->n != d->n) return set_err(h, NET_ERR_INVALID, "compressed matrix: n %lld != desc n %lld", (long long)c->n, (long long)d->n);
            if (c->k < 1 || c->v_len < 0 || c->v_len > d->n || c->d_ptr[0] != 0 || c->d_ptr[c->k] < 0)
                return set_err(h, NET_ERR_INVALID, "compressed matrix: bad table sizes");
            break;
        }
        default: return set_err(h, NET_ERR_INVALID, "unknown topology kind %d", t.kind);
    }
    return NET_OK;
}

// Inside the library a batch of B independent rings of N elements ("a large number
// of network instances simultaneously") is ONE net of B*N elements whose coupling
// matrix is block diagonal: desc.n becomes the total, the ring period is desc.n / desc.batch, and
// the state layout SoA [nvar][batch][N] is the SoA [nvar][B*N] every kernel already uses.
static int32_t normalise(const net_desc* in, net_desc* out) {
    int32_t rc = validate(nullptr, in);
    if (rc) return rc;
    *out = *in;
    out->n = in->n * (int64_t)in->batch;
    return NET_OK;
}

// Workspace layout.  Every region is 256-byte aligned.  `base` may be null (size query).
struct Layout {
    size_t total, state_bytes;
    Buffers b;
};

static size_t take(size_t& cur, size_t bytes) {
    size_t at = cur;
    cur += (bytes + 255) / 256 * 256;
    return at;
}

static Layout make_layout(const net_desc* d, char* base) {
    Layout L;
    memset(&L, 0, sizeof(L));
    const size_t es = d->dtype == NET_F32 ? 4 : 8;
    const int nv = model_nvar(d->model);
    const int64_t ld = round_up(d->n, 64);
    size_t cur = 0;
    auto P = [&](size_t bytes) -> void* { size_t at = take(cur, bytes); return base ? (void*)(base + at) : (void*)(uintptr_t)(at + 256); };
    const int fk = d->method == NET_METHOD_DIRECT ? FAST_NONE : fast_select(d);
    size_t state = (size_t)nv * ld * es;
    if (fast_state_bytes(d, fk) > state) state = fast_state_bytes(d, fk);
    L.state_bytes = state;
    L.b.y = P(state); L.b.Y2 = P(state); L.b.Y3 = P(state); L.b.Y4 = P(state);
    L.b.elem_param = P((size_t)ld * es);
    if (d->model == NET_MODEL_FHN2) {
        L.b.hist_x = P((size_t)(d->delay_steps + 2) * ld * es);
        L.b.hist_d = P((size_t)(d->delay_steps + 2) * ld * es);
    }
    if (d->model == NET_MODEL_HH && (fk == FAST_CSR_WARP || fk == FAST_CSR_BLOCKED)) {
        L.b.s_y = P((size_t)ld * es); L.b.s_Y2 = P((size_t)ld * es);
        L.b.s_Y3 = P((size_t)ld * es); L.b.s_Y4 = P((size_t)ld * es);
    }
    const net_topology& t = d->topo;
    if (t.kind == NET_TOPO_LATTICE)
        L.b.off = (int32_t*)P(sizeof(int32_t) * 3 * (size_t)(topo_lattice_noff(t.ndim, t.radius, 1) + 1));
    if (t.kind == NET_TOPO_CSR || t.kind == NET_TOPO_RANDOM_INDEGREE) {
        size_t nnz = t.kind == NET_TOPO_CSR ? (size_t)t.nnz : (size_t)d->n * (size_t)t.in_degree;
        L.b.row_ptr = (int64_t*)P(sizeof(int64_t) * (size_t)(d->n + 1));
        L.b.col_idx = (int32_t*)P(sizeof(int32_t) * (nnz + 1));
    }
    if (t.kind == NET_TOPO_COMPRESSED) {
        const net_compressed* c = t.compressed;
        L.b.cmp_v = (int32_t*)P(sizeof(int32_t) * (size_t)(c->v_len + 1));
        L.b.cmp_dptr = (int64_t*)P(sizeof(int64_t) * (size_t)(c->k + 1));
        L.b.cmp_dpos = (int32_t*)P(sizeof(int32_t) * (size_t)(c->d_ptr[c->k] + 1));
        L.b.cmp_c = (int32_t*)P(sizeof(int32_t) * (size_t)d->n);
        L.b.cmp_deg = (int32_t*)P(sizeof(int32_t) * (size_t)c->k);
    }
    L.b.flag = (int32_t*)P(64);
    L.b.obs_theta_prev = (double*)P(sizeof(double) * d->n);
    L.b.obs_wind = (double*)P(sizeof(double) * d->n);
    L.b.obs_ref = (double*)P(sizeof(double) * d->n);
    L.b.obs_vel = (double*)P(sizeof(double) * d->n);
    L.b.obs_tmp = (double*)P(sizeof(double) * 2 * d->n);
    L.b.obs_loc = (double*)P(sizeof(double) * d->n);
    L.b.obs_partial = (double*)P(sizeof(double) * 4096);
    L.b.obs_acc = (double*)P(sizeof(double) * 16);
    L.b.scratch_bytes = fast_scratch_bytes(d, fk);
    size_t staging = 8u << 20;  // host<->device staging for net_get_topology
    if (L.b.scratch_bytes < staging) L.b.scratch_bytes = staging;
    L.b.scratch = P(L.b.scratch_bytes);
    L.total = cur;
    return L;
}

static void fill_params(net* h, const void* params) {
    ModelParams& mp = h->mp;
    memset(&mp, 0, sizeof(mp));
    if (h->desc.model == NET_MODEL_KS) {
        const net_ks_params* p = (const net_ks_params*)params;
        mp.K = p->K; mp.alpha = p->alpha; mp.sin_a = sin(p->alpha); mp.cos_a = cos(p->alpha);
    } else if (h->desc.model == NET_MODEL_KSI) {
        const net_ksi_params* p = (const net_ksi_params*)params;
        mp.K = p->K; mp.alpha = p->alpha; mp.sin_a = sin(p->alpha); mp.cos_a = cos(p->alpha);
        mp.inv_m = 1.0 / p->m; mp.damp = p->eps;
    } else if (h->desc.model == NET_MODEL_FHN2) {
        const net_fhn2_params* p = (const net_fhn2_params*)params;
        mp.inv_eps = 1.0 / p->eps; mp.a = p->a; mp.sigma = p->sigma; mp.I_app = p->I_app;
        mp.noise_D = p->D; mp.noise_seed = p->seed;
    } else if (h->desc.model == NET_MODEL_FHN) {
        const net_fhn_params* p = (const net_fhn_params*)params;
        mp.inv_eps = 1.0 / p->eps; mp.a = p->a; mp.sigma = p->sigma;
        mp.buu = cos(p->phi); mp.buv = sin(p->phi); mp.bvu = -sin(p->phi); mp.bvv = cos(p->phi);
    } else {
        const net_hh_params* p = (const net_hh_params*)params;     // HHS: the same struct comes first
        if (h->desc.model == NET_MODEL_HHS) { mp.a_s = ((const net_hhs_params*)params)->a_s; mp.b_s = ((const net_hhs_params*)params)->b_s; }
        mp.gNa = p->gNa; mp.gK = p->gK; mp.gL = p->gL; mp.ENa = p->ENa; mp.EK = p->EK; mp.EL = p->EL;
        mp.inv_C = 1.0 / p->C; mp.g_syn = p->g_syn; mp.E_syn = p->E_syn; mp.theta_syn = p->theta_syn;
        mp.inv_k_syn = 1.0 / p->k_syn; mp.V_c = p->V_c; mp.n_c = p->n_c; mp.inv_V_s = 1.0 / p->V_s;
    }
}

template <class T>
__global__ void fill_kernel(T* p, int64_t n, T v) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x)
        p[i] = v;
}

static int32_t fill_elem_param(net* h, double v) {
    unsigned g = (unsigned)((h->ld + 255) / 256 > 2368 ? 2368 : (h->ld + 255) / 256);
    if (h->desc.dtype == NET_F32) fill_kernel<float><<<g, 256, 0, h->stream>>>((float*)h->b.elem_param, h->ld, (float)v);
    else fill_kernel<double><<<g, 256, 0, h->stream>>>((double*)h->b.elem_param, h->ld, v);
    h->launches += 1;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

// state copy between caller layout [nvar][n] and internal [nvar][ld]
static int32_t copy_state(net* h, void* internal, void* external, bool to_internal, bool ext_is_device) {
    cudaMemcpyKind kind = ext_is_device ? cudaMemcpyDeviceToDevice
                                        : (to_internal ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToHost);
    size_t row = (size_t)h->n * h->esize;
    if (h->pairs) {
        // interleaved internal layout: go through Y3 (dead between steps) as SoA staging
        void* soa = h->b.Y3;
        int32_t rc;
        if (to_internal) {
            OSC_CUDA(h, cudaMemcpy2DAsync(soa, (size_t)h->ld * h->esize, external, row, row, h->nvar, kind, h->stream));
            if ((rc = pairs_pack(h, soa, internal))) return rc;
        } else {
            if ((rc = pairs_unpack(h, internal, soa))) return rc;
            OSC_CUDA(h, cudaMemcpy2DAsync(external, row, soa, (size_t)h->ld * h->esize, row, h->nvar, kind, h->stream));
        }
        if (!ext_is_device) OSC_CUDA(h, cudaStreamSynchronize(h->stream));
        return NET_OK;
    }
    if (to_internal)
        OSC_CUDA(h, cudaMemcpy2DAsync(internal, (size_t)h->ld * h->esize, external, row, row, h->nvar, kind, h->stream));
    else
        OSC_CUDA(h, cudaMemcpy2DAsync(external, row, internal, (size_t)h->ld * h->esize, row, h->nvar, kind, h->stream));
    if (!ext_is_device) OSC_CUDA(h, cudaStreamSynchronize(h->stream));
    return NET_OK;
}

static void drop_graph(net* h) {
    if (h->graph_exec) { cudaGraphExecDestroy(h->graph_exec); h->graph_exec = nullptr; }
    if (h->graph) { cudaGraphDestroy(h->graph); h->graph = nullptr; }
    h->graph_steps = 0;
}

static int32_t run_stage(net* h, const StageArgs& a) {
    if (h->desc.model == NET_MODEL_FHN2) return delay_stage(h, a);
    if (h->method == NET_METHOD_FAST) return fast_stage(h, a);
    return direct_stage(h, a);
}

static StageArgs stage_args(net* h, int stage, double dt) {
    StageArgs a;
    memset(&a, 0, sizeof(a));
    const Buffers& b = h->b;
    a.y = b.y; a.Y2 = b.Y2; a.Y3 = b.Y3; a.elem_param = b.elem_param;
    a.n = h->n; a.ld = h->ld; a.dt = dt; a.stage = stage;
    switch (stage) {
        case 0: a.in = b.y; a.out = b.Y2; a.s_in = b.s_y; a.s_out = b.s_Y2; break;
        case 1: a.in = b.Y2; a.out = b.Y3; a.s_in = b.s_Y2; a.s_out = b.s_Y3; break;
        case 2: a.in = b.Y3; a.out = b.Y4; a.s_in = b.s_Y3; a.s_out = b.s_Y4; break;
        default: a.in = b.Y4; a.out = b.y; a.s_in = b.s_Y4; a.s_out = b.s_y; break;
    }
    return a;
}

// exchange fields derived from y (HH: S(V); KS on the bulk-copy lattice kernels: (cos, sin) phi)
static int32_t ensure_s(net* h) {
    if (h->s_valid) return NET_OK;
    int32_t rc = NET_OK;
    if (h->b.s_y) rc = hh_compute_s(h, h->b.y, h->b.s_y);
    if (rc == NET_OK) rc = fast_refresh_exchange(h, nullptr);
    if (rc) return rc;
    h->s_valid = 1;
    return NET_OK;
}

static int32_t enqueue_step(net* h, double dt) {
    for (int s = 0; s < 4; ++s) {
        int32_t rc = run_stage(h, stage_args(h, s, dt));
        if (rc) return rc;
    }
    h->hist_step += 1;      // NET_MODEL_FHN2: slot of the history ring, counter of the noise stream
    return NET_OK;
}

// Helpers of the adaptive integrator (adaptive.cu): vectors in the caller's layout [nvar][n] on the device.
int32_t state_to_external(net* h, void* d_dst) { return copy_state(h, h->b.y, d_dst, false, true); }
int32_t state_from_external(net* h, const void* d_src) {
    h->s_valid = 0;
    return copy_state(h, h->b.y, const_cast<void*>(d_src), true, true);
}
// k = f(x): x becomes the net's state (the caller restores its own afterwards), then the RHS-only
// instance of the net's stage kernel family, exactly as net_eval_rhs runs it
int32_t rhs_at(net* h, const void* d_x, void* d_k) {
    int32_t rc;
    // same layout inside and outside (no padding between the variables, no interleaved pairs): the
    // stage kernels read x and write k in place, only the exchange fields of x are rebuilt
    if (!h->pairs && h->n == h->ld && h->desc.model != NET_MODEL_FHN2 && !getenv("OSCNET_DP5_COPIES")) {
        h->s_valid = 0;                                   // the exchange fields no longer belong to y
        if (h->b.s_y && (rc = hh_compute_s(h, d_x, h->b.s_y))) return rc;
        if (h->method == NET_METHOD_FAST && (rc = fast_refresh_exchange(h, d_x))) return rc;
        StageArgs a = stage_args(h, 0, 0.0);
        a.stage = STAGE_RHS_ONLY;
        a.in = d_x;
        a.out = d_k;
        a.s_out = nullptr;
        return run_stage(h, a);
    }
    rc = state_from_external(h, d_x);
    if (rc) return rc;
    if ((rc = ensure_s(h))) return rc;
    StageArgs a = stage_args(h, 0, 0.0);
    a.stage = STAGE_RHS_ONLY;
    a.out = h->b.Y4;
    a.s_out = nullptr;
    if ((rc = run_stage(h, a))) return rc;
    return copy_state(h, h->b.Y4, d_k, false, true);
}

constexpr int GRAPH_STEPS = 8;

static int32_t integrate_plain(net* h, int64_t n_steps, double dt) {
    int32_t rc = ensure_s(h);
    if (rc) return rc;
    bool handled = false;
    rc = fast_integrate(h, n_steps, dt, &handled);
    if (rc) return rc;
    if (!handled) {
        int64_t left = n_steps;
        // the legacy default stream cannot be captured: plain launches there
        // (FHN2: the history slots and the noise counter change from step to step -- plain launches)
        const bool can_capture = h->stream != nullptr && h->stream != cudaStreamLegacy && h->desc.model != NET_MODEL_FHN2;
        if (left >= GRAPH_STEPS && can_capture) {
            if (!h->graph_exec || h->graph_dt != dt) {
                drop_graph(h);
                int64_t before = h->launches;
                OSC_CUDA(h, cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal));
                for (int q = 0; q < GRAPH_STEPS && rc == NET_OK; ++q) rc = enqueue_step(h, dt);
                cudaError_t e = cudaStreamEndCapture(h->stream, &h->graph);
                h->graph_kernels = h->launches - before;  // kernel nodes per replay
                h->launches = before;                     // capture itself launched nothing
                if (rc) { drop_graph(h); return rc; }
                if (e != cudaSuccess) return cuda_err(h, e, "cudaStreamEndCapture");
                OSC_CUDA(h, cudaGraphInstantiate(&h->graph_exec, h->graph, 0));
                h->graph_dt = dt;
                h->graph_steps = GRAPH_STEPS;
            }
            while (left >= GRAPH_STEPS) {
                OSC_CUDA(h, cudaGraphLaunch(h->graph_exec, h->stream));
                h->launches += h->graph_kernels;
                left -= GRAPH_STEPS;
            }
        }
        for (; left > 0; --left)
            if ((rc = enqueue_step(h, dt))) return rc;
    }
    h->step += n_steps;
    h->t += (double)n_steps * dt;
    return NET_OK;
}

// Every entry point runs on the device that owns the workspace, whatever device is current in
// the calling thread (the previous device is restored on return).
struct DevGuard {
    int prev = -1, dev = -1;
    explicit DevGuard(const net* h) {
        if (!h) return;
        dev = h->device;
        if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; return; }
        if (prev != dev) cudaSetDevice(dev); else prev = -1;
    }
    ~DevGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

}  // namespace oscnet

using namespace oscnet;

#pragma GCC visibility push(default)
extern "C" {

const char* net_version(void) { return "oscnet 0.1 sm_100a"; }

int32_t net_probe_latency(net_t* h, double* out4) {
    DevGuard guard_(h);
    if (!h || !out4) return set_err(h, NET_ERR_INVALID, "net or out4 is NULL");
    return ring_probe_latency(h, out4);
}

int32_t net_probe_peaks(net_t* h, double* out8) {
    DevGuard guard_(h);
    if (!h || !out8) return set_err(h, NET_ERR_INVALID, "net or out8 is NULL");
    return probe_peaks(h, out8);
}

const char* net_last_error(const net_t* h) { return h ? h->err : g_err; }

int32_t net_workspace_bytes(const net_desc* desc, size_t* bytes) {
    if (!bytes) return set_err(nullptr, NET_ERR_INVALID, "bytes is NULL");
    net_desc nd;
    int32_t rc = normalise(desc, &nd);
    if (rc) return rc;
    *bytes = make_layout(&nd, nullptr).total;
    return NET_OK;
}

int32_t net_create(const net_desc* user_desc, const void* params, size_t params_bytes, void* d_workspace,
                   size_t workspace_bytes, void* cuda_stream, net_t** out) {
    if (!out) return set_err(nullptr, NET_ERR_INVALID, "out is NULL");
    *out = nullptr;
    net_desc nd;
    int32_t rc = normalise(user_desc, &nd);
    if (rc) return rc;
    const net_desc* desc = &nd;                 // n = total elements of the batch from here on
    size_t want = desc->model == NET_MODEL_KS ? sizeof(net_ks_params)
                : desc->model == NET_MODEL_KSI ? sizeof(net_ksi_params)
                : desc->model == NET_MODEL_FHN ? sizeof(net_fhn_params)
                : desc->model == NET_MODEL_FHN2 ? sizeof(net_fhn2_params)
                : desc->model == NET_MODEL_HHS ? sizeof(net_hhs_params) : sizeof(net_hh_params);
    if (desc->model == NET_MODEL_KSI && params && params_bytes == want && !(((const net_ksi_params*)params)->m > 0.0))
        return set_err(nullptr, NET_ERR_INVALID, "KS with inertia: need m > 0");
    if (!params || params_bytes != want)
        return set_err(nullptr, NET_ERR_INVALID, "params is NULL or params_bytes %zu != %zu", params_bytes, want);
    if (!d_workspace) return set_err(nullptr, NET_ERR_INVALID, "d_workspace is NULL");
    if (((uintptr_t)d_workspace & 255) != 0) return set_err(nullptr, NET_ERR_SIZE, "d_workspace is not 256-byte aligned");
    Layout L = make_layout(desc, (char*)d_workspace);
    if (workspace_bytes < L.total)
        return set_err(nullptr, NET_ERR_SIZE, "workspace %zu bytes < required %zu", workspace_bytes, L.total);
    cudaPointerAttributes pattr;
    if (cudaPointerGetAttributes(&pattr, d_workspace) != cudaSuccess || pattr.type != cudaMemoryTypeDevice) {
        cudaGetLastError();
        return set_err(nullptr, NET_ERR_INVALID, "d_workspace is not device memory");
    }
    net* h = new (std::nothrow) net;
    if (!h) return set_err(nullptr, NET_ERR_INVALID, "out of host memory");
    memset(h, 0, sizeof(*h));
    h->device = pattr.device;
    DevGuard guard_(h);
    h->desc = *desc;
    h->desc.topo.row_ptr = nullptr;  // the caller's arrays are not kept
    h->desc.topo.col_idx = nullptr;
    h->desc.topo.compressed = nullptr;
    h->nvar = model_nvar(desc->model);
    h->esize = desc->dtype == NET_F32 ? 4 : 8;
    h->n = desc->n;
    h->ld = round_up(desc->n, 64);
    h->stream = (cudaStream_t)cuda_stream;
    h->b = L.b;
    h->state_bytes = L.state_bytes;
    fill_params(h, params);
    const int fk = desc->method == NET_METHOD_DIRECT ? FAST_NONE : fast_select(desc);
    if (desc->method == NET_METHOD_FAST && fk == FAST_NONE) {
        set_err(nullptr, NET_ERR_UNSUPPORTED, "no FAST kernel for this model/topology/shape");
        delete h;
        return NET_ERR_UNSUPPORTED;
    }
    h->fast_kind = fk;
    h->method = fk == FAST_NONE ? NET_METHOD_DIRECT : NET_METHOD_FAST;
    // the caller's topology pointers are needed once, by the builder
    h->desc.topo.row_ptr = desc->topo.row_ptr;
    h->desc.topo.col_idx = desc->topo.col_idx;
    h->desc.topo.compressed = desc->topo.compressed;
    rc = topo_build(h);
    h->desc.topo.row_ptr = nullptr;
    h->desc.topo.col_idx = nullptr;
    h->desc.topo.compressed = nullptr;
    if (rc == NET_OK) rc = fast_prepare(h);
    cudaError_t e = cudaSuccess;
    if (rc == NET_OK) {
        size_t state = h->state_bytes;
        e = cudaMemsetAsync(h->b.y, 0, state, h->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(h->b.Y2, 0, state, h->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(h->b.Y3, 0, state, h->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(h->b.Y4, 0, state, h->stream);
        if (e != cudaSuccess) rc = cuda_err(h, e, "cudaMemsetAsync(state)");
    }
    if (rc == NET_OK) {
        double v0 = desc->model == NET_MODEL_KS ? ((const net_ks_params*)params)->omega0
                  : desc->model == NET_MODEL_KSI ? ((const net_ksi_params*)params)->omega0
                  : (desc->model == NET_MODEL_HH || desc->model == NET_MODEL_HHS) ? ((const net_hh_params*)params)->I_ext0 : 0.0;
        rc = fill_elem_param(h, v0);
    }
    if (rc == NET_OK) {
        e = cudaStreamSynchronize(h->stream);
        if (e != cudaSuccess) rc = cuda_err(h, e, "cudaStreamSynchronize(net_create)");
    }
    if (rc != NET_OK) {
        memcpy(g_err, h->err, sizeof(g_err));
        delete h;
        return rc;
    }
    *out = h;
    return NET_OK;
}

int32_t net_destroy(net_t* h) {
    DevGuard guard_(h);
    if (!h) return NET_OK;
    drop_graph(h);
    delete h;
    return NET_OK;
}

int32_t net_set_state(net_t* h, const void* src, int32_t src_is_device) {
    DevGuard guard_(h);
    if (!h) return NET_ERR_INVALID;
    if (!src) return set_err(h, NET_ERR_INVALID, "src is NULL");
    h->s_valid = 0;
    int32_t rc = copy_state(h, h->b.y, const_cast<void*>(src), true, src_is_device != 0);
    if (rc == NET_OK && h->desc.model == NET_MODEL_FHN2) rc = delay_reset_history(h);   // constant initial function
    return rc;
}

int32_t net_get_state(net_t* h, void* dst, int32_t dst_is_device) {
    DevGuard guard_(h);
    if (!h) return NET_ERR_INVALID;
    if (!dst) return set_err(h, NET_ERR_INVALID, "dst is NULL");
    return copy_state(h, h->b.y, dst, false, dst_is_device != 0);
}

int32_t net_set_param_array(net_t* h, int32_t which, const void* src, int32_t src_is_device) {
    DevGuard guard_(h);
    if (!h) return NET_ERR_INVALID;
    if (!src) return set_err(h, NET_ERR_INVALID, "src is NULL");
    if (!((which == NET_PARAM_OMEGA && (h->desc.model == NET_MODEL_KS || h->desc.model == NET_MODEL_KSI)) ||
          (which == NET_PARAM_IEXT && (h->desc.model == NET_MODEL_HH || h->desc.model == NET_MODEL_HHS))))
        return set_err(h, NET_ERR_INVALID, "parameter array %d does not belong to model %d", which, h->desc.model);
    OSC_CUDA(h, cudaMemcpyAsync(h->b.elem_param, src, (size_t)h->n * h->esize,
                                src_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, h->stream));
    if (!src_is_device) OSC_CUDA(h, cudaStreamSynchronize(h->stream));
    return NET_OK;
}

int32_t net_hh_steady_gates(net_t* h) {
    DevGuard guard_(h);
    if (!h) return NET_ERR_INVALID;
    if (h->desc.model != NET_MODEL_HH && h->desc.model != NET_MODEL_HHS) return set_err(h, NET_ERR_INVALID, "net_hh_steady_gates on a non-HH net");
    return hh_steady_gates(h);
}

int32_t net_integrate(net_t* h, int64_t n_steps, double dt) {
    DevGuard guard_(h);
    if (!h) return NET_ERR_INVALID;
    if (n_steps < 0 || !(dt == dt)) return set_err(h, NET_ERR_INVALID, "n_steps < 0 or dt is NaN");
    if (n_steps == 0) return NET_OK;
    return integrate_plain(h, n_steps, dt);
}

int32_t net_integrate_observed(net_t* h, int64_t n_steps, double dt, int64_t obs_every) {
    DevGuard guard_(h);
    if (!h) return NET_ERR_INVALID;
    if (n_steps < 1 || obs_every < 1 || n_steps % obs_every != 0)
        return set_err(h, NET_ERR_INVALID, "need n_steps >= 1, obs_every >= 1 and n_steps %% obs_every == 0");
    int32_t rc = obs_window_begin(h);
    if (rc) return rc;
    const double t0 = h->t;
    {   // phase models on the persistent ring kernel: one launch, samples taken inside it
        int64_t first = (n_steps + 1) / 2;                              // smallest s with 2 s >= n_steps ...
        first = (first + obs_every - 1) / obs_every * obs_every;        // ... that is a sample step
        if (first < obs_every) first = obs_every;
        bool handled = false;
        if ((rc = ring_run_observed(h, n_steps, dt, obs_every, first, &handled))) return rc;
        if (handled) {
            h->step += n_steps;
            h->t += (double)n_steps * dt;
            if ((rc = obs_window_sample(h, first == n_steps))) return rc;      // the sample at n_steps
            return obs_window_finish(h, t0 + (double)first * dt, t0 + (double)n_steps * dt, (n_steps - first) / obs_every + 1);
        }
    }
    int64_t n_samples = 0, s_a = -1;
    for (int64_t s = obs_every; s <= n_steps; s += obs_every) {
        if ((rc = integrate_plain(h, obs_every, dt))) return rc;
        if (2 * s < n_steps) continue;
        if ((rc = obs_window_sample(h, s_a < 0))) return rc;
        if (s_a < 0) s_a = s;
        ++n_samples;
    }
    return obs_window_finish(h, t0 + (double)s_a * dt, t0 + (double)n_steps * dt, n_samples);
}

int32_t net_adaptive_workspace_bytes(net_t* h, size_t* bytes) {
    if (!h || !bytes) return set_err(h, NET_ERR_INVALID, "net or bytes is NULL");
    *bytes = adaptive_workspace_bytes(h);
    return NET_OK;
}

int32_t net_integrate_adaptive(net_t* h, double t_end, double rtol, double atol, double h0, int64_t max_attempts,
                               void* d_work, size_t work_bytes, double* out5) {
    DevGuard guard_(h);
    if (!h || !out5) return set_err(h, NET_ERR_INVALID, "net or out5 is NULL");
    if (h->desc.model == NET_MODEL_FHN2 && (h->desc.delay_steps > 0 || h->mp.noise_D != 0.0))
        return set_err(h, NET_ERR_UNSUPPORTED, "net_integrate_adaptive: eq. (2) with delay or noise runs under the fixed-step integrator only");
    return adaptive_integrate(h, t_end, rtol, atol, h0, max_attempts, d_work, work_bytes, out5);
}

int32_t net_integrate_adaptive_dense(net_t* h, int64_t n_out, const double* t_out, void* d_out, double rtol, double atol,
                                     double h0, int64_t max_attempts, void* d_work, size_t work_bytes, double* out5) {
    DevGuard guard_(h);
    if (!h || !out5) return set_err(h, NET_ERR_INVALID, "net or out5 is NULL");
    if (h->desc.model == NET_MODEL_FHN2 && (h->desc.delay_steps > 0 || h->mp.noise_D != 0.0))
        return set_err(h, NET_ERR_UNSUPPORTED, "net_integrate_adaptive_dense: eq. (2) with delay or noise runs under the fixed-step integrator only");
    return adaptive_integrate_dense(h, n_out, t_out, d_out, rtol, atol, h0, max_attempts, d_work, work_bytes, out5);
}

int32_t net_eval_rhs(net_t* h, void* dst, int32_t dst_is_device) {
    DevGuard guard_(h);
    if (!h) return NET_ERR_INVALID;
    if (!dst) return set_err(h, NET_ERR_INVALID, "dst is NULL");
    int32_t rc = ensure_s(h);
    if (rc) return rc;
    StageArgs a = stage_args(h, 0, 0.0);
    a.stage = STAGE_RHS_ONLY;
    a.out = h->b.Y4;  // scratch: Y4 is rewritten by the next step anyway
    a.s_out = nullptr;
    if ((rc = run_stage(h, a))) return rc;
    return copy_state(h, h->b.Y4, dst, false, dst_is_device != 0);
}

int32_t net_observables(net_t* h, int32_t what, void* dst, int32_t dst_is_device) {
    DevGuard guard_(h);
    if (!h) return NET_ERR_INVALID;
    if (!dst) return set_err(h, NET_ERR_INVALID, "dst is NULL");
    cudaMemcpyKind kind = dst_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    int32_t rc = NET_OK;
    const double* src = nullptr;
    size_t bytes = 0;
    double* theta = h->b.obs_tmp;  // first half of the 2n scratch
    switch (what) {
        case NET_OBS_PHASE:
            if ((rc = obs_phase(h, h->b.y, h->b.obs_loc))) return rc;
            src = h->b.obs_loc; bytes = sizeof(double) * h->n;
            break;
        case NET_OBS_GLOBAL_ORDER:
            if ((rc = obs_phase(h, h->b.y, theta))) return rc;
            if ((rc = obs_global_order(h, theta, h->b.obs_acc + 8))) return rc;
            src = h->b.obs_acc + 8; bytes = 2 * sizeof(double);
            break;
        case NET_OBS_REPLICA_ORDER:
            // obs_loc (n doubles) receives the 2 * batch results; n >= 2 * batch since every ring has n >= 2
            if (2 * (int64_t)h->desc.batch > h->n) return set_err(h, NET_ERR_UNSUPPORTED, "replica order parameter: rings of one element");
            if ((rc = obs_phase(h, h->b.y, theta))) return rc;
            if ((rc = obs_replica_order(h, theta, h->b.obs_loc))) return rc;
            src = h->b.obs_loc; bytes = 2 * sizeof(double) * (size_t)h->desc.batch;
            break;
        case NET_OBS_LOCAL_ORDER: {
            // obs_theta_prev doubles as theta scratch here (obs_tmp holds cos/sin); an observed
            // run re-initialises it at its first window sample
            double* th = h->b.obs_theta_prev;
            if ((rc = obs_phase(h, h->b.y, th))) return rc;
            if ((rc = obs_local_order(h, th, h->b.obs_loc))) return rc;
            src = h->b.obs_loc; bytes = sizeof(double) * h->n;
            break;
        }
        case NET_OBS_MEAN_PHASE_VELOCITY:
            if (!h->stats_valid) return set_err(h, NET_ERR_INVALID, "no net_integrate_observed window yet");
            src = h->b.obs_vel; bytes = sizeof(double) * h->n;
            break;
        case NET_OBS_STATS:
            if (!h->stats_valid) return set_err(h, NET_ERR_INVALID, "no net_integrate_observed window yet");
            if (dst_is_device) {
                OSC_CUDA(h, cudaMemcpyAsync(dst, h->stats, sizeof(h->stats), cudaMemcpyHostToDevice, h->stream));
                OSC_CUDA(h, cudaStreamSynchronize(h->stream));
            } else memcpy(dst, h->stats, sizeof(h->stats));
            return NET_OK;
        default: return set_err(h, NET_ERR_INVALID, "unknown observable %d", what);
    }
    OSC_CUDA(h, cudaMemcpyAsync(dst, src, bytes, kind, h->stream));
    if (!dst_is_device) OSC_CUDA(h, cudaStreamSynchronize(h->stream));
    return NET_OK;
}

int32_t net_get_topology(net_t* h, int64_t row_begin, int64_t row_count, int64_t* row_ptr,
                         int32_t* col_idx, int32_t dst_is_device) {
    DevGuard guard_(h);
    if (!h) return NET_ERR_INVALID;
    if (!row_ptr || !col_idx) return set_err(h, NET_ERR_INVALID, "row_ptr / col_idx is NULL");
    if (row_begin < 0 || row_count < 0 || row_begin + row_count > h->n)
        return set_err(h, NET_ERR_INVALID, "row range outside [0, n]");
    if (dst_is_device) return topo_expand(h, row_begin, row_count, row_ptr, col_idx);
    if ((h->tv.kind == NET_TOPO_CSR || h->tv.kind == NET_TOPO_RANDOM_INDEGREE) && h->desc.batch > 1 && h->degree_uniform < 0)
        return set_err(h, NET_ERR_UNSUPPORTED, "net_get_topology to host memory: batches of graphs with non-uniform rows (use a device destination)");
    if ((h->tv.kind == NET_TOPO_CSR || h->tv.kind == NET_TOPO_RANDOM_INDEGREE) && h->desc.batch == 1) {
        OSC_CUDA(h, cudaMemcpyAsync(row_ptr, h->b.row_ptr + row_begin, sizeof(int64_t) * (row_count + 1), cudaMemcpyDeviceToHost, h->stream));
        OSC_CUDA(h, cudaStreamSynchronize(h->stream));
        int64_t base = row_ptr[0], cnt = row_ptr[row_count] - base;
        for (int64_t r = 0; r <= row_count; ++r) row_ptr[r] -= base;
        if (cnt > 0) OSC_CUDA(h, cudaMemcpyAsync(col_idx, h->b.col_idx + base, sizeof(int32_t) * cnt, cudaMemcpyDeviceToHost, h->stream));
        OSC_CUDA(h, cudaStreamSynchronize(h->stream));
        return NET_OK;
    }
    if (h->tv.kind == NET_TOPO_COMPRESSED) {
        // EXTRACT chunk by chunk through the staging scratch (rows of at most cmp_maxdeg entries)
        const size_t per_row = sizeof(int32_t) * (size_t)(h->tv.cmp_maxdeg > 0 ? h->tv.cmp_maxdeg : 1) + sizeof(int64_t);
        int64_t chunk = (int64_t)((h->b.scratch_bytes - 512) / per_row);
        if (chunk < 1) return set_err(h, NET_ERR_SIZE, "staging scratch too small for one row");
        int64_t base = 0;
        row_ptr[0] = 0;
        for (int64_t r0 = 0; r0 < row_count; r0 += chunk) {
            const int64_t rows = row_count - r0 < chunk ? row_count - r0 : chunk;
            int64_t* d_ptr = (int64_t*)h->b.scratch;
            int32_t* d_idx = (int32_t*)((char*)h->b.scratch + round_up((int64_t)sizeof(int64_t) * (rows + 1), 256));
            int32_t rc = topo_expand(h, row_begin + r0, rows, d_ptr, d_idx);
            if (rc) return rc;
            OSC_CUDA(h, cudaMemcpyAsync(row_ptr + r0 + 1, d_ptr + 1, sizeof(int64_t) * rows, cudaMemcpyDeviceToHost, h->stream));
            OSC_CUDA(h, cudaStreamSynchronize(h->stream));
            const int64_t cnt = row_ptr[r0 + rows];
            if (cnt > 0) OSC_CUDA(h, cudaMemcpyAsync(col_idx + base, d_idx, sizeof(int32_t) * cnt, cudaMemcpyDeviceToHost, h->stream));
            OSC_CUDA(h, cudaStreamSynchronize(h->stream));
            for (int64_t r = 1; r <= rows; ++r) row_ptr[r0 + r] += base;
            base += cnt;
        }
        return NET_OK;
    }
    // ring / lattice: expand chunk by chunk through the staging scratch.  That region also holds
    // the exchange fields of y on the lattice FAST paths: have them rebuilt before the next stage.
    h->s_valid = 0;
    const int64_t deg = h->degree_uniform;
    const size_t per_row = sizeof(int32_t) * (size_t)(deg > 0 ? deg : 1) + sizeof(int64_t);
    int64_t chunk = (int64_t)((h->b.scratch_bytes - 256) / per_row);
    if (chunk < 1) return set_err(h, NET_ERR_SIZE, "staging scratch too small for one row");
    for (int64_t r0 = 0; r0 < row_count || r0 == 0; r0 += chunk) {
        int64_t rc_rows = row_count - r0 < chunk ? row_count - r0 : chunk;
        int64_t* d_ptr = (int64_t*)h->b.scratch;
        int32_t* d_idx = (int32_t*)((char*)h->b.scratch + round_up((int64_t)sizeof(int64_t) * (rc_rows + 1), 256));
        int32_t rc = topo_expand(h, row_begin + r0, rc_rows, d_ptr, d_idx);
        if (rc) return rc;
        if (rc_rows * deg > 0)
            OSC_CUDA(h, cudaMemcpyAsync(col_idx + r0 * deg, d_idx, sizeof(int32_t) * rc_rows * deg, cudaMemcpyDeviceToHost, h->stream));
        OSC_CUDA(h, cudaStreamSynchronize(h->stream));
        if (row_count == 0) break;
    }
    for (int64_t r = 0; r <= row_count; ++r) row_ptr[r] = r * deg;
    return NET_OK;
}

int32_t net_get_degree(net_t* h, int64_t* nnz, int32_t* uniform_degree) {
    if (!h) return NET_ERR_INVALID;
    if (nnz) *nnz = h->nnz;
    if (uniform_degree) *uniform_degree = h->degree_uniform;
    return NET_OK;
}

int32_t net_get_time(net_t* h, double* t, int64_t* step) {
    if (!h) return NET_ERR_INVALID;
    if (t) *t = h->t;
    if (step) *step = h->step;
    return NET_OK;
}

int32_t net_set_time(net_t* h, double t, int64_t step) {
    if (!h) return NET_ERR_INVALID;
    h->t = t;
    h->step = step;
    return NET_OK;
}

int32_t net_get_counters(net_t* h, int64_t* kernel_launches, int32_t* method_in_use) {
    if (!h) return NET_ERR_INVALID;
    if (kernel_launches) *kernel_launches = h->launches;
    if (method_in_use) *method_in_use = h->method;
    return NET_OK;
}

int32_t net_get_kernel_family(net_t* h, int32_t* family) {
    if (!h) return NET_ERR_INVALID;
    if (family) *family = h->method == NET_METHOD_FAST ? h->fast_kind : FAST_NONE;
    return NET_OK;
}

int32_t net_get_launch_config(net_t* h, int32_t* out8) {
    if (!h || !out8) return NET_ERR_INVALID;
    for (int q = 0; q < 8; ++q) out8[q] = 0;
    out8[0] = h->method == NET_METHOD_FAST ? h->fast_kind : FAST_NONE;
    if (out8[0] == FAST_LATTICE3D_V3) {
        const L3Geom& g = h->lat3[1];
        out8[1] = g.TXt; out8[2] = g.TYt; out8[3] = g.Lz; out8[4] = g.D;
        out8[5] = (int32_t)h->lat3_grid[1]; out8[6] = h->lat3_threads[1]; out8[7] = (int32_t)h->lat3_smem[1];
    } else if (out8[0] == FAST_LATTICE3D_V2) {
        out8[1] = h->lat2.TXt; out8[2] = h->lat2.TYt; out8[3] = h->lat2.Lz; out8[4] = h->lat2.D;
        out8[5] = (int32_t)h->lat2_grid; out8[6] = h->lat2_threads; out8[7] = (int32_t)h->lat2_smem;
    } else if (out8[0] == FAST_CSR_BLOCKED) {
        out8[1] = h->cb_pair; out8[2] = h->cb_es; out8[5] = (int32_t)h->cb_grid; out8[6] = 1024; out8[7] = (int32_t)h->cb_smem;
    }
    return NET_OK;
}

int32_t net_synchronize(net_t* h) {
    DevGuard guard_(h);
    if (!h) return NET_ERR_INVALID;
    OSC_CUDA(h, cudaStreamSynchronize(h->stream));
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

}  // extern "C"
#pragma GCC visibility pop
