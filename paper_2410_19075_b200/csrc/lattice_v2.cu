// Glue of the second-generation 3D lattice kernels (lattice_v2.cuh): support test, buffer
// roles of the Z-form RK4 stages, the ghost-padded interleaved-pair layout and its fill /
// unpack kernels, the KS exchange field.
#include "models.cuh"

namespace oscnet {

int32_t lattice_v2_entry_f32(net* h, const Lat2Args* a, int nops, int which_map);
int32_t lattice_v2_entry_f64(net* h, const Lat2Args* a, int nops, int which_map);

// x ghost width in pairs (the halo rounded up to whole 16-byte vectors), y ghost width = P
static int l2_gx(int dtype, int P) { return dtype == NET_F32 ? (P + 1) / 2 * 2 : P; }

static size_t padded_pairs(const net_desc* d) {
    const net_topology& t = d->topo;
    const int P = t.radius, GX = l2_gx(d->dtype, P);
    return (size_t)t.extent[2] * (size_t)(t.extent[1] + 2 * P) * (size_t)(t.extent[0] + 2 * GX);
}

bool lattice_v2_supported(const net_desc* d) {
    const net_topology& t = d->topo;
    if (t.kind != NET_TOPO_LATTICE || t.ndim != 3) return false;
    if (d->model != NET_MODEL_KS && d->model != NET_MODEL_FHN && d->model != NET_MODEL_KSI) return false;
    // radius 2, 4: every kernel generation; radius 6 (the paper's largest): the field-split kernel (KS, KSI)
    if (t.radius != 2 && t.radius != 4 && !(t.radius == 6 && d->model != NET_MODEL_FHN)) return false;
    // rows must be whole 16-byte vectors of the per-thread column group (X = 2 columns)
    return t.extent[0] % 2 == 0;
}

// bytes of one state buffer (FHN: the padded pair array; KS: plain phi)
size_t lattice_v2_state_bytes(const net_desc* d) {
    const size_t es = d->dtype == NET_F32 ? 4 : 8;
    if (d->model == NET_MODEL_FHN) return padded_pairs(d) * 2 * es + 256;
    return 0;
}

size_t lattice_v2_scratch_bytes(const net_desc* d) {
    if (d->model != NET_MODEL_KS && d->model != NET_MODEL_KSI) return 0;
    const size_t es = d->dtype == NET_F32 ? 4 : 8;
    size_t b = 2 * ((padded_pairs(d) * 2 * es + 255) / 256 * 256) + 512;     // E_a, E_b
    if (d->model == NET_MODEL_KSI) b += (size_t)round_up(d->n, 64) * es + 256;   // coupling term of the stage input
    return b;
}

int32_t lattice_v2_prepare(net* h) {
    h->ks_planar = 0;
    if (h->desc.model == NET_MODEL_KS) {
        char* s = (char*)h->b.scratch;
        h->E_a = s;
        h->E_b = s + (padded_pairs(&h->desc) * 2 * h->esize + 255) / 256 * 256;
    }
    int32_t rc = h->desc.dtype == NET_F32 ? lattice_v2_entry_f32(h, nullptr, 0, 0)
                                          : lattice_v2_entry_f64(h, nullptr, 0, 0);
    if (rc) return rc;
    if (h->desc.model == NET_MODEL_FHN) h->pairs = 1;
    else {
        // the ghost cells of E must never hold NaN bit patterns from stale memory: they are
        // rewritten by every producer, but zero them once for the first refresh
        OSC_CUDA(h, cudaMemsetAsync(h->E_a, 0, padded_pairs(&h->desc) * 2 * h->esize, h->stream));
        OSC_CUDA(h, cudaMemsetAsync(h->E_b, 0, padded_pairs(&h->desc) * 2 * h->esize, h->stream));
    }
    return NET_OK;
}

// Buffer roles per stage (Z form): in = y, Y2, Y3, Y4; out = Y2, Y3, Y4 (+ Z into Y2), y.
int32_t lattice_v2_stage(net* h, const StageArgs& sa) {
    const Buffers& b = h->b;
    const bool ks = h->desc.model == NET_MODEL_KS;
    Lat2Args a;
    memset(&a, 0, sizeof(a));
    a.dt = sa.dt; a.stage = sa.stage; a.omega = b.elem_param;
    int nops = 0, map = 0;
    switch (sa.stage) {
        case 0: map = 0; a.out = b.Y2; a.Eout = h->E_b;
                if (ks) { a.op0 = b.y; nops = 1; }
                break;
        case 1: map = 1; a.out = b.Y3; a.Eout = h->E_a; a.op0 = b.y; nops = 1; break;
        case 2: map = ks ? 0 : 2; a.out = b.Y4; a.out2 = b.Y2; a.Eout = h->E_b;
                a.op0 = b.y; a.op1 = b.Y2; a.op2 = b.Y3; nops = ks ? 3 : 2;
                break;
        case 3: map = ks ? 1 : 3; a.out = b.y; a.Eout = h->E_a; a.op0 = b.Y2; nops = 1; break;
        default: map = 0; a.out = sa.out; nops = 0; break;   // RHS of y
    }
    return h->desc.dtype == NET_F32 ? lattice_v2_entry_f32(h, &a, nops, map)
                                    : lattice_v2_entry_f64(h, &a, nops, map);
}

// ------------------------------------------------------------------ layout helpers
// MODE 0: pairs <- (soa[i], soa[ld+i]);  MODE 1: pairs <- (cos, sin) soa[i];  MODE 2: two planes
// (cos soa[i] | sin soa[i]).  Every padded position, ghosts included, takes the value of its
// periodic image.
template <class T, int MODE>
__global__ void pad_fill_kernel(const T* __restrict__ soa, T* __restrict__ pr, int nx, int ny, int nz,
                                int GX, int GY, int64_t ld) {
    const int nxp = nx + 2 * GX, nyp = ny + 2 * GY;
    const int64_t total = (int64_t)nz * nyp * nxp;
    for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        const int xp = (int)(e % nxp);
        const int64_t t = e / nxp;
        const int yp = (int)(t % nyp), z = (int)(t / nyp);
        int x = (xp - GX) % nx; if (x < 0) x += nx;
        int y = (yp - GY) % ny; if (y < 0) y += ny;
        const int64_t i = ((int64_t)z * ny + y) * nx + x;
        if (MODE == 0) { pr[2 * e] = soa[i]; pr[2 * e + 1] = soa[ld + i]; }
        else {
            T s, c;
            Math<T>::sincos(soa[i], &s, &c);
            if (MODE == 1) { pr[2 * e] = c; pr[2 * e + 1] = s; }
            else { pr[e] = c; pr[total + e] = s; }
        }
    }
}
template <class T>
__global__ void pad_unpack_kernel(const T* __restrict__ pr, T* __restrict__ soa, int nx, int ny, int nz,
                                  int GX, int GY, int64_t ld) {
    const int nxp = nx + 2 * GX, nyp = ny + 2 * GY;
    const int64_t n = (int64_t)nx * ny * nz;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int x = (int)(i % nx);
        const int64_t t = i / nx;
        const int y = (int)(t % ny), z = (int)(t / ny);
        const int64_t e = ((int64_t)z * nyp + (y + GY)) * nxp + (x + GX);
        soa[i] = pr[2 * e];
        soa[ld + i] = pr[2 * e + 1];
    }
}

static unsigned l2_grid_for(int64_t n) {
    int64_t b = (n + 255) / 256;
    return (unsigned)(b < 1 ? 1 : b > 148 * 16 ? 148 * 16 : b);
}

template <int MODE>
static int32_t pad_fill(net* h, const void* soa, void* pr) {
    const TopoView& tv = h->tv;
    const int GX = l2_gx(h->desc.dtype, tv.P), GY = tv.P;
    const unsigned g = l2_grid_for((int64_t)padded_pairs(&h->desc));
    if (h->desc.dtype == NET_F32)
        pad_fill_kernel<float, MODE><<<g, 256, 0, h->stream>>>((const float*)soa, (float*)pr, tv.nx, tv.ny, tv.nz, GX, GY, h->ld);
    else
        pad_fill_kernel<double, MODE><<<g, 256, 0, h->stream>>>((const double*)soa, (double*)pr, tv.nx, tv.ny, tv.nz, GX, GY, h->ld);
    h->launches += 1;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

int32_t pairs_pack(net* h, const void* soa, void* pairs) { return pad_fill<0>(h, soa, pairs); }

int32_t pairs_unpack(net* h, const void* pairs, void* soa) {
    const TopoView& tv = h->tv;
    const int GX = l2_gx(h->desc.dtype, tv.P), GY = tv.P;
    if (h->desc.dtype == NET_F32)
        pad_unpack_kernel<float><<<l2_grid_for(h->n), 256, 0, h->stream>>>((const float*)pairs, (float*)soa, tv.nx, tv.ny, tv.nz, GX, GY, h->ld);
    else
        pad_unpack_kernel<double><<<l2_grid_for(h->n), 256, 0, h->stream>>>((const double*)pairs, (double*)soa, tv.nx, tv.ny, tv.nz, GX, GY, h->ld);
    h->launches += 1;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

// exchange field E_a = (cos, sin) of the phase row of `state` ([nvar][ld]; nullptr = the net's y)
int32_t lattice_v2_refresh_exchange(net* h, const void* state) {
    if (h->desc.model != NET_MODEL_KS && h->desc.model != NET_MODEL_KSI) return NET_OK;
    const void* src = state ? state : h->b.y;
    return h->ks_planar ? pad_fill<2>(h, src, h->E_a) : pad_fill<1>(h, src, h->E_a);
}

}  // namespace oscnet

// ------------------------------------------------------------------ third generation (lat3_kernel.cuh)
// Same data layout as the second generation (ghost-padded pair arrays, KS exchange fields E_a / E_b);
// only the stage kernels differ.
namespace oscnet {

int32_t lattice_v3_entry_f32_fhn(net* h, int stage, double dt, void* rhs_out);
int32_t lattice_v3_entry_f32_ks(net* h, int stage, double dt, void* rhs_out);
int32_t lattice_v3_entry_f64_fhn(net* h, int stage, double dt, void* rhs_out);
int32_t lattice_v3_entry_f64_ks(net* h, int stage, double dt, void* rhs_out);
int32_t lattice_v3_entry_f32_ks6(net* h, int stage, double dt, void* rhs_out);
int32_t lattice_v3_entry_f64_ks6(net* h, int stage, double dt, void* rhs_out);

static int32_t l3_dispatch(net* h, int stage, double dt, void* rhs_out) {
    const bool ks = h->desc.model == NET_MODEL_KS || h->desc.model == NET_MODEL_KSI;   // KSI: the KS kernels' RHS instance
    if (ks && h->tv.P == 6)
        return h->desc.dtype == NET_F32 ? lattice_v3_entry_f32_ks6(h, stage, dt, rhs_out) : lattice_v3_entry_f64_ks6(h, stage, dt, rhs_out);
    if (h->desc.dtype == NET_F32)
        return ks ? lattice_v3_entry_f32_ks(h, stage, dt, rhs_out) : lattice_v3_entry_f32_fhn(h, stage, dt, rhs_out);
    return ks ? lattice_v3_entry_f64_ks(h, stage, dt, rhs_out) : lattice_v3_entry_f64_fhn(h, stage, dt, rhs_out);
}

bool lattice_v3_supported(const net_desc* d) {
    if (!lattice_v2_supported(d)) return false;
    if (getenv("OSCNET_NO_LAT3")) return false;
    // KS operand tiles are rows of scalars: whole 16-byte vectors
    if ((d->model == NET_MODEL_KS || d->model == NET_MODEL_KSI) && d->dtype == NET_F32 && d->topo.extent[0] % 4 != 0) return false;
    return true;
}

int32_t lattice_v3_prepare(net* h) {
    if (h->desc.model == NET_MODEL_KS || h->desc.model == NET_MODEL_KSI) {
        char* s = (char*)h->b.scratch;
        const size_t eb = (padded_pairs(&h->desc) * 2 * h->esize + 255) / 256 * 256;
        h->E_a = s;
        h->E_b = s + eb;
        h->ksi_c = s + 2 * eb + 256;          // KSI: omega + (K/Omega) sum sin(...) of the stage input
    }
    int32_t rc = l3_dispatch(h, -1, 0.0, nullptr);
    if (rc) return rc;
    if (h->desc.model == NET_MODEL_FHN) h->pairs = 1;
    else {
        OSC_CUDA(h, cudaMemsetAsync(h->E_a, 0, padded_pairs(&h->desc) * 2 * h->esize, h->stream));
        OSC_CUDA(h, cudaMemsetAsync(h->E_b, 0, padded_pairs(&h->desc) * 2 * h->esize, h->stream));
    }
    return NET_OK;
}

// Kuramoto-Sakaguchi with inertia (eq. (3) in full; the paper's own performance model,
// PAPER.md:327, :337-343) on the field-split lattice kernels: psi is a LOCAL variable, the coupling
// is the KS one, so a stage is (1) the RHS instance of lat3s_kernel on the exchange field E of the
// stage input -- c_i = omega_i + (K/Omega) sum_j sin(phi_j - phi_i - alpha), run sums and all --
// and (2) one pointwise kernel: phi' = psi, psi' = (c - eps psi)/m, the RK4 stage update of both
// variables, and E = (cos, sin) of the new phi with its periodic ghost images for the next stage.
template <class T>
__global__ void __launch_bounds__(256) ksi_update_kernel(StageArgs a, ModelParams mp, const T* __restrict__ c,
                                                        T* __restrict__ E, int nx, int ny, int nz, int HX, int P, long long plane) {
    const int64_t n = a.n, ld = a.ld;
    const T* __restrict__ in = (const T*)a.in;
    const int stage = a.stage;
    const T dt = (T)a.dt;
    const int nxp = nx + 2 * HX, nyp = ny + 2 * P;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const T xin[2] = {in[i], in[ld + i]};
        const T k[2] = {xin[1], (c[i] - T(mp.damp) * xin[1]) * T(mp.inv_m)};
        T o[2];
#pragma unroll
        for (int v = 0; v < 2; ++v) {
            T y = 0, y2 = 0, y3 = 0;
            if (stage != STAGE_RHS_ONLY) y = ((const T*)a.y)[v * ld + i];
            if (stage == 3) { y2 = ((const T*)a.Y2)[v * ld + i]; y3 = ((const T*)a.Y3)[v * ld + i]; }
            o[v] = stage_combine<T>(stage, dt, k[v], y, y2, y3, xin[v]);
            ((T*)a.out)[v * ld + i] = o[v];
        }
        if (stage == STAGE_RHS_ONLY) continue;
        T sn, cs;
        sincos_stage<T>(o[0], &sn, &cs);
        const int x = (int)(i % nx);
        const int64_t r = i / nx;
        const int y = (int)(r % ny), z = (int)(r / ny);
        const int64_t ip = ((int64_t)z * nyp + (y + P)) * nxp + (x + HX);
        const int gxs = x < HX ? nx : (x >= nx - HX ? -nx : 0);      // periodic images this element also owns
        const int gys = y < P ? ny : (y >= ny - P ? -ny : 0);
        auto put = [&](int64_t at) { E[at] = cs; E[plane + at] = sn; };
        put(ip);
        if (gxs) put(ip + gxs);
        if (gys) {
            put(ip + (int64_t)gys * nxp);
            if (gxs) put(ip + (int64_t)gys * nxp + gxs);
        }
    }
}

static int32_t ksi_lattice_stage(net* h, const StageArgs& sa) {
    int32_t rc = l3_dispatch(h, 4, 0.0, h->ksi_c);           // RHS instance of the KS kernel on E_a = E(stage input)
    if (rc) return rc;
    const TopoView& tv = h->tv;
    const int HX = l2_gx(h->desc.dtype, tv.P);
    const long long plane = (long long)(tv.nx + 2 * HX) * (tv.ny + 2 * tv.P) * tv.nz;
    const unsigned g = l2_grid_for(h->n);
    if (h->desc.dtype == NET_F32)
        ksi_update_kernel<float><<<g, 256, 0, h->stream>>>(sa, h->mp, (const float*)h->ksi_c, (float*)h->E_a, tv.nx, tv.ny, tv.nz, HX, tv.P, plane);
    else
        ksi_update_kernel<double><<<g, 256, 0, h->stream>>>(sa, h->mp, (const double*)h->ksi_c, (double*)h->E_a, tv.nx, tv.ny, tv.nz, HX, tv.P, plane);
    h->launches += 1;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

// ------------------------------------------------------------------ local order parameter
// R_i = |sum over the ball incl. i of e^{i theta_j}| / n_ball (reading R9) through the L3_LOC instance
// of the lattice kernels instead of one gather per link.  KS / KSI: the unit phasor field is the
// exchange field E(y) the stages keep anyway.  FHN: (u, v)/|(u, v)| of every padded position of y
// (ghosts hold the periodic images already) is written to Y3, which is dead between steps.
template <class T>
__global__ void unit_pairs_kernel(const T* __restrict__ y, T* __restrict__ out, int64_t pairs) {
    for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < pairs; e += (int64_t)gridDim.x * blockDim.x) {
        const T u = y[2 * e], v = y[2 * e + 1];
        // theta = atan2(v, u); (cos, sin) theta = (u, v)/r, and (1, 0) at the origin as atan2(0, 0) = 0
        const T r = sqrt(u * u + v * v);
        out[2 * e] = r > T(0) ? u / r : T(1);
        out[2 * e + 1] = r > T(0) ? v / r : T(0);
    }
}

template <class T>
__global__ void widen_kernel(const T* __restrict__ in, double* __restrict__ out, int64_t n) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) out[i] = (double)in[i];
}

bool lattice_v3_has_local_order(const net* h) {
    return h->method == NET_METHOD_FAST && h->fast_kind == FAST_LATTICE3D_V3 && !getenv("OSCNET_NO_FAST_OBS");
}

int32_t lattice_v3_local_order(net* h, double* d_out) {
    int32_t rc;
    const bool f32 = h->desc.dtype == NET_F32;
    if (h->desc.model == NET_MODEL_FHN) {
        const int64_t pairs = (int64_t)padded_pairs(&h->desc);
        if (f32) unit_pairs_kernel<float><<<l2_grid_for(pairs), 256, 0, h->stream>>>((const float*)h->b.y, (float*)h->b.Y3, pairs);
        else unit_pairs_kernel<double><<<l2_grid_for(pairs), 256, 0, h->stream>>>((const double*)h->b.y, (double*)h->b.Y3, pairs);
        h->launches += 1;
    } else if (!h->s_valid) {
        if ((rc = lattice_v2_refresh_exchange(h, nullptr))) return rc;
        h->s_valid = 1;
    }
    // fp32 nets: the kernel writes float (into Y4, rewritten by the next step), widened afterwards
    void* out = f32 ? h->b.Y4 : (void*)d_out;
    if ((rc = l3_dispatch(h, 5, 0.0, out))) return rc;
    if (f32) {
        widen_kernel<float><<<l2_grid_for(h->n), 256, 0, h->stream>>>((const float*)h->b.Y4, d_out, h->n);
        h->launches += 1;
    }
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

int32_t lattice_v3_stage(net* h, const StageArgs& sa) {
    if (h->desc.model == NET_MODEL_KSI) return ksi_lattice_stage(h, sa);
    return l3_dispatch(h, sa.stage == STAGE_RHS_ONLY ? 4 : sa.stage, sa.dt, sa.out);
}

}  // namespace oscnet
