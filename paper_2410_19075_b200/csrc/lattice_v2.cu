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
    if (t.radius != 2 && t.radius != 4) return false;
    if (d->model != NET_MODEL_KS && d->model != NET_MODEL_FHN) return false;
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
    if (d->model != NET_MODEL_KS) return 0;
    const size_t es = d->dtype == NET_F32 ? 4 : 8;
    return 2 * ((padded_pairs(d) * 2 * es + 255) / 256 * 256) + 512;     // E_a, E_b
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

int32_t lattice_v2_refresh_exchange(net* h) {
    if (h->desc.model != NET_MODEL_KS) return NET_OK;
    return h->ks_planar ? pad_fill<2>(h, h->b.y, h->E_a) : pad_fill<1>(h, h->b.y, h->E_a);
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

static int32_t l3_dispatch(net* h, int stage, double dt, void* rhs_out) {
    const bool ks = h->desc.model == NET_MODEL_KS;
    if (h->desc.dtype == NET_F32)
        return ks ? lattice_v3_entry_f32_ks(h, stage, dt, rhs_out) : lattice_v3_entry_f32_fhn(h, stage, dt, rhs_out);
    return ks ? lattice_v3_entry_f64_ks(h, stage, dt, rhs_out) : lattice_v3_entry_f64_fhn(h, stage, dt, rhs_out);
}

bool lattice_v3_supported(const net_desc* d) {
    if (!lattice_v2_supported(d)) return false;
    if (getenv("OSCNET_NO_LAT3")) return false;
    // KS operand tiles are rows of scalars: whole 16-byte vectors
    if (d->model == NET_MODEL_KS && d->dtype == NET_F32 && d->topo.extent[0] % 4 != 0) return false;
    return true;
}

int32_t lattice_v3_prepare(net* h) {
    if (h->desc.model == NET_MODEL_KS) {
        char* s = (char*)h->b.scratch;
        h->E_a = s;
        h->E_b = s + (padded_pairs(&h->desc) * 2 * h->esize + 255) / 256 * 256;
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

int32_t lattice_v3_stage(net* h, const StageArgs& sa) {
    return l3_dispatch(h, sa.stage == STAGE_RHS_ONLY ? 4 : sa.stage, sa.dt, sa.out);
}

}  // namespace oscnet
