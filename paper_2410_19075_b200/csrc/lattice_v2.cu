// Glue of the second-generation 3D lattice kernels (lattice_v2.cuh): support test, buffer
// roles of the Z-form RK4 stages, the interleaved-pair state layout and the KS exchange field.
#include "models.cuh"

namespace oscnet {

int32_t lattice_v2_entry_f32(net* h, const Lat2Args* a, int nops, Lat2* g, int* threads, size_t* smem, unsigned* grid);
int32_t lattice_v2_entry_f64(net* h, const Lat2Args* a, int nops, Lat2* g, int* threads, size_t* smem, unsigned* grid);

bool lattice_v2_supported(const net_desc* d) {
    const net_topology& t = d->topo;
    if (t.kind != NET_TOPO_LATTICE || t.ndim != 3) return false;
    if (t.radius != 2 && t.radius != 4) return false;
    if (d->model != NET_MODEL_KS && d->model != NET_MODEL_FHN) return false;
    // rows must be whole 16-byte vectors of the per-thread column group (X = 4 fp32, 2 fp64)
    const int64_t xmul = d->dtype == NET_F32 ? 4 : 2;
    return t.extent[0] % xmul == 0;
}

size_t lattice_v2_scratch_bytes(const net_desc* d) {
    if (d->model != NET_MODEL_KS) return 0;
    const size_t es = d->dtype == NET_F32 ? 4 : 8;
    const size_t ld = (size_t)round_up(d->n, 64);
    return 2 * (2 * ld * es) + 512;     // E_a, E_b
}

int32_t lattice_v2_prepare(net* h) {
    int32_t rc = h->desc.dtype == NET_F32
        ? lattice_v2_entry_f32(h, nullptr, 0, &h->lat2, &h->lat2_threads, &h->lat2_smem, &h->lat2_grid)
        : lattice_v2_entry_f64(h, nullptr, 0, &h->lat2, &h->lat2_threads, &h->lat2_smem, &h->lat2_grid);
    if (rc) return rc;
    if (h->desc.model == NET_MODEL_FHN) {
        h->pairs = 1; h->var_stride = 1; h->elem_stride = 2;
    } else {
        char* s = (char*)h->b.scratch;
        h->E_a = s;
        h->E_b = s + round_up((int64_t)(2 * h->ld * h->esize), 256);
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
    int nops = 0;
    switch (sa.stage) {
        case 0: a.Ein = ks ? h->E_a : b.y; a.out = b.Y2; a.Eout = h->E_b;
                if (ks) { a.op0 = b.y; nops = 1; }
                break;
        case 1: a.Ein = ks ? h->E_b : b.Y2; a.out = b.Y3; a.Eout = h->E_a; a.op0 = b.y; nops = 1; break;
        case 2: a.Ein = ks ? h->E_a : b.Y3; a.out = b.Y4; a.out2 = b.Y2; a.Eout = h->E_b;
                a.op0 = b.y; a.op1 = b.Y2; a.op2 = b.Y3; nops = ks ? 3 : 2;
                break;
        case 3: a.Ein = ks ? h->E_b : b.Y4; a.out = b.y; a.Eout = h->E_a; a.op0 = b.Y2; nops = 1; break;
        default: a.Ein = ks ? h->E_a : sa.in; a.out = sa.out; nops = 0; break;   // RHS of y
    }
    return h->desc.dtype == NET_F32
        ? lattice_v2_entry_f32(h, &a, nops, &h->lat2, &h->lat2_threads, &h->lat2_smem, &h->lat2_grid)
        : lattice_v2_entry_f64(h, &a, nops, &h->lat2, &h->lat2_threads, &h->lat2_smem, &h->lat2_grid);
}

// ------------------------------------------------------------------ layout helpers
template <class T>
__global__ void pack_kernel(const T* __restrict__ soa, T* __restrict__ pr, int64_t n, int64_t ld) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        pr[2 * i] = soa[i];
        pr[2 * i + 1] = soa[ld + i];
    }
}
template <class T>
__global__ void unpack_kernel(const T* __restrict__ pr, T* __restrict__ soa, int64_t n, int64_t ld) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        soa[i] = pr[2 * i];
        soa[ld + i] = pr[2 * i + 1];
    }
}
template <class T>
__global__ void ks_exchange_kernel(const T* __restrict__ phi, T* __restrict__ E, int64_t n) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        T s, c;
        Math<T>::sincos(phi[i], &s, &c);
        E[2 * i] = c;
        E[2 * i + 1] = s;
    }
}

static unsigned l2_grid_for(int64_t n) {
    int64_t b = (n + 255) / 256;
    return (unsigned)(b < 1 ? 1 : b > 148 * 16 ? 148 * 16 : b);
}

int32_t pairs_pack(net* h, const void* soa, void* pairs) {
    if (h->desc.dtype == NET_F32) pack_kernel<float><<<l2_grid_for(h->n), 256, 0, h->stream>>>((const float*)soa, (float*)pairs, h->n, h->ld);
    else pack_kernel<double><<<l2_grid_for(h->n), 256, 0, h->stream>>>((const double*)soa, (double*)pairs, h->n, h->ld);
    h->launches += 1;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}
int32_t pairs_unpack(net* h, const void* pairs, void* soa) {
    if (h->desc.dtype == NET_F32) unpack_kernel<float><<<l2_grid_for(h->n), 256, 0, h->stream>>>((const float*)pairs, (float*)soa, h->n, h->ld);
    else unpack_kernel<double><<<l2_grid_for(h->n), 256, 0, h->stream>>>((const double*)pairs, (double*)soa, h->n, h->ld);
    h->launches += 1;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}
int32_t lattice_v2_refresh_exchange(net* h) {
    if (h->desc.model != NET_MODEL_KS) return NET_OK;
    if (h->desc.dtype == NET_F32) ks_exchange_kernel<float><<<l2_grid_for(h->n), 256, 0, h->stream>>>((const float*)h->b.y, (float*)h->E_a, h->n);
    else ks_exchange_kernel<double><<<l2_grid_for(h->n), 256, 0, h->stream>>>((const double*)h->b.y, (double*)h->E_a, h->n);
    h->launches += 1;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

}  // namespace oscnet
