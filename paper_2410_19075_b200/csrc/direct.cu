// DIRECT method: one thread per element, one term per neighbour gathered from global
// memory -- the formulation of Alg. 1 fused with the RK4 stage update.
// It is the in-GPU reference the FAST kernels are measured against (error of the rewrite).
#include "models.cuh"

namespace oscnet {

template <class T, int MODEL, int TOPO>
__global__ void __launch_bounds__(256) direct_stage_kernel(StageArgs a, ModelParams mp, TopoView tv) {
    const int64_t n = a.n, ld = a.ld;
    const T* __restrict__ in = (const T*)a.in;
    const T* __restrict__ yb = (const T*)a.y;
    const T* __restrict__ Y2 = (const T*)a.Y2;
    const T* __restrict__ Y3 = (const T*)a.Y3;
    T* __restrict__ out = (T*)a.out;
    const T* __restrict__ ep = (const T*)a.elem_param;
    const int stage = a.stage;
    const T dt = (T)a.dt;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
        constexpr int NV = MODEL == NET_MODEL_KS ? 1 : (MODEL == NET_MODEL_FHN || MODEL == NET_MODEL_KSI) ? 2 : MODEL == NET_MODEL_HHS ? 5 : 4;
        T k[NV], xin[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) xin[v] = in[v * ld + i];
        if (MODEL == NET_MODEL_KS) {
            T sum = 0;
            const T pa = xin[0] + T(mp.alpha);
            int deg = for_each_neighbor<TOPO>(tv, n, i, [&](int64_t j) {
                sum += Math<T>::sin(in[j] - pa);
            });
            T inv = deg > 0 ? T(1) / T(deg) : T(0);
            k[0] = ks_rhs_direct<T>(mp, ep[i], sum, inv);
        } else if (MODEL == NET_MODEL_KSI) {
            // eq. (3) in full: phi' = psi, psi' = (-eps psi + omega + (K/Omega) sum sin(...)) / m
            T sum = 0;
            const T pa = xin[0] + T(mp.alpha);
            int deg = for_each_neighbor<TOPO>(tv, n, i, [&](int64_t j) {
                sum += Math<T>::sin(in[j] - pa);
            });
            T inv = deg > 0 ? T(1) / T(deg) : T(0);
            k[0] = xin[1];
            k[1] = (ks_rhs_direct<T>(mp, ep[i], sum, inv) - T(mp.damp) * xin[1]) * T(mp.inv_m);
        } else if (MODEL == NET_MODEL_FHN) {
            T Cu = 0, Cv = 0;
            int deg = for_each_neighbor<TOPO>(tv, n, i, [&](int64_t j) {
                Cu += in[j] - xin[0];
                Cv += in[ld + j] - xin[1];
            });
            T inv = deg > 0 ? T(1) / T(deg) : T(0);
            fhn_rhs<T>(mp, xin[0], xin[1], Cu, Cv, inv, &k[0], &k[1]);
        } else if (MODEL == NET_MODEL_HHS) {
            // eq. (1) with the gating ODE (reading R18): the links carry the presynaptic gate s_j
            T ssum = 0;
            int deg = for_each_neighbor<TOPO>(tv, n, i, [&](int64_t j) { ssum += in[4 * ld + j]; });
            T inv = deg > 0 ? T(1) / T(deg) : T(0);
            hh_rhs<T>(mp, xin[0], xin[1], xin[2], xin[3], ep[i], ssum, inv, &k[0], &k[1], &k[2], &k[3]);
            k[NV - 1] = T(mp.a_s) * hh_syn_activation<T>(mp, xin[0]) * (T(1) - xin[NV - 1]) - T(mp.b_s) * xin[NV - 1];
        } else {
            T ssum = 0;
            int deg = for_each_neighbor<TOPO>(tv, n, i, [&](int64_t j) {
                ssum += hh_syn_activation<T>(mp, in[j]);
            });
            T inv = deg > 0 ? T(1) / T(deg) : T(0);
            hh_rhs<T>(mp, xin[0], xin[1], xin[2], xin[3], ep[i], ssum, inv, &k[0], &k[1], &k[2],
                      &k[3]);
        }
#pragma unroll
        for (int v = 0; v < NV; ++v) {
            T y = 0, y2 = 0, y3 = 0;
            if (stage != STAGE_RHS_ONLY) y = yb[v * ld + i];
            if (stage == 3) { y2 = Y2[v * ld + i]; y3 = Y3[v * ld + i]; }
            out[v * ld + i] = stage_combine<T>(stage, dt, k[v], y, y2, y3, xin[v]);
        }
    }
}

template <class T, int MODEL>
static int32_t launch_topo(net* h, const StageArgs& a) {
    int64_t blocks = (a.n + 255) / 256;
    if (blocks > 148 * 64) blocks = 148 * 64;
    dim3 g((unsigned)blocks), b(256);
    switch (h->tv.kind) {
        case NET_TOPO_RING:
            direct_stage_kernel<T, MODEL, NET_TOPO_RING><<<g, b, 0, h->stream>>>(a, h->mp, h->tv);
            break;
        case NET_TOPO_LATTICE:
            direct_stage_kernel<T, MODEL, NET_TOPO_LATTICE><<<g, b, 0, h->stream>>>(a, h->mp, h->tv);
            break;
        case NET_TOPO_CSR:
            direct_stage_kernel<T, MODEL, NET_TOPO_CSR><<<g, b, 0, h->stream>>>(a, h->mp, h->tv);
            break;
        case NET_TOPO_COMPRESSED:
            direct_stage_kernel<T, MODEL, NET_TOPO_COMPRESSED><<<g, b, 0, h->stream>>>(a, h->mp, h->tv);
            break;
        default:
            direct_stage_kernel<T, MODEL, NET_TOPO_RANDOM_INDEGREE><<<g, b, 0, h->stream>>>(a, h->mp, h->tv);
            break;
    }
    h->launches += 1;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

template <class T>
static int32_t launch_model(net* h, const StageArgs& a) {
    switch (h->desc.model) {
        case NET_MODEL_KS: return launch_topo<T, NET_MODEL_KS>(h, a);
        case NET_MODEL_FHN: return launch_topo<T, NET_MODEL_FHN>(h, a);
        case NET_MODEL_KSI: return launch_topo<T, NET_MODEL_KSI>(h, a);
        case NET_MODEL_HHS: return launch_topo<T, NET_MODEL_HHS>(h, a);
        default: return launch_topo<T, NET_MODEL_HH>(h, a);
    }
}

int32_t direct_stage(net* h, const StageArgs& a) {
    return h->desc.dtype == NET_F32 ? launch_model<float>(h, a) : launch_model<double>(h, a);
}

// ------------------------------------------------------------------ HH helpers
template <class T>
__global__ void hh_s_kernel(const T* __restrict__ V, T* __restrict__ s, int64_t n, ModelParams mp) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x)
        s[i] = hh_syn_activation<T>(mp, V[i]);
}

int32_t hh_compute_s(net* h, const void* V, void* s) {
    int64_t blocks = (h->n + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    if (h->desc.dtype == NET_F32)
        hh_s_kernel<float><<<(unsigned)blocks, 256, 0, h->stream>>>((const float*)V, (float*)s, h->n, h->mp);
    else
        hh_s_kernel<double><<<(unsigned)blocks, 256, 0, h->stream>>>((const double*)V, (double*)s, h->n, h->mp);
    h->launches += 1;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

template <class T>
__global__ void hh_gates_kernel(T* __restrict__ y, int64_t n, int64_t ld, int with_s, ModelParams mp) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
        T am, bm, ah, bh, an, bn;
        hh_rates<T>(y[i], &am, &bm, &ah, &bh, &an, &bn);
        y[ld + i] = am / (am + bm);
        y[2 * ld + i] = ah / (ah + bh);
        y[3 * ld + i] = an / (an + bn);
        if (with_s) {       // HHS: gating variable at a_s S/(a_s S + b_s)
            const T S = hh_syn_activation<T>(mp, y[i]);
            y[4 * ld + i] = T(mp.a_s) * S / (T(mp.a_s) * S + T(mp.b_s));
        }
    }
}

int32_t hh_steady_gates(net* h) {
    int64_t blocks = (h->n + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    if (h->desc.dtype == NET_F32)
        hh_gates_kernel<float><<<(unsigned)blocks, 256, 0, h->stream>>>((float*)h->b.y, h->n, h->ld, h->desc.model == NET_MODEL_HHS, h->mp);
    else
        hh_gates_kernel<double><<<(unsigned)blocks, 256, 0, h->stream>>>((double*)h->b.y, h->n, h->ld, h->desc.model == NET_MODEL_HHS, h->mp);
    h->launches += 1;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

}  // namespace oscnet
