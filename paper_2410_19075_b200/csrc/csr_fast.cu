// FAST method for graph topologies (CSR given at run time or the seeded random graph):
// warp-per-row gathers.  A block owns ROWS consecutive rows.  Phase 1: each warp walks its
// share of the rows; the 32 lanes read 32 consecutive col_idx (coalesced, streamed once from
// HBM) and gather the neighbours' exchange variable (L2-resident), then reduce by shuffles.
// Phase 2: one thread per row evaluates the local vector field and the fused RK4 stage update
// with all lanes busy.  For HH the gathered quantity is the precomputed synaptic activation
// s_j = S(V_j) that the producing stage wrote next to its output, so each of the Omega terms
// costs one 8-byte gather instead of an exp (eq. (1); rows are in-neighbour
// lists).
#include "models.cuh"

namespace oscnet {

constexpr int CSR_THREADS = 256;
constexpr int CSR_ROWS = 256;

template <class T, int MODEL>
__global__ void __launch_bounds__(CSR_THREADS) csr_warp_stage_kernel(StageArgs a, ModelParams mp, TopoView tv) {
    constexpr int NS = MODEL == NET_MODEL_FHN ? 2 : 1;  // sums per row
    __shared__ T sums[NS][CSR_ROWS];
    __shared__ int degs[CSR_ROWS];
    const int64_t n = a.n, ld = a.ld;
    const T* __restrict__ in = (const T*)a.in;
    // gathered quantity: HH the precomputed S(V_j); HHS the presynaptic gate s_j (state variable 4);
    // KS / KSI the phase; FHN u (and v)
    const T* __restrict__ gsrc = MODEL == NET_MODEL_HH ? (const T*)a.s_in : MODEL == NET_MODEL_HHS ? in + 4 * ld : in;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    constexpr int NW = CSR_THREADS / 32;
    const int ku = tv.k_uniform;
    const int64_t nblk = (n + CSR_ROWS - 1) / CSR_ROWS;
    for (int64_t blk = blockIdx.x; blk < nblk; blk += gridDim.x) {
        const int64_t row0 = blk * CSR_ROWS;
        // ---- phase 1: gather
        for (int r = warp; r < CSR_ROWS; r += NW) {
            const int64_t i = row0 + r;
            if (i >= n) break;
            int64_t b, e;
            if (ku > 0) { b = i * (int64_t)ku; e = b + ku; }
            else { b = tv.row_ptr[i]; e = tv.row_ptr[i + 1]; }
            T s0 = 0, s1 = 0;
            T pa = 0;
            if (MODEL == NET_MODEL_KS || MODEL == NET_MODEL_KSI) pa = in[i] + T(mp.alpha);
            // warp-uniform trip count; up to four independent gathers in flight per lane
#pragma unroll 1
            for (int64_t qb = b + lane; qb - lane < e; qb += 128) {
                int32_t j[4];
                T g[4], g2[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) j[u] = (qb + 32 * u < e) ? __ldcs(tv.col_idx + qb + 32 * u) : -1;
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    g[u] = j[u] >= 0 ? gsrc[j[u]] : T(0);
                    if (MODEL == NET_MODEL_FHN) g2[u] = j[u] >= 0 ? in[ld + j[u]] : T(0);
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    if (MODEL == NET_MODEL_KS || MODEL == NET_MODEL_KSI) s0 += j[u] >= 0 ? Math<T>::sin(g[u] - pa) : T(0);
                    else {
                        s0 += g[u];
                        if (MODEL == NET_MODEL_FHN) s1 += g2[u];
                    }
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                s0 += __shfl_xor_sync(0xffffffffu, s0, o);
                if (NS == 2) s1 += __shfl_xor_sync(0xffffffffu, s1, o);
            }
            if (lane == 0) {
                sums[0][r] = s0;
                if (NS == 2) sums[NS - 1][r] = s1;
                degs[r] = (int)(e - b);
            }
        }
        __syncthreads();
        // ---- phase 2: local field + stage update, one thread per row
        {
            const int r = threadIdx.x;
            const int64_t i = row0 + r;
            if (i < n) {
                constexpr int NV = MODEL == NET_MODEL_KS ? 1 : (MODEL == NET_MODEL_FHN || MODEL == NET_MODEL_KSI) ? 2 : MODEL == NET_MODEL_HHS ? 5 : 4;
                T xin[NV], k[NV];
#pragma unroll
                for (int v = 0; v < NV; ++v) xin[v] = in[v * ld + i];
                const int deg = degs[r];
                const T inv = deg > 0 ? T(1) / T(deg) : T(0);
                const T* ep = (const T*)a.elem_param;
                if (MODEL == NET_MODEL_KS) {
                    k[0] = ks_rhs_direct<T>(mp, ep[i], sums[0][r], inv);
                } else if (MODEL == NET_MODEL_KSI) {       // eq. (3) in full: psi is a local variable
                    k[0] = xin[NV - 1];
                    k[NV - 1] = (ks_rhs_direct<T>(mp, ep[i], sums[0][r], inv) - T(mp.damp) * xin[NV - 1]) * T(mp.inv_m);
                } else if (MODEL == NET_MODEL_FHN) {
                    T Cu = sums[0][r] - T(deg) * xin[0];
                    T Cv = sums[NS - 1][r] - T(deg) * xin[1];
                    fhn_rhs<T>(mp, xin[0], xin[1], Cu, Cv, inv, &k[0], &k[1]);
                } else {
                    hh_rhs<T>(mp, xin[0], xin[1], xin[2], xin[3], ep[i], sums[0][r], inv, &k[0],
                              &k[1], &k[2], &k[3]);
                    if (MODEL == NET_MODEL_HHS)            // gating ODE of eq. (1), reading R18
                        k[NV - 1] = T(mp.a_s) * hh_syn_activation<T>(mp, xin[0]) * (T(1) - xin[NV - 1]) - T(mp.b_s) * xin[NV - 1];
                }
                const int stage = a.stage;
                const T dt = (T)a.dt;
                T* out = (T*)a.out;
#pragma unroll
                for (int v = 0; v < NV; ++v) {
                    T y = 0, y2 = 0, y3 = 0;
                    if (stage != STAGE_RHS_ONLY) y = ((const T*)a.y)[v * ld + i];
                    if (stage == 3) { y2 = ((const T*)a.Y2)[v * ld + i]; y3 = ((const T*)a.Y3)[v * ld + i]; }
                    T o = stage_combine<T>(stage, dt, k[v], y, y2, y3, xin[v]);
                    out[v * ld + i] = o;
                    if (MODEL == NET_MODEL_HH && v == 0 && a.s_out)
                        ((T*)a.s_out)[i] = hh_syn_activation<T>(mp, o);
                }
            }
        }
        __syncthreads();
    }
}

template <class T>
static int32_t launch(net* h, const StageArgs& a) {
    int64_t nblk = (a.n + CSR_ROWS - 1) / CSR_ROWS;
    unsigned g = (unsigned)(nblk < 148 * 8 ? nblk : 148 * 8);
    switch (h->desc.model) {
        case NET_MODEL_KS: csr_warp_stage_kernel<T, NET_MODEL_KS><<<g, CSR_THREADS, 0, h->stream>>>(a, h->mp, h->tv); break;
        case NET_MODEL_FHN: csr_warp_stage_kernel<T, NET_MODEL_FHN><<<g, CSR_THREADS, 0, h->stream>>>(a, h->mp, h->tv); break;
        case NET_MODEL_KSI: csr_warp_stage_kernel<T, NET_MODEL_KSI><<<g, CSR_THREADS, 0, h->stream>>>(a, h->mp, h->tv); break;
        case NET_MODEL_HHS: csr_warp_stage_kernel<T, NET_MODEL_HHS><<<g, CSR_THREADS, 0, h->stream>>>(a, h->mp, h->tv); break;
        default: csr_warp_stage_kernel<T, NET_MODEL_HH><<<g, CSR_THREADS, 0, h->stream>>>(a, h->mp, h->tv); break;
    }
    h->launches += 1;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

int32_t csr_warp_stage(net* h, const StageArgs& a) {
    return h->desc.dtype == NET_F32 ? launch<float>(h, a) : launch<double>(h, a);
}

}  // namespace oscnet
