// FAST method for large graph topologies, second generation (config 4): column-blocked gathers
// from shared memory.
//
// What bounds the warp-per-row kernel (csr_fast.cu) on B200 is not HBM but the L1TEX t-stage:
// every one of the Omega gathers per row is its own 32-byte sector, about 1.5 cycles per gather
// and SM whether it hits L1, L2 or neither (profiles/r01_lat3_ncu.md, cfg 4).  Random 8-byte
// reads from SHARED memory cost 0.2 cycles.  So the exchange variable s_j = S(V_j) (eq. (1),
// PAPER.md:48-60; one value per element, written by the producing stage) is staged through
// shared memory block by block:
//   * the columns are cut into B blocks of W elements (the s block of W values fills the shared
//     memory of a CTA), the rows into chunks of up to 8192 (one persistent CTA of 1024 threads
//     each; thread t owns rows t, t + 1024, ... of its chunk and keeps their sums in registers
//     for the whole stage);
//   * once per net the CSR arrays are re-ordered into a blocked ELL form: for every (chunk c,
//     block b, row l) FOUR 16-bit slots (one 8-byte word, coalesced across the rows of a warp)
//     holding the first four sources of row l that lie in block b, as indices local to the block;
//     unused slots point at one of the zeros that follow the block (one per bank), so the gather
//     loop has no branch and no trip count; the order of the slots of a word is chosen against
//     shared-memory bank conflicts (cb_place_slots).  The few entries beyond four per (row, block) -- 5 % on config 4 -- go to a
//     per-row overflow list and are gathered from global memory after the last block;
//   * per stage a CTA walks b = 0..B-1: bulk-copy s[b*W .. (b+1)*W) into shared memory
//     (cp.async.bulk on an mbarrier; all CTAs read the same block at about the same time, L2
//     serves it) while the threads fetch their slot words, then four shared-memory gathers per row;
//   * after the last block the thread adds its overflow entries, evaluates the local vector
//     field and the fused RK4 stage update of its rows (coalesced: consecutive threads own
//     consecutive rows).
// Rows are in-neighbour lists; the sum is reordered only by block, which is
// within the summation-order freedom of DESIGN.md R12.
#include <stdlib.h>

#include "lat_common.cuh"

namespace oscnet {

constexpr int CB_THREADS = 1024;
constexpr int CB_MMAX = 8;                 // rows per thread
constexpr int CB_SLOTS = 4;                // 16-bit slots per (row, block)
constexpr unsigned CB_COPY = 32768;        // bytes per bulk copy

struct CbGeom {
    int64_t n;
    int32_t W, B;                // columns per block, number of blocks
    int32_t CR, nchunks, M;      // rows per chunk (multiple of 32), chunks, rows per thread
    const uint2* slots;          // [nchunks][B][CR] words of four 16-bit local indices
    const int32_t* ovf_ptr;      // [nchunks * CR + 1] overflow list of every row
    const int32_t* ovf_idx;      // global source indices
    void* partial;               // pair kernel: [nchunks * CR] sums of the partner's half of the blocks
    unsigned* pair_flag;         // pair kernel: [nchunks] launches completed by every CTA
};

__device__ __forceinline__ void cb_bulk_load(void* dst, const void* src, unsigned bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void cb_prefetch_l2(const void* src, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ double cb_lds(unsigned addr, double) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ float cb_lds(unsigned addr, float) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}

// ------------------------------------------------------------------ build kernels (once per net)
// One thread per (padded) row walks its sorted entries once: the first CB_SLOTS sources of every
// column block go to the slot word of (chunk, block, row), the rest are counted (FILL = false)
// or written to the row's overflow list (FILL = true).  flag[4] != 0: rows not sorted by column.
// Slot order (FILL = false).  The stage kernel reads slot k of NBK consecutive rows with one
// shared-memory wavefront if their addresses fall into different banks (NBK = 128 bytes / element:
// the 16 lanes of a half-warp for fp64, the 32 lanes of a warp for fp32); random sources made
// 52 % of the wavefronts of config 4 bank conflicts (profiles/r01_final_ncu.md).  Which of the
// four slots of a word holds which source is free, and so is the bank of the zero an unused slot
// points at (NBK zeros follow the s block), so the rows of a group are placed one after the
// other, each taking the permutation of its sources that collides least with the rows before it.
__device__ const unsigned char CB_PERM[24][4] = {
    {0, 1, 2, 3}, {0, 1, 3, 2}, {0, 2, 1, 3}, {0, 2, 3, 1}, {0, 3, 1, 2}, {0, 3, 2, 1}, {1, 0, 2, 3}, {1, 0, 3, 2},
    {1, 2, 0, 3}, {1, 2, 3, 0}, {1, 3, 0, 2}, {1, 3, 2, 0}, {2, 0, 1, 3}, {2, 0, 3, 1}, {2, 1, 0, 3}, {2, 1, 3, 0},
    {2, 3, 0, 1}, {2, 3, 1, 0}, {3, 0, 1, 2}, {3, 0, 2, 1}, {3, 1, 0, 2}, {3, 1, 2, 0}, {3, 2, 0, 1}, {3, 2, 1, 0}};

__device__ __forceinline__ void cb_place_slots(unsigned (&s)[CB_SLOTS], int n, unsigned W, int nbk, bool arrange) {
    if (!arrange) return;
    const int lane = threadIdx.x & 31, gbase = lane / nbk * nbk;
    const unsigned all = nbk == 32 ? 0xffffffffu : (1u << nbk) - 1u;
    unsigned mask[CB_SLOTS] = {0u, 0u, 0u, 0u};      // banks taken at slot position k by the rows placed so far
    int zb[CB_SLOTS] = {-1, -1, -1, -1};             // bank of the zero the unused slots at position k read
    unsigned out[CB_SLOTS] = {s[0], s[1], s[2], s[3]};
    for (int j = 0; j < nbk; ++j) {
        if (lane - gbase == j) {
            int best = 0, bestc = 1 << 30;
            for (int p = 0; p < 24; ++p) {
                int cst = 0;
                for (int e = 0; e < n; ++e) cst += (int)((mask[CB_PERM[p][e]] >> (s[e] % (unsigned)nbk)) & 1u);
                if (cst < bestc) { bestc = cst; best = p; }
            }
            bool used[CB_SLOTS] = {false, false, false, false};
            for (int e = 0; e < n; ++e) {
                const int pos = CB_PERM[best][e];
                out[pos] = s[e]; used[pos] = true;
                mask[pos] |= 1u << (s[e] % (unsigned)nbk);
            }
            for (int pos = 0; pos < CB_SLOTS; ++pos)
                if (!used[pos]) {
                    if (zb[pos] < 0) {
                        const unsigned fr = ~mask[pos] & all;
                        zb[pos] = fr ? __ffs((int)fr) - 1 : 0;
                        mask[pos] |= 1u << zb[pos];
                    }
                    out[pos] = W + (unsigned)zb[pos];
                }
        }
#pragma unroll
        for (int k = 0; k < CB_SLOTS; ++k) {
            mask[k] = __shfl_sync(0xffffffffu, mask[k], gbase + j);
            zb[k] = __shfl_sync(0xffffffffu, zb[k], gbase + j);
        }
    }
#pragma unroll
    for (int k = 0; k < CB_SLOTS; ++k) s[k] = out[k];
}

template <bool FILL>
__global__ void cb_build_kernel(CbGeom g, const int64_t* __restrict__ row_ptr, const int32_t* __restrict__ col_idx,
                                int32_t ku, uint2* slots, int32_t* ovf_cnt, const int32_t* __restrict__ ovf_ptr,
                                int32_t* ovf_idx, int64_t ovf_cap, int32_t* flag, int nbk) {
    // whole warps walk the loops together: rows are padded to multiples of 32 per chunk
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < (int64_t)g.nchunks * g.CR;
         i += (int64_t)gridDim.x * blockDim.x) {
        const int c = (int)(i / g.CR), l = (int)(i % g.CR);      // chunks are contiguous ranges of CR rows
        int64_t q = 0, e0 = 0;
        if (i < g.n) {
            if (ku > 0) { q = i * (int64_t)ku; e0 = q + ku; }
            else { q = row_ptr[i]; e0 = row_ptr[i + 1]; }
        }
        int64_t nov = 0;
        const int64_t obase = FILL ? (int64_t)ovf_ptr[i] : 0;
        for (int b = 0; b < g.B; ++b) {
            const int64_t lo = (int64_t)b * g.W, hi = lo + g.W;
            unsigned s[CB_SLOTS];
#pragma unroll
            for (int k = 0; k < CB_SLOTS; ++k) s[k] = (unsigned)g.W;
            int cnt = 0;
            while (q < e0 && col_idx[q] < hi) {
                const int32_t j = col_idx[q++];
                if (j < lo) atomicExch(flag + 4, 2);             // not sorted
#pragma unroll
                for (int k = 0; k < CB_SLOTS; ++k)
                    if (cnt == k) s[k] = (unsigned)(j - lo);
                if (cnt >= CB_SLOTS) {
                    if (FILL && obase + nov < ovf_cap) ovf_idx[obase + nov] = j;
                    ++nov;
                }
                ++cnt;
            }
            if (!FILL) {
                __syncwarp();
                cb_place_slots(s, cnt < CB_SLOTS ? cnt : CB_SLOTS, (unsigned)g.W, nbk, nbk > 0);
                slots[((int64_t)c * g.B + b) * g.CR + l] = make_uint2(s[0] | s[1] << 16, s[2] | s[3] << 16);
            }
        }
        if (q != e0) atomicExch(flag + 4, 2);
        if (!FILL) ovf_cnt[i] = (int32_t)(nov > 0x7fffffff ? 0x7fffffff : nov);
    }
}

// exclusive scan of int32 counts into ptr[0..n] (one CTA); total > cap sets flag[4] = 3
__global__ void __launch_bounds__(1024) cb_scan_kernel(int64_t n, const int32_t* cnt, int32_t* ptr, int64_t cap, int32_t* flag) {
    __shared__ int64_t wsum[32];
    __shared__ int64_t carry_s;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int64_t base = 0; base < n; base += 1024) {
        const int64_t s = base + threadIdx.x;
        const int64_t own = s < n ? cnt[s] : 0;
        int64_t v = own;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int64_t u = __shfl_up_sync(0xffffffffu, v, o);
            if (lane >= o) v += u;
        }
        if (lane == 31) wsum[warp] = v;
        __syncthreads();
        int64_t off = carry_s;
        for (int w = 0; w < warp; ++w) off += wsum[w];
        v += off;
        if (s < n) ptr[s] = (int32_t)((v - own) > cap ? cap : (v - own));
        __syncthreads();
        if (threadIdx.x == 1023) carry_s = v;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        if (carry_s > cap) atomicExch(flag + 4, 3);
        ptr[n] = (int32_t)(carry_s > cap ? cap : carry_s);
        flag[5] = (int32_t)(carry_s > 0x7fffffff ? 0x7fffffff : carry_s);
    }
}

// ------------------------------------------------------------------ stage kernel
// Local vector field + fused RK4 stage update of row i given its gathered sum (HH: sum of s_j).
template <class T>
__device__ __forceinline__ void cb_finish_hh(const StageArgs& a, const ModelParams& mp, int64_t i, T ssum, int deg) {
    const int64_t ld = a.ld;
    const T* __restrict__ in = (const T*)a.in;
    T xin[4], k[4];
#pragma unroll
    for (int v = 0; v < 4; ++v) xin[v] = in[v * ld + i];
    const T inv = deg > 0 ? T(1) / T(deg) : T(0);
    hh_rhs<T>(mp, xin[0], xin[1], xin[2], xin[3], ((const T*)a.elem_param)[i], ssum, inv, &k[0], &k[1], &k[2], &k[3]);
    const int stage = a.stage;
    const T dt = (T)a.dt;
    T* out = (T*)a.out;
#pragma unroll
    for (int v = 0; v < 4; ++v) {
        T y = 0, y2 = 0, y3 = 0;
        if (stage != STAGE_RHS_ONLY) y = ((const T*)a.y)[v * ld + i];
        if (stage == 3) { y2 = ((const T*)a.Y2)[v * ld + i]; y3 = ((const T*)a.Y3)[v * ld + i]; }
        const T o = stage_combine<T>(stage, dt, k[v], y, y2, y3, xin[v]);
        out[v * ld + i] = o;
        if (v == 0 && a.s_out) ((T*)a.s_out)[i] = hh_syn_activation<T>(mp, o);
    }
}

template <class T, int M>
__global__ void __launch_bounds__(CB_THREADS, 1)
csr_blocked_stage_kernel(StageArgs a, ModelParams mp, TopoView tv, CbGeom g) {
    extern __shared__ __align__(128) unsigned char cb_smem[];
    __shared__ uint64_t bar;
    constexpr unsigned SH = sizeof(T) == 8 ? 3u : 2u;          // index -> byte offset
    constexpr unsigned MASK = 0xffffu << SH;
    T* sblk = reinterpret_cast<T*>(cb_smem);                   // W values of s, then the zero slot
    const unsigned sblk_a = smem_u32(cb_smem);
    const T* __restrict__ gsrc = (const T*)a.s_in;
    const int t = threadIdx.x;
    if (t == 0) {
        mbar_init(&bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (t < 128 / (int)sizeof(T)) sblk[g.W + t] = T(0);          // one zero per bank for the unused slots
    __syncthreads();
    unsigned phase = 0;
    for (int c = blockIdx.x; c < g.nchunks; c += gridDim.x) {
        const int64_t row0 = (int64_t)c * g.CR;
        T acc[M];
#pragma unroll
        for (int m = 0; m < M; ++m) acc[m] = T(0);
        for (int b = 0; b < g.B; ++b) {
            const int64_t col0 = (int64_t)b * g.W;
            const uint2* __restrict__ sl = g.slots + ((int64_t)c * g.B + b) * g.CR;
            __syncthreads();                       // every thread is done with the previous block
            if (t == 0) {
                const int64_t cnt = g.n - col0 < g.W ? g.n - col0 : g.W;
                constexpr int V = 16 / (int)sizeof(T);
                const unsigned bytes = (unsigned)((cnt + V - 1) / V * V * sizeof(T));   // inside ld (multiple of 64)
                mbar_expect_tx(&bar, bytes);
                for (unsigned o = 0; o < bytes; o += CB_COPY)
                    cb_bulk_load(cb_smem + o, (const unsigned char*)(gsrc + col0) + o, bytes - o < CB_COPY ? bytes - o : CB_COPY, &bar);
            } else if (t == 32 && b + 1 < g.B) {   // next block's slot words towards L2
                cb_prefetch_l2(sl + g.CR, (unsigned)((size_t)g.CR * sizeof(uint2)));
            }
            // while the block is in flight: this thread's slot words (coalesced, 8 bytes per row)
            uint2 w[M];
#pragma unroll
            for (int m = 0; m < M; ++m) {
                const int l = m * CB_THREADS + t;
                w[m] = l < g.CR ? __ldg(sl + l) : make_uint2((unsigned)g.W * 0x10001u, (unsigned)g.W * 0x10001u);
            }
            mbar_wait(&bar, phase);
            phase ^= 1u;
#pragma unroll
            for (int m = 0; m < M; ++m) {
                const T v0 = cb_lds(sblk_a + ((w[m].x << SH) & MASK), T(0));
                const T v1 = cb_lds(sblk_a + ((w[m].x >> (16 - SH)) & MASK), T(0));
                const T v2 = cb_lds(sblk_a + ((w[m].y << SH) & MASK), T(0));
                const T v3 = cb_lds(sblk_a + ((w[m].y >> (16 - SH)) & MASK), T(0));
                acc[m] += (v0 + v1) + (v2 + v3);
            }
        }
        // ---- overflow entries, local field + stage update of this thread's rows
#pragma unroll
        for (int m = 0; m < M; ++m) {
            const int l = m * CB_THREADS + t;
            const int64_t i = row0 + l;
            if (l >= g.CR || i >= g.n) continue;
            T sum = acc[m];
            const int q1 = g.ovf_ptr[i + 1];
            for (int q = g.ovf_ptr[i]; q < q1; ++q) sum += gsrc[g.ovf_idx[q]];
            const int deg = tv.k_uniform > 0 ? tv.k_uniform : (int)(tv.row_ptr[i + 1] - tv.row_ptr[i]);
            cb_finish_hh<T>(a, mp, i, sum, deg);
        }
    }
}

// Pair form (2D partition).  What bounds the kernel above on config 4 is the L2 -> SM traffic of
// the s blocks: each of the 148 CTAs streams ALL of s every stage (1.18 GB).  Here CTAs 2p and
// 2p + 1 both take the rows of chunks 2p AND 2p + 1 but only one half of the column blocks each,
// so every CTA streams half of s (the slot-word and gather work per CTA is unchanged); the two
// halves of every row sum meet through global memory: each CTA publishes its sums for the
// partner's chunk, raises its launch counter (release), waits for the partner's (acquire) and
// finishes its own chunk as  (blocks of the lower half) + (blocks of the upper half).  The launch
// is cooperative, so the two CTAs of a pair are co-resident.
__device__ __forceinline__ unsigned cb_ld_acquire(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void cb_st_release(unsigned* p, unsigned v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

template <class T, int M>
__global__ void __launch_bounds__(CB_THREADS, 1)
csr_blocked_pair_kernel(StageArgs a, ModelParams mp, TopoView tv, CbGeom g) {
    extern __shared__ __align__(128) unsigned char cb_smem[];
    __shared__ uint64_t bar;
    __shared__ unsigned epoch_s;
    constexpr unsigned SH = sizeof(T) == 8 ? 3u : 2u;
    constexpr unsigned MASK = 0xffffu << SH;
    T* sblk = reinterpret_cast<T*>(cb_smem);
    const unsigned sblk_a = smem_u32(cb_smem);
    const T* __restrict__ gsrc = (const T*)a.s_in;
    const int t = threadIdx.x;
    const int pair = blockIdx.x >> 1, half = blockIdx.x & 1;
    if (t == 0) {
        mbar_init(&bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        epoch_s = g.pair_flag[blockIdx.x] + 1u;        // launches are stream-ordered: the partner's counter is at the same value
    }
    if (t < 128 / (int)sizeof(T)) sblk[g.W + t] = T(0);
    __syncthreads();
    const int bh = (g.B + 1) / 2;
    const int b_lo = half ? bh : 0, b_hi = half ? g.B : bh;
    unsigned phase = 0;
    T acc0[M], acc1[M];                                // rows of chunk 2p, of chunk 2p + 1
#pragma unroll
    for (int m = 0; m < M; ++m) { acc0[m] = T(0); acc1[m] = T(0); }
    for (int b = b_lo; b < b_hi; ++b) {
        const int64_t col0 = (int64_t)b * g.W;
        const uint2* __restrict__ sl0 = g.slots + ((int64_t)(2 * pair) * g.B + b) * g.CR;
        const uint2* __restrict__ sl1 = g.slots + ((int64_t)(2 * pair + 1) * g.B + b) * g.CR;
        __syncthreads();                           // every thread is done with the previous block
        if (t == 0) {
            const int64_t cnt = g.n - col0 < g.W ? g.n - col0 : g.W;
            constexpr int V = 16 / (int)sizeof(T);
            const unsigned bytes = (unsigned)((cnt + V - 1) / V * V * sizeof(T));
            mbar_expect_tx(&bar, bytes);
            for (unsigned o = 0; o < bytes; o += CB_COPY)
                cb_bulk_load(cb_smem + o, (const unsigned char*)(gsrc + col0) + o, bytes - o < CB_COPY ? bytes - o : CB_COPY, &bar);
        } else if (b + 1 < b_hi && (t == 32 || t == 64)) {   // next block's slot words towards L2
            cb_prefetch_l2((t == 32 ? sl0 : sl1) + g.CR, (unsigned)((size_t)g.CR * sizeof(uint2)));
        }
        uint2 w[M], u[M];                          // both chunks' slot words are in flight while the block arrives
#pragma unroll
        for (int m = 0; m < M; ++m) {
            const int l = m * CB_THREADS + t;
            w[m] = l < g.CR ? __ldg(sl0 + l) : make_uint2((unsigned)g.W * 0x10001u, (unsigned)g.W * 0x10001u);
            u[m] = l < g.CR ? __ldg(sl1 + l) : make_uint2((unsigned)g.W * 0x10001u, (unsigned)g.W * 0x10001u);
        }
        mbar_wait(&bar, phase);
        phase ^= 1u;
#pragma unroll
        for (int m = 0; m < M; ++m) {
            const T v0 = cb_lds(sblk_a + ((w[m].x << SH) & MASK), T(0));
            const T v1 = cb_lds(sblk_a + ((w[m].x >> (16 - SH)) & MASK), T(0));
            const T v2 = cb_lds(sblk_a + ((w[m].y << SH) & MASK), T(0));
            const T v3 = cb_lds(sblk_a + ((w[m].y >> (16 - SH)) & MASK), T(0));
            acc0[m] += (v0 + v1) + (v2 + v3);
            const T x0 = cb_lds(sblk_a + ((u[m].x << SH) & MASK), T(0));
            const T x1 = cb_lds(sblk_a + ((u[m].x >> (16 - SH)) & MASK), T(0));
            const T x2 = cb_lds(sblk_a + ((u[m].y << SH) & MASK), T(0));
            const T x3 = cb_lds(sblk_a + ((u[m].y >> (16 - SH)) & MASK), T(0));
            acc1[m] += (x0 + x1) + (x2 + x3);
        }
    }
    // ---- publish the sums of the partner's chunk, wait for the partner's sums of mine
    const int c_own = 2 * pair + half, c_other = 2 * pair + (1 - half);
    T* part = (T*)g.partial;
#pragma unroll
    for (int m = 0; m < M; ++m) {
        const int l = m * CB_THREADS + t;
        if (l < g.CR) __stcg(part + (int64_t)c_other * g.CR + l, half ? acc0[m] : acc1[m]);
    }
    __threadfence();
    __syncthreads();
    if (t == 0) {
        const unsigned epoch = epoch_s;
        cb_st_release(g.pair_flag + blockIdx.x, epoch);
        while (cb_ld_acquire(g.pair_flag + (blockIdx.x ^ 1)) < epoch) {}
    }
    __syncthreads();
    const int64_t row0 = (int64_t)c_own * g.CR;
#pragma unroll
    for (int m = 0; m < M; ++m) {
        const int l = m * CB_THREADS + t;
        const int64_t i = row0 + l;
        if (l >= g.CR || i >= g.n) continue;
        const T mine = half ? acc1[m] : acc0[m];
        const T theirs = __ldcg(part + row0 + l);
        T sum = half ? theirs + mine : mine + theirs;      // lower half of the blocks + upper half
        const int q1 = g.ovf_ptr[i + 1];
        for (int q = g.ovf_ptr[i]; q < q1; ++q) sum += gsrc[g.ovf_idx[q]];
        const int deg = tv.k_uniform > 0 ? tv.k_uniform : (int)(tv.row_ptr[i + 1] - tv.row_ptr[i]);
        cb_finish_hh<T>(a, mp, i, sum, deg);
    }
}

// ------------------------------------------------------------------ host side
constexpr size_t CB_SMEM_BUDGET = 224 * 1024;   // of the 227 KB a CTA may own

static int64_t cb_nnz(const net_desc* d) {
    return d->topo.kind == NET_TOPO_CSR ? d->topo.nnz : d->n * (int64_t)d->topo.in_degree;
}

// Geometry from the descriptor alone (the workspace query has no device).  W: as many columns as
// the shared memory takes, but no more than keep the mean number of sources per (row, block)
// near 2.2, so that the four slots hold all but a few per cent of the entries.  Chunks of rows so
// that one wave of persistent CTAs covers the net.  OSCNET_CSRB = "W,CR" overrides (tests use it
// to get several blocks and chunks on small nets).
static bool cb_geometry(const net_desc* d, CbGeom* g) {
    const net_topology& t = d->topo;
    if (d->model != NET_MODEL_HH) return false;
    if (t.kind != NET_TOPO_CSR && t.kind != NET_TOPO_RANDOM_INDEGREE) return false;
    const int64_t n = d->n;
    const size_t es = d->dtype == NET_F32 ? 4 : 8;
    int want_w = 0, want_cr = 0;
    if (const char* e = getenv("OSCNET_CSRB")) sscanf(e, "%d,%d", &want_w, &want_cr);
    if (want_w <= 0 && n < 32768) return false;          // small nets: the warp-per-row kernel
    if (cb_nnz(d) > 0x7fffffffLL) return false;           // 32-bit overflow pointers
    const int sms = 148;
    int64_t CR = round_up((n + sms - 1) / sms, 32);
    if (want_cr > 0) CR = round_up(want_cr, 32);
    if (CR > CB_MMAX * CB_THREADS) CR = CB_MMAX * CB_THREADS;
    const int64_t nchunks = (n + CR - 1) / CR;
    int W = (int)(CB_SMEM_BUDGET / es) - 32;
    if (W > 65488) W = 65488;                             // W .. W + 31 are the indices of the zero slots
    int B = (int)((n + W - 1) / W);
    const double mean_deg = (double)cb_nnz(d) / (double)n;
    const int B_fill = (int)(mean_deg / 2.2 + 0.999);     // blocks that bring the mean per slot word to 2.2
    if (B_fill > B) B = B_fill;
    if (B > n / 16) B = (int)(n / 16 > 0 ? n / 16 : 1);
    W = (int)round_up((n + B - 1) / B, 16);               // equal blocks, 16-element granules
    if (want_w > 0) W = (int)round_up(want_w < 16 ? 16 : (want_w > 65488 ? 65488 : want_w), 16);
    B = (int)((n + W - 1) / W);
    if (nchunks * B > (int64_t)1 << 24) return false;
    memset(g, 0, sizeof(*g));
    g->n = n; g->W = W; g->B = B; g->CR = (int)CR; g->nchunks = (int)nchunks;
    g->M = (int)((CR + CB_THREADS - 1) / CB_THREADS);
    return true;
}

bool csr_blocked_supported(const net_desc* d) {
    CbGeom g;
    return cb_geometry(d, &g);
}

// scratch: slots | ovf_ptr | ovf_cnt | ovf_idx.  The overflow list may take a quarter of nnz;
// a graph that needs more (far from uniform rows) goes back to the warp-per-row kernel.
struct CbLayout { size_t slots, ovf_ptr, ovf_cnt, ovf_idx, partial, pair_flag, total; int64_t ovf_cap; };
static CbLayout cb_layout(const net_desc* d, const CbGeom& g) {
    CbLayout L;
    size_t cur = 0;
    auto take = [&](size_t bytes) { size_t at = cur; cur += (bytes + 255) / 256 * 256; return at; };
    const size_t rows = (size_t)g.nchunks * g.CR;
    L.ovf_cap = cb_nnz(d) / 4 + 1024;
    L.slots = take(rows * (size_t)g.B * sizeof(uint2));
    L.ovf_ptr = take((rows + 1) * sizeof(int32_t));
    L.ovf_cnt = take((rows + 1) * sizeof(int32_t));
    L.ovf_idx = take((size_t)L.ovf_cap * sizeof(int32_t));
    L.partial = take(rows * (d->dtype == NET_F32 ? 4 : 8));
    L.pair_flag = take((size_t)g.nchunks * sizeof(unsigned) + 64);
    L.total = cur;
    return L;
}

size_t csr_blocked_scratch_bytes(const net_desc* d) {
    CbGeom g;
    if (!cb_geometry(d, &g)) return 0;
    return cb_layout(d, g).total;
}

template <class T>
static const void* cb_kernel_for(int M) {
    switch (M) {
        case 1: return (const void*)csr_blocked_stage_kernel<T, 1>;
        case 2: return (const void*)csr_blocked_stage_kernel<T, 2>;
        case 3: return (const void*)csr_blocked_stage_kernel<T, 3>;
        case 4: return (const void*)csr_blocked_stage_kernel<T, 4>;
        case 5: return (const void*)csr_blocked_stage_kernel<T, 5>;
        case 6: return (const void*)csr_blocked_stage_kernel<T, 6>;
        case 7: return (const void*)csr_blocked_stage_kernel<T, 7>;
        default: return (const void*)csr_blocked_stage_kernel<T, 8>;
    }
}

template <class T>
static const void* cb_pair_kernel_for(int M) {
    switch (M) {
        case 1: return (const void*)csr_blocked_pair_kernel<T, 1>;
        case 2: return (const void*)csr_blocked_pair_kernel<T, 2>;
        case 3: return (const void*)csr_blocked_pair_kernel<T, 3>;
        case 4: return (const void*)csr_blocked_pair_kernel<T, 4>;
        case 5: return (const void*)csr_blocked_pair_kernel<T, 5>;
        case 6: return (const void*)csr_blocked_pair_kernel<T, 6>;
        case 7: return (const void*)csr_blocked_pair_kernel<T, 7>;
        default: return (const void*)csr_blocked_pair_kernel<T, 8>;
    }
}

// Builds the blocked ELL arrays in the scratch region.  NET_ERR_UNSUPPORTED (rows not sorted,
// overflow list too long) sends the net back to the warp-per-row kernel.
int32_t csr_blocked_prepare(net* h) {
    CbGeom g;
    if (!cb_geometry(&h->desc, &g)) return NET_ERR_UNSUPPORTED;
    const CbLayout L = cb_layout(&h->desc, g);
    if (L.total > h->b.scratch_bytes) return NET_ERR_UNSUPPORTED;
    char* s = (char*)h->b.scratch;
    uint2* slots = (uint2*)(s + L.slots);
    int32_t* ovf_ptr = (int32_t*)(s + L.ovf_ptr);
    int32_t* ovf_cnt = (int32_t*)(s + L.ovf_cnt);
    int32_t* ovf_idx = (int32_t*)(s + L.ovf_idx);
    g.slots = slots; g.ovf_ptr = ovf_ptr; g.ovf_idx = ovf_idx;
    g.partial = s + L.partial; g.pair_flag = (unsigned*)(s + L.pair_flag);
    cudaStream_t st = h->stream;
    OSC_CUDA(h, cudaMemsetAsync(g.pair_flag, 0, (size_t)g.nchunks * sizeof(unsigned), st));
    const int64_t rows = (int64_t)g.nchunks * g.CR;
    const unsigned grid = (unsigned)((rows + 255) / 256 > 148 * 16 ? 148 * 16 : (rows + 255) / 256);
    const int32_t ku = h->tv.k_uniform;
    OSC_CUDA(h, cudaMemsetAsync(h->b.flag + 4, 0, 2 * sizeof(int32_t), st));   // flag[4]: verdict, flag[5]: overflow entries
    const int nbk = getenv("OSCNET_CSRB_NOARRANGE") ? 0 : 128 / (int)h->esize;
    cb_build_kernel<false><<<grid, 256, 0, st>>>(g, h->tv.row_ptr, h->tv.col_idx, ku, slots, ovf_cnt, nullptr, nullptr, 0, h->b.flag, nbk);
    cb_scan_kernel<<<1, 1024, 0, st>>>(rows, ovf_cnt, ovf_ptr, L.ovf_cap, h->b.flag);
    cb_build_kernel<true><<<grid, 256, 0, st>>>(g, h->tv.row_ptr, h->tv.col_idx, ku, nullptr, nullptr, ovf_ptr, ovf_idx, L.ovf_cap, h->b.flag, 0);
    h->launches += 3;
    OSC_CUDA(h, cudaGetLastError());
    int32_t flag[2] = {0, 0};
    OSC_CUDA(h, cudaMemcpyAsync(flag, h->b.flag + 4, sizeof(flag), cudaMemcpyDeviceToHost, st));
    OSC_CUDA(h, cudaStreamSynchronize(st));
    if (flag[0] != 0) return NET_ERR_UNSUPPORTED;
    const size_t smem = ((size_t)g.W + 32) * h->esize;        // + the zero slots
    if (smem > CB_SMEM_BUDGET + 1024) return NET_ERR_UNSUPPORTED;
    const void* kern = h->desc.dtype == NET_F32 ? cb_kernel_for<float>(g.M) : cb_kernel_for<double>(g.M);
    OSC_CUDA(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    static_assert(sizeof(CbGeom) <= sizeof(((net*)0)->cb_geom), "cb_geom storage too small");
    memcpy(h->cb_geom, &g, sizeof(g));
    h->cb_grid = (unsigned)(g.nchunks < sms ? g.nchunks : sms);
    h->cb_smem = smem;
    // pair form: one chunk per CTA, an even number of them, all co-resident (cooperative launch)
    h->cb_pair = 0;
    int coop = 0;
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
    const char* pe = getenv("OSCNET_CSRB_PAIR");
    if (coop && g.nchunks % 2 == 0 && g.nchunks <= sms && g.B >= 2 && !(pe && atoi(pe) == 0)) {
        const void* pk = h->desc.dtype == NET_F32 ? cb_pair_kernel_for<float>(g.M) : cb_pair_kernel_for<double>(g.M);
        int occ = 0;
        if (cudaFuncSetAttribute(pk, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) == cudaSuccess &&
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, pk, CB_THREADS, smem) == cudaSuccess && occ * sms >= g.nchunks)
            h->cb_pair = 1;
        else cudaGetLastError();
    }
    if (getenv("OSCNET_VERBOSE"))
        fprintf(stderr, "csr_blocked: W %d B %d CR %d chunks %d M %d overflow %d of %lld entries smem %zu grid %u scratch %zu pair %d\n",
                g.W, g.B, g.CR, g.nchunks, g.M, flag[1], (long long)h->nnz, smem, h->cb_grid, L.total, h->cb_pair);
    return NET_OK;
}

int32_t csr_blocked_stage(net* h, const StageArgs& a) {
    CbGeom g;
    memcpy(&g, h->cb_geom, sizeof(g));
    const void* kern = h->desc.dtype == NET_F32 ? cb_kernel_for<float>(g.M) : cb_kernel_for<double>(g.M);
    StageArgs aa = a;
    void* params[] = {&aa, &h->mp, &h->tv, &g};
    if (h->cb_pair) {
        const void* pk = h->desc.dtype == NET_F32 ? cb_pair_kernel_for<float>(g.M) : cb_pair_kernel_for<double>(g.M);
        cudaLaunchConfig_t cfg;
        memset(&cfg, 0, sizeof(cfg));
        cfg.gridDim = dim3((unsigned)g.nchunks);
        cfg.blockDim = dim3(CB_THREADS);
        cfg.dynamicSmemBytes = h->cb_smem;
        cfg.stream = h->stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeCooperative;
        attr[0].val.cooperative = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        OSC_CUDA(h, cudaLaunchKernelExC(&cfg, pk, params));
    } else {
        OSC_CUDA(h, cudaLaunchKernel(kern, dim3(h->cb_grid), dim3(CB_THREADS), params, h->cb_smem, h->stream));
    }
    h->launches += 1;
    return NET_OK;
}

}  // namespace oscnet
