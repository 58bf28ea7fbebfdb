// FAST method for large graph topologies, second generation (config 4): column-blocked gathers
// from shared memory.
//
// What bounds the warp-per-row kernel (csr_fast.cu) on B200 is not HBM but the L1TEX t-stage:
// every one of the Omega gathers per row is its own 32-byte sector, about 1.5 cycles per gather
// and SM whether it hits L1, L2 or neither (profiles/r01_lat3_ncu.md, cfg 4).  Random 8-byte
// reads from SHARED memory cost 0.2 cycles.  So the exchange variable s_j = S(V_j) (eq. (1),
// PAPER.md:48-60; one value per element, written by the producing stage) is staged through
// shared memory block by block:
//   * the columns are cut into B blocks of W elements (W * sizeof(T) ~ 200 KB), the rows into
//     chunks of up to 8192 (one persistent CTA of 1024 threads each, thread t owns rows
//     t, t + 1024, ... of its chunk and keeps their sums in registers for the whole stage);
//   * once per net the CSR arrays are re-ordered into segments (chunk c, block b): the entries
//     of the chunk's rows whose source lies in block b, row after row, as 16-bit indices local
//     to the block (half the bytes of col_idx) packed two to a 32-bit word (a run of odd length
//     ends with the index W of a slot that holds 0), plus 16-bit row offsets in words;
//   * per stage a CTA walks b = 0..B-1: bulk-copy s[b*W .. (b+1)*W) into shared memory
//     (cp.async.bulk on an mbarrier; all CTAs read the same block at about the same time, L2
//     serves it), then every thread adds the entries of its rows in this block;
//   * after the last block the thread evaluates the local vector field and the fused RK4 stage
//     update of its rows (coalesced: consecutive threads own consecutive rows).
// Rows are in-neighbour lists; the sum is reordered only by block, which is
// within the summation-order freedom of DESIGN.md R12.
#include <stdlib.h>

#include "lat_common.cuh"

namespace oscnet {

constexpr int CB_THREADS = 1024;
constexpr int CB_MMAX = 8;                 // rows per thread
constexpr unsigned CB_COPY = 32768;        // bytes per bulk copy

struct CbGeom {
    int64_t n;
    int32_t W, B;                // columns per block, number of blocks
    int32_t CR, nchunks, M;      // rows per chunk (multiple of 32), chunks, rows per thread
    int32_t nseg;                // nchunks * B
    const uint16_t* eidx;        // segment entries: source index local to the block
    const uint16_t* roff;        // [nseg][CR + 1] offsets of the rows inside their segment
    const int64_t* segbase;      // [nseg + 1] first entry of each segment (multiples of 8)
};

__device__ __forceinline__ void cb_bulk_load(void* dst, const void* src, unsigned bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void cb_prefetch_l2(const void* src, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}

__device__ __forceinline__ unsigned cb_lds_u32(unsigned addr) {
    unsigned v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
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
// counts: roff[seg(c, b)][l + 1] = index pairs (words) of row (c, l) in block b; roff[seg][0] = 0
__global__ void cb_count_kernel(CbGeom g, const int64_t* __restrict__ row_ptr, const int32_t* __restrict__ col_idx,
                                int32_t ku, uint16_t* roff, int32_t* flag) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < (int64_t)g.nchunks * g.CR;
         i += (int64_t)gridDim.x * blockDim.x) {
        const int c = (int)(i / g.CR), l = (int)(i % g.CR);
        const int64_t row = i;                       // chunks are contiguous row ranges of CR rows
        int64_t b0 = 0, e0 = 0;
        if (row < g.n) {
            if (ku > 0) { b0 = row * (int64_t)ku; e0 = b0 + ku; }
            else { b0 = row_ptr[row]; e0 = row_ptr[row + 1]; }
        }
        int64_t q = b0;
        for (int b = 0; b < g.B; ++b) {
            const int64_t hi = (int64_t)(b + 1) * g.W;
            int cnt = 0;
            while (q < e0 && col_idx[q] < hi) { ++q; ++cnt; }
            cnt = (cnt + 1) / 2;                     // 32-bit words of two indices
            if (cnt > 65535) { atomicExch(flag + 4, 1); cnt = 65535; }
            uint16_t* seg = roff + ((int64_t)c * g.B + b) * (g.CR + 1);
            seg[l + 1] = (uint16_t)cnt;
            if (l == 0) seg[0] = 0;
        }
        if (q != e0) atomicExch(flag + 4, 2);       // rows must be sorted by column (canonical CSR)
    }
}

// inclusive scan of every segment's word counts in place; total in ENTRIES (two per word,
// rounded up to 8) to segtot
__global__ void __launch_bounds__(1024) cb_scan_kernel(CbGeom g, uint16_t* roff, int64_t* segtot, int32_t* flag) {
    __shared__ uint32_t wsum[32];
    __shared__ uint32_t carry_s;
    uint16_t* seg = roff + (int64_t)blockIdx.x * (g.CR + 1);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < g.CR; base += 1024) {
        const int l = base + threadIdx.x;
        uint32_t v = l < g.CR ? seg[l + 1] : 0u;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t u = __shfl_up_sync(0xffffffffu, v, o);
            if (lane >= o) v += u;
        }
        if (lane == 31) wsum[warp] = v;
        __syncthreads();
        uint32_t off = carry_s;
        for (int w = 0; w < warp; ++w) off += wsum[w];
        v += off;
        if (l < g.CR) {
            if (v > 65535u) { atomicExch(flag + 4, 3); v = 65535u; }
            seg[l + 1] = (uint16_t)v;
        }
        __syncthreads();
        if (threadIdx.x == 1023) carry_s = v;
        __syncthreads();
    }
    if (threadIdx.x == 0) segtot[blockIdx.x] = (2 * (int64_t)carry_s + 7) / 8 * 8;
}

// exclusive scan of the segment totals (one CTA)
__global__ void __launch_bounds__(1024) cb_segbase_kernel(int32_t nseg, const int64_t* segtot, int64_t* segbase) {
    __shared__ int64_t wsum[32];
    __shared__ int64_t carry_s;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < nseg; base += 1024) {
        const int s = base + threadIdx.x;
        const int64_t own = s < nseg ? segtot[s] : 0;
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
        if (s < nseg) segbase[s] = v - own;
        __syncthreads();
        if (threadIdx.x == 1023) carry_s = v;
        __syncthreads();
    }
    if (threadIdx.x == 0) segbase[nseg] = carry_s;
}

__global__ void cb_fill_kernel(CbGeom g, const int64_t* __restrict__ row_ptr, const int32_t* __restrict__ col_idx,
                               int32_t ku, const uint16_t* __restrict__ roff, const int64_t* __restrict__ segbase,
                               uint16_t* eidx) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < (int64_t)g.nchunks * g.CR;
         i += (int64_t)gridDim.x * blockDim.x) {
        if (i >= g.n) continue;
        const int c = (int)(i / g.CR), l = (int)(i % g.CR);
        int64_t q, e0;
        if (ku > 0) { q = i * (int64_t)ku; e0 = q + ku; }
        else { q = row_ptr[i]; e0 = row_ptr[i + 1]; }
        for (int b = 0; b < g.B && q < e0; ++b) {
            const int64_t lo = (int64_t)b * g.W, hi = lo + g.W;
            const int64_t s = (int64_t)c * g.B + b;
            int64_t dst = segbase[s] + 2 * (int64_t)roff[s * (g.CR + 1) + l];
            int cnt = 0;
            while (q < e0 && col_idx[q] < hi) { eidx[dst++] = (uint16_t)(col_idx[q++] - lo); ++cnt; }
            if (cnt & 1) eidx[dst] = (uint16_t)g.W;     // the zero slot
        }
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

// ES: the segment's entries are staged in shared memory next to the s block (same mbarrier);
// otherwise (a segment too long for the budget) they are read from global memory.
template <class T, int M, bool ES>
__global__ void __launch_bounds__(CB_THREADS, 1)
csr_blocked_stage_kernel(StageArgs a, ModelParams mp, TopoView tv, CbGeom g) {
    extern __shared__ __align__(128) unsigned char cb_smem[];
    __shared__ uint64_t bar;
    T* sblk = reinterpret_cast<T*>(cb_smem);                 // W values of s + the zero slot
    const size_t ent_at = ((size_t)g.W + 16) * sizeof(T);
    constexpr unsigned SH = sizeof(T) == 8 ? 3u : 2u;          // index -> byte offset
    constexpr unsigned MASK = 0xffffu << SH;
    const unsigned sblk_a = smem_u32(cb_smem);
    const unsigned zw_a = sblk_a + ((unsigned)g.W + 8u) * (unsigned)sizeof(T);   // word (W, W)
    const unsigned sent_a = sblk_a + (unsigned)ent_at;
    const T* __restrict__ gsrc = (const T*)a.s_in;
    const int t = threadIdx.x;
    const int CR1 = g.CR + 1;
    if (t == 0) {
        mbar_init(&bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        sblk[g.W] = T(0);
        *reinterpret_cast<unsigned*>(cb_smem + ((size_t)g.W + 8) * sizeof(T)) = (unsigned)g.W | (unsigned)g.W << 16;
    }
    __syncthreads();
    unsigned phase = 0;
    for (int c = blockIdx.x; c < g.nchunks; c += gridDim.x) {
        const int64_t row0 = (int64_t)c * g.CR;
        T acc[M];
        unsigned offs[M];            // o0 | o1 << 16 of the current block
        bool ok[M];
#pragma unroll
        for (int m = 0; m < M; ++m) {
            acc[m] = T(0);
            const int l = m * CB_THREADS + t;
            ok[m] = l < g.CR && row0 + l < g.n;
        }
        auto load_offs = [&](int b, unsigned (&o)[M]) {
            const uint16_t* ro = g.roff + ((int64_t)c * g.B + b) * CR1;
#pragma unroll
            for (int m = 0; m < M; ++m) {
                const int l = m * CB_THREADS + t;
                o[m] = ok[m] ? ((unsigned)__ldg(ro + l) | ((unsigned)__ldg(ro + l + 1) << 16)) : 0u;
            }
        };
        load_offs(0, offs);
        for (int b = 0; b < g.B; ++b) {
            const int64_t s = (int64_t)c * g.B + b;
            const int64_t col0 = (int64_t)b * g.W;
            __syncthreads();                       // every thread is done with the previous block
            if (t == 0) {
                int64_t cnt = g.n - col0 < g.W ? g.n - col0 : g.W;
                constexpr int V = 16 / (int)sizeof(T);
                const unsigned bytes = (unsigned)((cnt + V - 1) / V * V * sizeof(T));   // inside ld (multiple of 64)
                const int64_t e0 = g.segbase[s];
                const unsigned ebytes = ES ? (unsigned)((g.segbase[s + 1] - e0) * 2) : 0u;   // multiple of 16
                mbar_expect_tx(&bar, bytes + ebytes);
                for (unsigned o = 0; o < bytes; o += CB_COPY)
                    cb_bulk_load(cb_smem + o, (const unsigned char*)(gsrc + col0) + o, bytes - o < CB_COPY ? bytes - o : CB_COPY, &bar);
                for (unsigned o = 0; o < ebytes; o += CB_COPY)
                    cb_bulk_load(cb_smem + ent_at + o, (const unsigned char*)(g.eidx + e0) + o, ebytes - o < CB_COPY ? ebytes - o : CB_COPY, &bar);
            } else if (t == 32 && b + 1 < g.B) {   // next segment's entries towards L2
                const int64_t e0 = g.segbase[s + 1], e1 = g.segbase[s + 2];
                const unsigned bytes = (unsigned)((e1 - e0) * 2);
                if (bytes) cb_prefetch_l2(g.eidx + e0, bytes);
            }
            // while the block is in flight: next block's offsets (and, without staged entries, the
            // first two entries of every row)
            const unsigned* __restrict__ ent = reinterpret_cast<const unsigned*>(g.eidx + g.segbase[s]);
            unsigned first[ES ? 1 : M], nxt[M];
            if constexpr (!ES) {
#pragma unroll
                for (int m = 0; m < M; ++m) {
                    const unsigned o0 = offs[m] & 0xffffu, o1 = offs[m] >> 16;
                    first[m] = o0 < o1 ? __ldg(ent + o0) : ((unsigned)g.W | (unsigned)g.W << 16);
                }
            }
            if (b + 1 < g.B) load_offs(b + 1, nxt);
            mbar_wait(&bar, phase);
            phase ^= 1u;
            // warp-uniform trip counts (the longest run among the 32 lanes); lanes whose run is
            // over read the word that points twice at the zero slot, so the body has no branch
#pragma unroll
            for (int m = 0; m < M; ++m) {
                const unsigned o0 = offs[m] & 0xffffu, np = (offs[m] >> 16) - o0;
                const unsigned kmax = __reduce_max_sync(0xffffffffu, np);
                T a0 = T(0), a1 = T(0);
                if constexpr (ES) {
                    const unsigned p0 = sent_a + o0 * 4u;
#pragma unroll 2
                    for (unsigned k = 0; k < kmax; ++k) {
                        const unsigned w = cb_lds_u32(k < np ? p0 + k * 4u : zw_a);
                        a0 += cb_lds(sblk_a + ((w << SH) & MASK), T(0));
                        a1 += cb_lds(sblk_a + ((w >> (16 - SH)) & MASK), T(0));
                    }
                } else {
                    const unsigned* __restrict__ src = ent + o0;
                    if (np > 0) { a0 = sblk[first[m] & 0xffffu]; a1 = sblk[first[m] >> 16]; }
#pragma unroll 1
                    for (unsigned k = 1; k < kmax; ++k) {
                        if (k < np) {
                            const unsigned w = __ldg(src + k);
                            a0 += sblk[w & 0xffffu];
                            a1 += sblk[w >> 16];
                        }
                    }
                }
                acc[m] += a0 + a1;
            }
            if (b + 1 < g.B) {
#pragma unroll
                for (int m = 0; m < M; ++m) offs[m] = nxt[m];
            }
        }
        // ---- local field + stage update of this thread's rows
#pragma unroll
        for (int m = 0; m < M; ++m) {
            if (!ok[m]) continue;
            const int64_t i = row0 + m * CB_THREADS + t;
            const int deg = tv.k_uniform > 0 ? tv.k_uniform : (int)(tv.row_ptr[i + 1] - tv.row_ptr[i]);
            cb_finish_hh<T>(a, mp, i, acc[m], deg);
        }
    }
}

// ------------------------------------------------------------------ host side
constexpr size_t CB_SMEM_BUDGET = 224 * 1024;   // of the 227 KB a CTA may own

static int64_t cb_nnz(const net_desc* d) {
    return d->topo.kind == NET_TOPO_CSR ? d->topo.nnz : d->n * (int64_t)d->topo.in_degree;
}

// Geometry from the descriptor alone (the workspace query has no device): W from the shared
// memory budget, chunks of rows so that one wave of persistent CTAs covers the net.
// OSCNET_CSRB = "W,CR" overrides (tests use it to get several blocks and chunks on small nets).
static bool cb_geometry(const net_desc* d, CbGeom* g) {
    const net_topology& t = d->topo;
    if (d->model != NET_MODEL_HH) return false;
    if (t.kind != NET_TOPO_CSR && t.kind != NET_TOPO_RANDOM_INDEGREE) return false;
    const int64_t n = d->n;
    const size_t es = d->dtype == NET_F32 ? 4 : 8;
    int want_w = 0, want_cr = 0;
    if (const char* e = getenv("OSCNET_CSRB")) sscanf(e, "%d,%d", &want_w, &want_cr);
    if (want_w <= 0 && n < 32768) return false;          // small nets: the warp-per-row kernel
    const int sms = 148;
    int64_t CR = round_up((n + sms - 1) / sms, 32);
    if (want_cr > 0) CR = round_up(want_cr, 32);
    if (CR > CB_MMAX * CB_THREADS) CR = CB_MMAX * CB_THREADS;
    const int64_t nchunks = (n + CR - 1) / CR;
    // shared memory = s block (W elements) + the entries of one segment (about nnz / (chunks B)
    // 16-bit indices, 25 % slack for uneven rows): fixed point of W over three rounds
    const double per_chunk = (double)cb_nnz(d) / (double)nchunks;
    int W = (int)(CB_SMEM_BUDGET / es);
    for (int it = 0; it < 3; ++it) {
        const double Bq = (double)n / W < 1.0 ? 1.0 : (double)n / W;
        const double seg_bytes = 1.25 * (per_chunk / Bq + 0.5 * (double)CR) * 2.0 + 1024.0;   // odd runs are padded
        const double w = ((double)CB_SMEM_BUDGET - seg_bytes) / (double)es - 16.0;
        W = w < 1024.0 ? 1024 : (int)w;
    }
    if (W > 65520) W = 65520;                             // W itself is the index of the zero slot
    if (want_w > 0) W = want_w < 16 ? 16 : (want_w > 65520 ? 65520 : want_w);
    const int B0 = (int)((n + W - 1) / W);
    W = (int)round_up((n + B0 - 1) / B0, 16);             // equal blocks, 16-element granules
    const int B = (int)((n + W - 1) / W);
    if (nchunks * B > (int64_t)1 << 24) return false;
    memset(g, 0, sizeof(*g));
    g->n = n; g->W = W; g->B = B; g->CR = (int)CR; g->nchunks = (int)nchunks;
    g->M = (int)((CR + CB_THREADS - 1) / CB_THREADS);
    g->nseg = (int)(nchunks * B);
    return true;
}

bool csr_blocked_supported(const net_desc* d) {
    CbGeom g;
    return cb_geometry(d, &g);
}

// scratch: eidx | roff | segbase | segtot
struct CbLayout { size_t eidx, roff, segbase, segtot, total; };
static CbLayout cb_layout(const net_desc* d, const CbGeom& g) {
    CbLayout L;
    size_t cur = 0;
    auto take = [&](size_t bytes) { size_t at = cur; cur += (bytes + 255) / 256 * 256; return at; };
    const size_t nnz = (size_t)cb_nnz(d), pairs = (size_t)g.nchunks * g.CR * (size_t)g.B;
    L.eidx = take((nnz + (nnz < pairs ? nnz : pairs) + 8 * (size_t)g.nseg + 64) * sizeof(uint16_t));   // + one pad per odd run
    L.roff = take((size_t)g.nseg * (g.CR + 1) * sizeof(uint16_t) + 64);
    L.segbase = take(((size_t)g.nseg + 2) * sizeof(int64_t));
    L.segtot = take(((size_t)g.nseg + 2) * sizeof(int64_t));
    L.total = cur;
    return L;
}

size_t csr_blocked_scratch_bytes(const net_desc* d) {
    CbGeom g;
    if (!cb_geometry(d, &g)) return 0;
    return cb_layout(d, g).total;
}

template <class T, bool ES>
static const void* cb_kernel_for_m(int M) {
    switch (M) {
        case 1: return (const void*)csr_blocked_stage_kernel<T, 1, ES>;
        case 2: return (const void*)csr_blocked_stage_kernel<T, 2, ES>;
        case 3: return (const void*)csr_blocked_stage_kernel<T, 3, ES>;
        case 4: return (const void*)csr_blocked_stage_kernel<T, 4, ES>;
        case 5: return (const void*)csr_blocked_stage_kernel<T, 5, ES>;
        case 6: return (const void*)csr_blocked_stage_kernel<T, 6, ES>;
        case 7: return (const void*)csr_blocked_stage_kernel<T, 7, ES>;
        default: return (const void*)csr_blocked_stage_kernel<T, 8, ES>;
    }
}
template <class T>
static const void* cb_kernel_for(int M, bool es) {
    return es ? cb_kernel_for_m<T, true>(M) : cb_kernel_for_m<T, false>(M);
}

// Builds the segment arrays in the scratch region.  NET_ERR_UNSUPPORTED (a segment longer than
// 65535 entries, rows not sorted) sends the net back to the warp-per-row kernel.
int32_t csr_blocked_prepare(net* h) {
    CbGeom g;
    if (!cb_geometry(&h->desc, &g)) return NET_ERR_UNSUPPORTED;
    const CbLayout L = cb_layout(&h->desc, g);
    if (L.total > h->b.scratch_bytes) return NET_ERR_UNSUPPORTED;
    char* s = (char*)h->b.scratch;
    uint16_t* eidx = (uint16_t*)(s + L.eidx);
    uint16_t* roff = (uint16_t*)(s + L.roff);
    int64_t* segbase = (int64_t*)(s + L.segbase);
    int64_t* segtot = (int64_t*)(s + L.segtot);
    g.eidx = eidx; g.roff = roff; g.segbase = segbase;
    cudaStream_t st = h->stream;
    const int64_t rows = (int64_t)g.nchunks * g.CR;
    const unsigned grid = (unsigned)((rows + 255) / 256 > 148 * 16 ? 148 * 16 : (rows + 255) / 256);
    const int32_t ku = h->tv.k_uniform;
    OSC_CUDA(h, cudaMemsetAsync(h->b.flag + 4, 0, sizeof(int32_t), st));   // flag[4]: this builder's verdict
    cb_count_kernel<<<grid, 256, 0, st>>>(g, h->tv.row_ptr, h->tv.col_idx, ku, roff, h->b.flag);
    cb_scan_kernel<<<g.nseg, 1024, 0, st>>>(g, roff, segtot, h->b.flag);
    cb_segbase_kernel<<<1, 1024, 0, st>>>(g.nseg, segtot, segbase);
    cb_fill_kernel<<<grid, 256, 0, st>>>(g, h->tv.row_ptr, h->tv.col_idx, ku, roff, segbase, eidx);
    h->launches += 4;
    OSC_CUDA(h, cudaGetLastError());
    int32_t flag = 0;
    OSC_CUDA(h, cudaMemcpyAsync(&flag, h->b.flag + 4, sizeof(flag), cudaMemcpyDeviceToHost, st));
    OSC_CUDA(h, cudaStreamSynchronize(st));
    if (flag != 0) return NET_ERR_UNSUPPORTED;
    // longest segment: do its entries fit next to the s block?
    int64_t maxseg = 0;
    {
        int64_t* tot = (int64_t*)malloc(sizeof(int64_t) * (size_t)g.nseg);
        if (!tot) return set_err(h, NET_ERR_INVALID, "out of host memory");
        cudaError_t e = cudaMemcpyAsync(tot, segtot, sizeof(int64_t) * (size_t)g.nseg, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        for (int q = 0; q < g.nseg && e == cudaSuccess; ++q) maxseg = tot[q] > maxseg ? tot[q] : maxseg;
        free(tot);
        if (e != cudaSuccess) return cuda_err(h, e, "segment totals");
    }
    const size_t sblock = ((size_t)g.W + 16) * h->esize;      // + the zero slot, 128-byte granule
    const bool es = sblock + (size_t)maxseg * 2 <= CB_SMEM_BUDGET;
    const size_t smem = sblock + (es ? (size_t)maxseg * 2 : 0);
    if (smem > CB_SMEM_BUDGET) return NET_ERR_UNSUPPORTED;
    const void* kern = h->desc.dtype == NET_F32 ? cb_kernel_for<float>(g.M, es) : cb_kernel_for<double>(g.M, es);
    OSC_CUDA(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    static_assert(sizeof(CbGeom) <= sizeof(((net*)0)->cb_geom), "cb_geom storage too small");
    memcpy(h->cb_geom, &g, sizeof(g));
    h->cb_grid = (unsigned)(g.nchunks < sms ? g.nchunks : sms);
    h->cb_smem = smem;
    h->cb_es = es ? 1 : 0;
    if (getenv("OSCNET_VERBOSE"))
        fprintf(stderr, "csr_blocked: W %d B %d CR %d chunks %d M %d maxseg %lld entries_in_smem %d smem %zu grid %u scratch %zu\n",
                g.W, g.B, g.CR, g.nchunks, g.M, (long long)maxseg, (int)es, smem, h->cb_grid, L.total);
    return NET_OK;
}

int32_t csr_blocked_stage(net* h, const StageArgs& a) {
    CbGeom g;
    memcpy(&g, h->cb_geom, sizeof(g));
    const bool es = h->cb_es != 0;
    const void* kern = h->desc.dtype == NET_F32 ? cb_kernel_for<float>(g.M, es) : cb_kernel_for<double>(g.M, es);
    StageArgs aa = a;
    void* params[] = {&aa, &h->mp, &h->tv, &g};
    OSC_CUDA(h, cudaLaunchKernel(kern, dim3(h->cb_grid), dim3(CB_THREADS), params, h->cb_smem, h->stream));
    h->launches += 1;
    return NET_OK;
}

}  // namespace oscnet
