// Host side of the third-generation 3D lattice kernels (lat3_kernel.cuh): tile / pipeline /
// chunk selection, TMA tensor maps of the stencil sources and of the operand tiles, launch.
// Included by one translation unit per (dtype, model) so that the build stays parallel.
#pragma once
#include <stdlib.h>

#include "lat3_kernel.cuh"
#include "lat3s_kernel.cuh"

namespace oscnet {

// thread shape per (dtype, P): X columns x TY rows of outputs per thread
template <class T, int P> struct L3Shape;
template <> struct L3Shape<float, 2> { static constexpr int X = 2, TY = 4; };
template <> struct L3Shape<float, 4> { static constexpr int X = 2, TY = 2; };
template <> struct L3Shape<double, 2> { static constexpr int X = 2, TY = 2; };
template <> struct L3Shape<double, 4> { static constexpr int X = 2, TY = 1; };
// radius 6 (the paper's largest): field-split kernel only (KS / KS with inertia)
template <> struct L3Shape<float, 6> { static constexpr int X = 2, TY = 2; };
template <> struct L3Shape<double, 6> { static constexpr int X = 2, TY = 2; };
constexpr int L3_MAXT = 288;     // up to 8 consumer warps + the producer warp
constexpr int L3_MINB = 1;
// KS runs the field-split kernel (lat3s_kernel.cuh): two lanes per 2 x 2 block of outputs, the
// exchange field E as two planes (cos | sin)
template <class T, int MODEL, int P> struct L3Sh {
    static constexpr bool SPLIT = MODEL == NET_MODEL_KS;
    static constexpr int X = SPLIT ? 2 : L3Shape<T, P>::X;
    static constexpr int TY = SPLIT ? 2 : L3Shape<T, P>::TY;   // fp32 with TY = 4 measured slower (2.03e10 vs 2.30e10 on cfg 3a)
    static constexpr int UPW = SPLIT ? 16 : 32;      // blocks of X x TY outputs per consumer warp
    // fp32 field-split: 7 consumer warps + producer, two CTAs per SM => 128 registers per thread
    // (fp64 at 160 threads x 3 CTAs, 128 registers: 1.10e10 against 1.08e10 on cfg 3b -- not kept)
    static constexpr int MAXT = (SPLIT && sizeof(T) == 4) ? 256 : L3_MAXT;
    static constexpr int MINB = (SPLIT && sizeof(T) == 4 && P <= 4) ? 2 : L3_MINB;   // P = 6: 13 open planes, one CTA per SM
};

// Field-split kernel: extra columns of the staged box that make the shared-memory row pitch
// continue the bank sequence where a thread-row ends, so that a half-warp (fp32, LDS.64) or
// quarter-warp (fp64, LDS.128) of consecutive blocks that straddles two thread-rows still covers
// 128 consecutive bytes modulo 128 (the ncu capture of the unpadded kernel: 40 % of the
// shared-memory wavefronts of cfg 3a were such conflicts).  -1: no pitch does it for this width.
template <class T> inline int l3s_pad(int TXt, int HX, int TY) {
    const int q = 16 / (int)sizeof(T);                     // scalars per 16 bytes (TMA inner-box granule)
    for (int pad = 0; pad * (int)sizeof(T) < 128; pad += q)
        if (((TY * (TXt + 2 * HX + pad) - TXt) * (int)sizeof(T)) % 128 == 0) return pad;
    return -1;
}
// The same for the pair kernel (elements are (u, v) pairs of 2 sizeof(T) bytes; a thread reads X = 2 of them
// per 16 or 32 bytes): cfg 5, tile 78 x 16, had 32 % of its shared-memory wavefronts in such conflicts with the
// shared-memory data pipe the busiest unit of the SM (71 %; profiles/r02_ncu.md).
template <class T> inline int l3p_pad(int TXt, int HX, int TY) {
    const int eb = 2 * (int)sizeof(T);
    const int q = eb >= 16 ? 1 : 16 / eb;
    for (int pad = 0; pad * eb < 128; pad += q)
        if (((TY * (TXt + 2 * HX + pad) - TXt) * eb) % 128 == 0) return pad;
    return -1;
}

typedef CUresult (*l3_encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                 const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                 CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline int32_t l3_encoder(net* h, l3_encode_fn* out) {
    static l3_encode_fn encode = nullptr;
    if (!encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
        if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn)
            return set_err(h, NET_ERR_CUDA, "cuTensorMapEncodeTiled is not available from the driver");
        encode = (l3_encode_fn)fn;
    }
    *out = encode;
    return NET_OK;
}

// 3D map over an array of `esz`-byte elements (4 or 8) with extents (ex, ey, ez) and box (bx, by, 1)
inline int32_t l3_encode(net* h, CUtensorMap* tm, void* base, int esz, uint64_t ex, uint64_t ey, uint64_t ez,
                         uint32_t bx, uint32_t by) {
    l3_encode_fn encode;
    int32_t rc = l3_encoder(h, &encode);
    if (rc) return rc;
    cuuint64_t dims[3] = {ex, ey, ez};
    cuuint64_t strides[2] = {ex * (uint64_t)esz, ex * ey * (uint64_t)esz};
    cuuint32_t box[3] = {bx, by, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = encode(tm, esz == 4 ? CU_TENSOR_MAP_DATA_TYPE_UINT32 : CU_TENSOR_MAP_DATA_TYPE_UINT64, 3, base,
                        dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                        CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return set_err(h, NET_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
    return NET_OK;
}

// 4D map over two planes of `esz`-byte elements: extents (ex, ey, ez, 2), box (bx, by, 1, 2)
inline int32_t l3_encode_planes(net* h, CUtensorMap* tm, void* base, int esz, uint64_t ex, uint64_t ey, uint64_t ez,
                                uint32_t bx, uint32_t by) {
    l3_encode_fn encode;
    int32_t rc = l3_encoder(h, &encode);
    if (rc) return rc;
    cuuint64_t dims[4] = {ex, ey, ez, 2};
    const uint64_t e8 = (uint64_t)esz;
    cuuint64_t strides[3] = {ex * e8, ex * ey * e8, ex * ey * ez * e8};
    cuuint32_t box[4] = {bx, by, 1, 2};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = encode(tm, esz == 4 ? CU_TENSOR_MAP_DATA_TYPE_UINT32 : CU_TENSOR_MAP_DATA_TYPE_UINT64, 4, base, dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                        CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return set_err(h, NET_ERR_CUDA, "cuTensorMapEncodeTiled (planes) failed (%d)", (int)r);
    return NET_OK;
}

template <class T, int MODEL, int P, int STAGE>
static auto l3_kernel_ptr() {
    typedef L3Sh<T, MODEL, P> S;
    if constexpr (S::SPLIT) {
        // accumulator addressing (ROT of lat3_kernel.cuh), measured on a B200 at P = 4:
        //   fp32 (cfg 3a, e10 osc-steps/s): ROT 0 (nine plane bodies, 146 KB of SASS) 2.26 | 1: 1.97 | 2: 2.42 |
        //     3: 2.50 | 4: 2.53 | 5: 2.57 | 6: 2.43 | 7: 2.38 -- five bodies (73 KB) still sit in the instruction
        //     cache, six do not;
        //   fp64 (cfg 3b): ROT 1: 1.19 | 2: 1.25 | 3: 1.19 (spills at the 168-register cap of two CTAs per SM).
        //   P = 6, fp64 (cfg 6c, e9): ROT 1: 3.20 | 2: 3.06 | 3: 2.47 (13 open planes: spills grow with the group).
        constexpr int ROT0 = P > 4 ? 1 : P == 4 ? (sizeof(T) == 4 ? 5 : 2) : 0;
        return lat3s_kernel<T, P, STAGE, S::TY, S::MAXT, S::MINB, ROT0>;
    } else {
        // FHN, P = 2, fp32 (cfg 5, HBM-bound): ROT 0 (five bodies, 53-65 KB) 5.53e10 | 2: 5.60e10 | 3: 5.31e10 -- noise
        constexpr int ROTF = (P > 2 && sizeof(T) == 4) ? 1 : 0;
        return lat3_kernel<T, MODEL, P, STAGE, S::X, S::TY, L3_MAXT, L3_MINB, ROTF>;
    }
}

inline size_t l3_smem_bytes(const L3Geom& g, int P, int nt) {
    return 256 + (size_t)(P + 1 + g.D) * g.st_stride + (size_t)(g.D + 1) * nt * g.op_stride;
}

// Calls f(TXt, SY, score) for every tile the staged boxes and the thread budget allow.  Score:
// lane / cover efficiency over the halo overhead, with the measured preferences below.
template <class T, int MODEL, int P, class F>
static int32_t l3_enumerate(int nx, int ny, int want_tx, int want_sy, F&& f) {
    typedef L3Sh<T, MODEL, P> S;
    constexpr int X = S::X, TY = S::TY;
    constexpr int HX = l2_hx<T>(P);
    constexpr int U8 = 2 * (int)sizeof(T) / 8;
    constexpr bool KS = MODEL == NET_MODEL_KS;
    const int xq = (KS && sizeof(T) == 4) ? 4 : X;
    for (int tiles_x = 1; tiles_x <= nx / xq; ++tiles_x) {
        int TXt = ((nx + tiles_x - 1) / tiles_x + xq - 1) / xq * xq;
        if (want_tx > 0) TXt = (want_tx + xq - 1) / xq * xq;
        if (TXt > nx) TXt = nx;
        const int tx = (nx + TXt - 1) / TXt;
        const int QX = TXt / X;
        if ((TXt + 2 * HX) * U8 > 256) { if (want_tx > 0) return NET_ERR_UNSUPPORTED; continue; }
        for (int SY = 1; (SY * QX + S::UPW - 1) / S::UPW * 32 <= S::MAXT - 32 && SY * TY <= 256 - 2 * P; ++SY) {
            if (want_sy > 0 && SY != want_sy) continue;
            const int TYt = SY * TY, ty = (ny + TYt - 1) / TYt;
            const int units = QX * SY, warps = (units + S::UPW - 1) / S::UPW;
            const double lane_eff = (double)units / ((double)S::UPW * warps);
            const double cover = (double)nx * ny / ((double)tx * TXt * ty * TYt);
            const double halo = (double)(TXt + 2 * HX) * (TYt + 2 * P) / ((double)TXt * TYt);
            // small CTAs (about four consumer warps) desynchronise better; mild preference
            const double size_pen = warps <= 4 ? 1.0 : 1.0 - 0.02 * (warps - 4);
            // shared-memory banks: the lanes of one vector-load phase (8 lanes of LDS.128) that fall
            // on the next strip of rows are TY staged rows further on; if that distance is a
            // multiple of 128 bytes they hit the banks of the lanes before them (measured: 39 % of
            // the wavefronts of cfg 5 were such conflicts).  Phases never straddle strips when QX
            // is a multiple of 8.  fp64 planes: the rule that held on cfg 3b is simply >= 16
            // threads per staged row.
            constexpr bool PLANAR = S::SPLIT;
            const int row_bytes = (TXt + 2 * HX) * (PLANAR ? (int)sizeof(T) : 2 * (int)sizeof(T));
            const bool straddle = QX % 8 != 0 && SY > 1;
            const bool ppad = !getenv("OSCNET_L3P_NOPAD");
            const double bank_pen = PLANAR ? (QX % (sizeof(T) == 8 ? 8 : 16) != 0 && l3s_pad<T>(TXt, HX, TY) < 0 ? 0.85 : 1.0)
                                  : ppad ? (straddle && QX % (sizeof(T) == 8 ? 4 : 8) != 0 && l3p_pad<T>(TXt, HX, TY) < 0 ? 0.85 : 1.0)
                                         : ((straddle && (TY * row_bytes) % 128 == 0) ? 0.85 : 1.0);
            f(TXt, SY, lane_eff * cover * size_pen * bank_pen / (1.0 + 0.25 * (halo - 1.0)));
        }
        if (want_tx > 0) break;
    }
    return NET_OK;
}

// Geometry of one stage.  Tiles: the (TXt, SY) with the best lane / cover efficiency among
// those whose staged boxes TMA can take; pipeline depth D: the deepest that still leaves
// `want_ctas` CTAs per SM; grid: fewest planes on the longest CTA.  OSCNET_LAT3 = "TXt,SY,Lz,D,CTAS[,A]"
// overrides (Lz > 0: chunks of Lz planes, no tail -- or, with A < Lz, that many chunks shortened to A
// planes and a tail over the rest; Lz < 0: -Lz CTAs with equal spans of the whole space).
template <class T, int MODEL, int P, int STAGE>
static int32_t l3_configure_stage(net* h) {
    typedef L3Sh<T, MODEL, P> S;
    constexpr int X = S::X, TY = S::TY;
    constexpr int HX = l2_hx<T>(P);
    constexpr int U8 = 2 * (int)sizeof(T) / 8;
    constexpr bool KS = MODEL == NET_MODEL_KS;
    constexpr int NT = L3Ops<MODEL, STAGE>::N;
    const TopoView& tv = h->tv;
    L3Geom g;
    memset(&g, 0, sizeof(g));
    g.nx = tv.nx; g.ny = tv.ny; g.nz = tv.nz;
    int want_tx = 0, want_sy = 0, want_lz = 0, want_d = 0, want_ctas = 0, want_a = 0;
    if (const char* e = getenv("OSCNET_LAT3")) sscanf(e, "%d,%d,%d,%d,%d,%d", &want_tx, &want_sy, &want_lz, &want_d, &want_ctas, &want_a);
    if (want_ctas <= 0) want_ctas = h->l3_force_ctas > 0 ? h->l3_force_ctas : 2;
    // operand / stencil rows must be whole 16-byte vectors: scalar f32 tiles need TXt % 4 == 0
    const int xq = (KS && sizeof(T) == 4) ? 4 : X;
    if (g.nx % xq != 0) return NET_ERR_UNSUPPORTED;
    if (want_tx <= 0 && h->l3_force_tx > 0) { want_tx = h->l3_force_tx; want_sy = h->l3_force_sy; }   // autotuned
    double best = -1.0;
    int rc_enum = l3_enumerate<T, MODEL, P>(g.nx, g.ny, want_tx, want_sy, [&](int TXt, int SY, double score) {
        if (score > best) {
            best = score; g.TXt = TXt; g.TYt = SY * TY; g.QX = TXt / X; g.SY = SY;
            g.tiles_x = (g.nx + TXt - 1) / TXt; g.tiles_y = (g.ny + g.TYt - 1) / g.TYt;
        }
    });
    if (rc_enum) return rc_enum;
    if (best < 0) return NET_ERR_UNSUPPORTED;
    g.PW = g.TXt + 2 * HX;
    if (S::SPLIT && g.QX % (sizeof(T) == 8 ? 8 : 16) != 0 && !getenv("OSCNET_L3S_NOPAD")) {
        const int pad = l3s_pad<T>(g.TXt, HX, TY);
        if (pad > 0 && (g.PW + pad) * U8 <= 256) g.PW += pad;
    }
    if (!S::SPLIT && g.SY > 1 && g.QX % (sizeof(T) == 8 ? 4 : 8) != 0 && !getenv("OSCNET_L3P_NOPAD")) {
        const int pad = l3p_pad<T>(g.TXt, HX, TY);
        if (pad > 0 && (g.PW + pad) * U8 <= 256) g.PW += pad;
    }
    g.PH = g.TYt + 2 * P;
    g.ncw = (g.QX * g.SY + S::UPW - 1) / S::UPW;
    g.st_bytes = (unsigned)((size_t)g.PW * g.PH * 2 * sizeof(T));
    g.st_stride = (g.st_bytes + 127u) / 128u * 128u;
    g.op_bytes = (unsigned)((size_t)g.TXt * g.TYt * (KS ? 1 : 2) * sizeof(T));
    g.op_stride = (g.op_bytes + 127u) / 128u * 128u;
    const int threads = 32 * (g.ncw + 1);
    auto kern = l3_kernel_ptr<T, MODEL, P, STAGE>();
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const size_t smem_cap = 227 * 1024;
    g.D = 0;
    for (int D = 4; D >= 1; --D) {
        g.D = D;
        if (want_d > 0) g.D = want_d;
        if (l3_smem_bytes(g, P, NT) * want_ctas + 1024 * want_ctas <= smem_cap || want_d > 0) break;
        g.D = 0;
    }
    if (g.D == 0) {      // not even D = 1 at the wanted occupancy: one CTA per SM, deepest pipeline that fits
        for (int D = 4; D >= 1 && g.D == 0; --D) { g.D = D; if (l3_smem_bytes(g, P, NT) + 1024 > smem_cap) g.D = 0; }
        if (g.D == 0) return NET_ERR_UNSUPPORTED;
    }
    const size_t smem = l3_smem_bytes(g, P, NT);
    if (smem + 1024 > smem_cap) return NET_ERR_UNSUPPORTED;
    OSC_CUDA(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    OSC_CUDA(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, threads, smem));
    if (occ < 1) return NET_ERR_UNSUPPORTED;
    // Grid (l3_span in lat3_kernel.cuh): chunk-aligned CTAs, tiles x chunks of them, marching in step;
    // where they leave part of a single wave empty, shorter chunks plus a tail of equal spans over the
    // planes left at the top of the columns.  Cost = waves x planes of the longest CTA, a chunk paying
    // its 2P lead-in planes (+ 4 for the pipeline restart).  l3_force_tail < 0: aligned only.
    const int64_t slots = (int64_t)occ * sms, tiles = (int64_t)g.tiles_x * g.tiles_y;
    const int64_t SP = tiles * g.nz;                                         // tile-planes of one stage
    const int HZ = 2 * P + 4;
    double best_cost = -1.0;
    int64_t grid = tiles;
    g.Lz = g.nz; g.nchunks = 1;
    const bool allow_tail = h->l3_force_tail >= 0 && want_lz == 0 && !getenv("OSCNET_LAT3_NO_TAIL");
    for (int nch = 1; nch <= g.nz; ++nch) {
        const int Lz = (g.nz + nch - 1) / nch;
        const int chunks = (g.nz + Lz - 1) / Lz;
        const int64_t m = tiles * chunks;
        const int64_t waves = (m + slots - 1) / slots;
        const double cost = (double)(waves * (Lz + HZ));
        if (best_cost < 0 || cost < best_cost) { best_cost = cost; g.Lz = Lz; g.nchunks = chunks; grid = m; }
        if (!allow_tail || m >= slots) continue;
        const int64_t gt = slots - m;                                        // CTAs of the tail
        // lead-in planes only accumulate (no finisher): about 3/4 of a plane each; a span of Lt planes
        // in columns of r planes starts 1 + Lt / r segments on average (fit to A sweeps on cfg 3a / 3b:
        // optimum at 87-91 of 100 planes)
        const double lead = 0.75 * (2 * P);
        for (int a = Lz - 1; a >= 8 * P && 2 * a >= Lz; --a) {    // short chunks: the tail's lead-ins cost more than they fill (cfg 6b: 6.8e9 aligned, 6.2e9 with a tail)
            const int64_t r = g.nz - (int64_t)chunks * a;
            if (r <= 0) continue;
            const double Lt = (double)(tiles * r) / (double)gt;
            const double tail = Lt + (1.0 + Lt / (double)r) * lead + (HZ - lead), main = a + HZ;   // same scale as `cost`
            const double c2 = main > tail ? main : tail;
            if (c2 < best_cost) { best_cost = c2; g.Lz = a; g.nchunks = chunks; grid = slots; }
        }
    }
    if (want_lz > 0) {
        g.Lz = want_lz; g.nchunks = (g.nz + g.Lz - 1) / g.Lz; grid = tiles * g.nchunks;
        if (want_a > 0 && want_a < want_lz && tiles * g.nchunks < slots && (int64_t)g.nchunks * want_a < g.nz) { g.Lz = want_a; grid = slots; }
    }
    if (want_lz < 0 && -(int64_t)want_lz <= SP) { g.Lz = 0; g.nchunks = 0; grid = -want_lz; }   // equal spans over everything
    h->lat3[STAGE] = g;
    h->lat3_threads[STAGE] = threads;
    h->lat3_smem[STAGE] = smem;
    h->lat3_grid[STAGE] = (unsigned)grid;
    if (getenv("OSCNET_VERBOSE"))
        fprintf(stderr, "lat3 stage %d: tile %dx%d (QX %d SY %d, %d consumer warps) tiles %dx%d Lz %d chunks %d D %d smem %zu occ %d grid %u\n",
                STAGE, g.TXt, g.TYt, g.QX, g.SY, g.ncw, g.tiles_x, g.tiles_y, g.Lz, g.nchunks, g.D, smem, occ, h->lat3_grid[STAGE]);
    return NET_OK;
}

// all stages + tensor maps for the tile l3_configure_stage picks (by score, or h->l3_force_*)
template <class T, int MODEL, int P>
static int32_t l3_configure_tile(net* h) {
    constexpr int HX = l2_hx<T>(P);
    constexpr int U8 = 2 * (int)sizeof(T) / 8;
    constexpr bool KS = MODEL == NET_MODEL_KS;
    int32_t rc;
    if ((rc = l3_configure_stage<T, MODEL, P, L3_S0>(h))) return rc;
    if ((rc = l3_configure_stage<T, MODEL, P, L3_S1>(h))) return rc;
    if ((rc = l3_configure_stage<T, MODEL, P, L3_S2>(h))) return rc;
    if ((rc = l3_configure_stage<T, MODEL, P, L3_S3>(h))) return rc;
    if ((rc = l3_configure_stage<T, MODEL, P, L3_RHS>(h))) return rc;
    if ((rc = l3_configure_stage<T, MODEL, P, L3_LOC>(h))) return rc;
    // the tile is the same for every stage (only D differs), so one set of maps serves all
    const L3Geom& g = h->lat3[0];
    const uint64_t nxp = (uint64_t)g.nx + 2 * HX, nyp = (uint64_t)g.ny + 2 * P;
    void* st_src[4] = {h->b.y, h->b.Y2, h->b.Y3, h->b.Y4};
    if (KS) { st_src[0] = h->E_a; st_src[1] = h->E_b; }
    constexpr bool PLANAR = L3Sh<T, MODEL, P>::SPLIT;   // (cos | sin) planes instead of pairs (lat3s_kernel.cuh)
    for (int st = 0; st < 6; ++st) h->lat3[st].plane = (long long)(nxp * nyp * (uint64_t)g.nz);
    for (int k = 0; k < (KS ? 2 : 4); ++k) {
        if (PLANAR) rc = l3_encode_planes(h, &h->tm3_st[k], st_src[k], (int)sizeof(T), nxp, nyp, (uint64_t)g.nz, (uint32_t)g.PW, (uint32_t)g.PH);
        else rc = l3_encode(h, &h->tm3_st[k], st_src[k], 8, nxp * U8, nyp, (uint64_t)g.nz, (uint32_t)(g.PW * U8), (uint32_t)g.PH);
        if (rc) return rc;
    }
    h->ks_planar = PLANAR ? 1 : 0;
    if (KS) {
        void* op_src[4] = {h->b.y, h->b.Y2, h->b.Y3, h->b.elem_param};
        for (int k = 0; k < 4; ++k)
            if ((rc = l3_encode(h, &h->tm3_op[k], op_src[k], (int)sizeof(T), (uint64_t)g.nx, (uint64_t)g.ny, (uint64_t)g.nz, (uint32_t)g.TXt, (uint32_t)g.TYt))) return rc;
    } else {
        void* op_src[2] = {h->b.y, h->b.Y2};
        for (int k = 0; k < 2; ++k)
            if ((rc = l3_encode(h, &h->tm3_op[k], op_src[k], 8, nxp * U8, nyp, (uint64_t)g.nz, (uint32_t)(g.TXt * U8), (uint32_t)g.TYt))) return rc;
        h->tm3_op[2] = h->tm3_op[0];
        h->tm3_op[3] = h->tm3_op[0];
    }
    return NET_OK;
}

template <class T, int MODEL, int P>
static L3Params<T> l3_params(const net* h, int stage, double dt) {
    L3Params<T> p;
    memset(&p, 0, sizeof(p));
    const ModelParams& mp = h->mp;
    const int n_ball = h->tv.noff + (h->tv.include_self ? 0 : 1);
    const int deg = h->tv.noff;
    const double inv_deg = deg > 0 ? 1.0 / deg : 0.0;
    const double hh = stage == 0 || stage == 1 ? 0.5 * dt : stage == 2 ? dt : stage == 3 ? dt / 6.0 : 0.0;
    p.h = (T)hh;
    p.nb = (T)n_ball;
    const double s = mp.sigma * inv_deg;
    p.cuu = (T)(s * mp.buu * mp.inv_eps); p.cuv = (T)(s * mp.buv * mp.inv_eps);
    p.cvu = (T)(s * mp.bvu); p.cvv = (T)(s * mp.bvv);
    p.ie = (T)mp.inv_eps; p.ie3 = (T)(-mp.inv_eps / 3.0); p.a = (T)mp.a;
    p.kd = (T)(mp.K * inv_deg); p.ca = (T)mp.cos_a; p.sa = (T)mp.sin_a;
    p.inv_nb = (T)(1.0 / n_ball);
    p.include_self = h->tv.include_self;
    return p;
}

template <class T, int MODEL, int P, int STAGE>
static int32_t l3_launch_stage(net* h, const L3Ptrs& a, double dt, const CUtensorMap& st, const CUtensorMap* op) {
    auto kern = l3_kernel_ptr<T, MODEL, P, STAGE>();
    const L3Params<T> p = l3_params<T, MODEL, P>(h, STAGE, dt);
    kern<<<h->lat3_grid[STAGE], h->lat3_threads[STAGE], h->lat3_smem[STAGE], h->stream>>>(
        st, op[0], op[1], op[2], op[3], a, p, h->lat3[STAGE]);
    h->launches += 1;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

// Buffer roles per stage (Z form): in = y, Y2, Y3, Y4; out = Y2, Y3, Y4 (+ Z into Y2), y.
template <class T, int MODEL, int P>
static int32_t l3_stage(net* h, int stage, double dt, void* rhs_out) {
    constexpr bool KS = MODEL == NET_MODEL_KS;
    const Buffers& b = h->b;
    L3Ptrs a;
    memset(&a, 0, sizeof(a));
    CUtensorMap op[4] = {h->tm3_op[0], h->tm3_op[0], h->tm3_op[0], h->tm3_op[0]};
    const CUtensorMap* tm = h->tm3_st;
    const CUtensorMap* to = h->tm3_op;     // FHN: y, Y2 | KS: y, Y2, Y3, omega
    switch (stage) {
        case 0:
            a.out = b.Y2; a.Eout = h->E_b;
            if (KS) { op[0] = to[0]; op[1] = to[3]; }
            return l3_launch_stage<T, MODEL, P, L3_S0>(h, a, dt, tm[0], op);
        case 1:
            a.out = b.Y3; a.Eout = h->E_a;
            op[0] = to[0];
            if (KS) op[1] = to[3];
            return l3_launch_stage<T, MODEL, P, L3_S1>(h, a, dt, tm[1], op);
        case 2:
            a.out = b.Y4; a.out2 = b.Y2; a.Eout = h->E_b;
            op[0] = to[0]; op[1] = to[1];
            if (KS) { op[2] = to[2]; op[3] = to[3]; }
            return l3_launch_stage<T, MODEL, P, L3_S2>(h, a, dt, tm[KS ? 0 : 2], op);
        case 3:
            a.out = b.y; a.Eout = h->E_a;
            op[0] = to[1];                     // Z lives in Y2
            if (KS) op[1] = to[3];
            return l3_launch_stage<T, MODEL, P, L3_S3>(h, a, dt, tm[KS ? 1 : 3], op);
        case 5:     // local order parameter: KS reads E(y) = E_a, FHN the unit phasor field staged in Y3
            a.out = rhs_out;
            return l3_launch_stage<T, MODEL, P, L3_LOC>(h, a, dt, tm[KS ? 0 : 2], op);
        default:
            a.out = rhs_out;
            if (KS) op[0] = to[3];
            return l3_launch_stage<T, MODEL, P, L3_RHS>(h, a, dt, tm[0], op);
    }
}

// Tile autotuner ("measure, don't guess"): the score of l3_enumerate ranks tiles by geometry, but
// bank conflicts, wave quantisation and the depth of the pipeline decide among the leaders (cfg 5:
// 4.8e10 with the best-scoring tile, 5.3e10 with the best-measured one).  For nets large enough to
// matter the best-scoring tile of each of the leading tile widths is timed on one whole RK4 step
// (zeroed buffers; net_create re-zeroes the state afterwards) and the fastest is kept.  The
// arithmetic of every output is the same for every tile, so results do not depend on the pick.
// OSCNET_LAT3 (explicit geometry) or OSCNET_NO_AUTOTUNE switch it off.
template <class T, int MODEL, int P>
static int32_t l3_configure(net* h) {
    typedef L3Sh<T, MODEL, P> S;
    h->l3_force_tx = h->l3_force_sy = h->l3_force_ctas = h->l3_force_tail = 0;
    int32_t rc = l3_configure_tile<T, MODEL, P>(h);
    if (rc) return rc;
    if (getenv("OSCNET_LAT3") || getenv("OSCNET_NO_AUTOTUNE") || h->n < (1 << 19)) return NET_OK;
    // OSCNET_LAT3_PICK = "TXt,SY,CTAS,TAIL": the autotuner's pick of an earlier run (it prints the line
    // under OSCNET_VERBOSE), so that a profiler pass -- whose replays disturb the timing pass -- captures
    // the geometry the plain run used
    if (const char* e = getenv("OSCNET_LAT3_PICK")) {
        int tx = 0, sy = 0, ctas = 0, tail = 0;
        if (sscanf(e, "%d,%d,%d,%d", &tx, &sy, &ctas, &tail) == 4 && tx > 0 && sy > 0) {
            h->l3_force_tx = tx; h->l3_force_sy = sy; h->l3_force_ctas = ctas; h->l3_force_tail = tail;
            return l3_configure_tile<T, MODEL, P>(h);
        }
    }
    struct Cand { int tx, sy; double score; int ctas, tail; };
    constexpr int KMAX = 10;
    Cand cand[KMAX];
    int nc = 0;
    l3_enumerate<T, MODEL, P>(h->tv.nx, h->tv.ny, 0, 0, [&](int TXt, int SY, double score) {
        for (int q = 0; q < nc; ++q)
            if (cand[q].tx == TXt) {           // one entry per tile width: its best SY
                if (score > cand[q].score) { cand[q].sy = SY; cand[q].score = score; }
                return;
            }
        if (nc < KMAX) { cand[nc++] = Cand{TXt, SY, score, 2, 0}; return; }
        int worst = 0;
        for (int q = 1; q < nc; ++q) if (cand[q].score < cand[worst].score) worst = q;
        if (score > cand[worst].score) cand[worst] = Cand{TXt, SY, score, 2, 0};
    });
    const size_t sb = h->state_bytes;
    OSC_CUDA(h, cudaMemsetAsync(h->b.y, 0, sb, h->stream));
    OSC_CUDA(h, cudaMemsetAsync(h->b.Y2, 0, sb, h->stream));
    OSC_CUDA(h, cudaMemsetAsync(h->b.Y3, 0, sb, h->stream));
    OSC_CUDA(h, cudaMemsetAsync(h->b.Y4, 0, sb, h->stream));
    OSC_CUDA(h, cudaMemsetAsync(h->b.elem_param, 0, (size_t)h->ld * h->esize, h->stream));
    if (MODEL == NET_MODEL_KS) {
        const size_t eb = (size_t)h->lat3[0].plane * 2 * sizeof(T);
        OSC_CUDA(h, cudaMemsetAsync(h->E_a, 0, eb, h->stream));
        OSC_CUDA(h, cudaMemsetAsync(h->E_b, 0, eb, h->stream));
    }
    cudaEvent_t e0, e1;
    OSC_CUDA(h, cudaEventCreate(&e0));
    OSC_CUDA(h, cudaEventCreate(&e1));
    float best_ms = -1.f;
    int best = -1;
    const int64_t launches_before = h->launches;
    auto time_cand = [&](const Cand& c, float* ms_out) -> bool {
        h->l3_force_tx = c.tx; h->l3_force_sy = c.sy; h->l3_force_ctas = c.ctas; h->l3_force_tail = c.tail;
        if (l3_configure_tile<T, MODEL, P>(h) != NET_OK) return false;
        float ms = 0.f;
        bool ok = true;
        // one warm-up pass, then the fastest of three timed passes (a single pass is noisy enough to
        // flip the ranking of tiles a few per cent apart)
        for (int rep = 0; rep < 4 && ok; ++rep) {
            ok = cudaEventRecord(e0, h->stream) == cudaSuccess;
            for (int st = 0; st < 4 && ok; ++st) ok = l3_stage<T, MODEL, P>(h, st, 1e-3, nullptr) == NET_OK;   // one whole RK4 step
            float one = 0.f;
            ok = ok && cudaEventRecord(e1, h->stream) == cudaSuccess && cudaEventSynchronize(e1) == cudaSuccess &&
                 cudaEventElapsedTime(&one, e0, e1) == cudaSuccess;
            if (rep >= 1 && (rep == 1 || one < ms)) ms = one;
        }
        if (getenv("OSCNET_VERBOSE"))
            fprintf(stderr, "lat3 autotune: tile %dx%d ctas %d %s grid %u (%d x %d planes) score %.3f -> %.3f ms%s\n", c.tx, c.sy * S::TY, c.ctas,
                    c.tail < 0 ? "aligned" : "tail ok", h->lat3_grid[0], h->lat3[0].nchunks, h->lat3[0].Lz, c.score, ms, ok ? "" : " (failed)");
        *ms_out = ms;
        return ok;
    };
    // every tile at three pipeline depths (the deepest that leaves 2, 3, 4 CTAs' worth of shared
    // memory): deeper is not better -- cfg 3a, tile 40x8: D = 2 2.3e10, D = 4 2.0e10 osc-steps/s
    // and with / without a tail of spans in the last wave (the tail fills the SMs a chunk-aligned grid
    // leaves half empty, but its CTAs do not march in step with their neighbours: cfg 3b gains, cfg 5 loses)
    Cand best_c = Cand{0, 0, 0.0, 0, 0};
    for (int q = 0; q < nc; ++q)
        for (int ctas = 2; ctas <= 4; ++ctas)
            for (int tail = -1; tail <= 0; ++tail) {
                Cand c = cand[q];
                c.ctas = ctas; c.tail = tail;
                if (tail == 0) {             // same grid as the aligned pick: nothing new to time
                    h->l3_force_tx = c.tx; h->l3_force_sy = c.sy; h->l3_force_ctas = c.ctas; h->l3_force_tail = -1;
                    if (l3_configure_tile<T, MODEL, P>(h) != NET_OK) continue;
                    const unsigned ga = h->lat3_grid[0];
                    const int la = h->lat3[0].Lz;
                    h->l3_force_tail = 0;
                    if (l3_configure_tile<T, MODEL, P>(h) != NET_OK || (h->lat3_grid[0] == ga && h->lat3[0].Lz == la)) continue;
                }
                float ms;
                if (time_cand(c, &ms) && (best < 0 || ms < best_ms)) { best = q; best_ms = ms; best_c = c; }
            }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    h->launches = launches_before;
    if (cudaGetLastError() != cudaSuccess) best = -1;
    if (best >= 0) { h->l3_force_tx = best_c.tx; h->l3_force_sy = best_c.sy; h->l3_force_ctas = best_c.ctas; h->l3_force_tail = best_c.tail; }
    else h->l3_force_tx = h->l3_force_sy = h->l3_force_ctas = h->l3_force_tail = 0;
    if (getenv("OSCNET_VERBOSE"))
        fprintf(stderr, "lat3 autotune pick: OSCNET_LAT3_PICK=%d,%d,%d,%d\n", h->l3_force_tx, h->l3_force_sy, h->l3_force_ctas, h->l3_force_tail);
    return l3_configure_tile<T, MODEL, P>(h);
}

// entry point of one (dtype, model, radius), for radii that have a translation unit of their own
template <class T, int MODEL, int P>
static int32_t l3_entry_p(net* h, int stage, double dt, void* rhs_out) {
    if (h->tv.P != P) return NET_ERR_UNSUPPORTED;
    return stage < 0 ? l3_configure<T, MODEL, P>(h) : l3_stage<T, MODEL, P>(h, stage, dt, rhs_out);
}

// entry point of one (dtype, model): configure (stage < 0) or launch
template <class T, int MODEL>
static int32_t l3_entry(net* h, int stage, double dt, void* rhs_out) {
    const int P = h->tv.P;
    if (P == 2) return stage < 0 ? l3_configure<T, MODEL, 2>(h) : l3_stage<T, MODEL, 2>(h, stage, dt, rhs_out);
    if (P == 4) return stage < 0 ? l3_configure<T, MODEL, 4>(h) : l3_stage<T, MODEL, 4>(h, stage, dt, rhs_out);
    return NET_ERR_UNSUPPORTED;
}

}  // namespace oscnet
