// Host side of the second-generation 3D lattice kernels: tile / chunk selection, TMA tensor
// maps of the ghost-padded pair arrays, shared-memory opt-in, launch.  Included by
// lattice_v2_f32.cu and lattice_v2_f64.cu (one dtype per translation unit keeps the build parallel).
#pragma once
#include <stdlib.h>

#include "lattice_v2.cuh"

namespace oscnet {

// thread shape per (dtype, P): X columns x TY rows per thread, CTA size bound
template <class T, int P> struct L2Shape;
template <> struct L2Shape<float, 2> { static constexpr int X = 2, TY = 4, MAXT = 384; };
template <> struct L2Shape<float, 4> { static constexpr int X = 2, TY = 2, MAXT = 256; };
template <> struct L2Shape<double, 2> { static constexpr int X = 2, TY = 2, MAXT = 256; };
template <> struct L2Shape<double, 4> { static constexpr int X = 2, TY = 1, MAXT = 256; };

inline size_t l2_smem_bytes(const Lat2& g, size_t pair_bytes) {
    const size_t plane = ((size_t)g.PW * g.PH * pair_bytes + 127) / 128 * 128;
    return 128 + (size_t)g.NS * plane;
}

// One 3D tensor map per pair array: 8-byte elements, (nxp*U8, nyp, nz), box (PW*U8, PH, 1).
inline int32_t l2_encode_tmap(net* h, CUtensorMap* tm, void* base, const Lat2& g, int HX, int P, size_t pair_bytes) {
    typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn encode = nullptr;
    if (!encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
        if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn)
            return set_err(h, NET_ERR_CUDA, "cuTensorMapEncodeTiled is not available from the driver");
        encode = (encode_fn)fn;
    }
    const cuuint64_t u8 = pair_bytes / 8;
    const cuuint64_t nxp = (cuuint64_t)g.nx + 2 * HX, nyp = (cuuint64_t)g.ny + 2 * P;
    cuuint64_t dims[3] = {nxp * u8, nyp, (cuuint64_t)g.nz};
    cuuint64_t strides[2] = {nxp * pair_bytes, nxp * nyp * pair_bytes};
    cuuint32_t box[3] = {(cuuint32_t)(g.PW * u8), (cuuint32_t)g.PH, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = encode(tm, CU_TENSOR_MAP_DATA_TYPE_UINT64, 3, base, dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                        CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return set_err(h, NET_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
    return NET_OK;
}

// Tile selection.  xy tiles as wide as the CTA allows (small halo fraction), z chunks as long as
// the grid allows (every chunk recomputes the in-plane sums of its 2P halo planes), as many
// planes in flight as shared memory holds.  OSCNET_LAT2 = "TXt,TYt,Lz,D" overrides (tuning).
template <class T, int MODEL, int P>
static int32_t l2_configure(net* h) {
    typedef L2Shape<T, P> S;
    constexpr int X = S::X, TY = S::TY, MAXT = S::MAXT;
    constexpr int HX = l2_hx<T>(P);
    constexpr int U8 = 2 * (int)sizeof(T) / 8;
    const TopoView& tv = h->tv;
    Lat2 g;
    memset(&g, 0, sizeof(g));
    g.nx = tv.nx; g.ny = tv.ny; g.nz = tv.nz;
    g.include_self = tv.include_self;
    g.n_ball = tv.noff + (tv.include_self ? 0 : 1);
    if (g.nx % X != 0 || (g.nx * (int)sizeof(T) * 2) % 16 != 0) return NET_ERR_UNSUPPORTED;
    int want_tx = 0, want_ty = 0, want_lz = 0, want_d = 0;
    if (const char* e = getenv("OSCNET_LAT2")) sscanf(e, "%d,%d,%d,%d", &want_tx, &want_ty, &want_lz, &want_d);
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    // x: fewest tiles such that a tile row is at most 64 threads and the TMA box at most 256 elements
    int max_tx = 64 * X;
    if ((max_tx + 2 * HX) * U8 > 256) max_tx = (256 / U8 - 2 * HX) / X * X;
    g.tiles_x = (g.nx + max_tx - 1) / max_tx;
    g.TXt = ((g.nx + g.tiles_x - 1) / g.tiles_x + X - 1) / X * X;
    if (want_tx > 0) g.TXt = (want_tx + X - 1) / X * X;
    if (g.TXt > g.nx) g.TXt = g.nx;
    g.tiles_x = (g.nx + g.TXt - 1) / g.TXt;
    g.QX = g.TXt / X;
    int strips = (g.ny + TY - 1) / TY;
    g.SY = MAXT / g.QX < strips ? MAXT / g.QX : strips;
    if (want_ty > 0) g.SY = (want_ty + TY - 1) / TY;
    if (g.SY < 1 || g.QX * g.SY > MAXT) return NET_ERR_UNSUPPORTED;
    g.TYt = g.SY * TY;
    g.tiles_y = (g.ny + g.TYt - 1) / g.TYt;
    g.PW = g.TXt + 2 * HX;
    g.PH = g.TYt + 2 * P;
    if (g.PW * U8 > 256 || g.PH > 256) return NET_ERR_UNSUPPORTED;
    g.D = want_d > 0 ? want_d : 6;
    g.NS = P + 1 + g.D;
    const int threads = (g.QX * g.SY + 31) / 32 * 32;
    size_t smem = l2_smem_bytes(g, 2 * sizeof(T));
    while (smem > 200 * 1024 && g.D > 1) { g.D -= 1; g.NS -= 1; smem = l2_smem_bytes(g, 2 * sizeof(T)); }
    if (smem > 220 * 1024) return NET_ERR_UNSUPPORTED;
    constexpr int NOPS_BIG = MODEL == NET_MODEL_KS ? 3 : 2;
    auto kern = lattice3d_v2_kernel<T, MODEL, P, X, TY, 1, MAXT>;
    OSC_CUDA(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    OSC_CUDA(h, cudaFuncSetAttribute(lattice3d_v2_kernel<T, MODEL, P, X, TY, 0, MAXT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    OSC_CUDA(h, cudaFuncSetAttribute(lattice3d_v2_kernel<T, MODEL, P, X, TY, NOPS_BIG, MAXT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    OSC_CUDA(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, threads, smem));
    if (occ < 1) return NET_ERR_UNSUPPORTED;
    const int64_t slots = (int64_t)occ * sms, tiles = (int64_t)g.tiles_x * g.tiles_y;
    int64_t best_cost = -1;
    for (int nch = 1; nch <= g.nz; ++nch) {
        const int Lz = (g.nz + nch - 1) / nch;
        const int chunks = (g.nz + Lz - 1) / Lz;
        const int64_t waves = (tiles * chunks + slots - 1) / slots;
        const int64_t cost = waves * (Lz + 2 * P + 2);
        if (best_cost < 0 || cost < best_cost) { best_cost = cost; g.Lz = Lz; g.nchunks = chunks; }
    }
    if (want_lz > 0) { g.Lz = want_lz; g.nchunks = (g.nz + g.Lz - 1) / g.Lz; }
    h->lat2 = g;
    h->lat2_threads = threads;
    h->lat2_smem = smem;
    h->lat2_grid = (unsigned)(tiles * g.nchunks);
    // tensor maps of the stencil sources
    void* src[4] = {h->b.y, h->b.Y2, h->b.Y3, h->b.Y4};
    if (MODEL == NET_MODEL_KS) { src[0] = h->E_a; src[1] = h->E_b; }
    for (int k = 0; k < (MODEL == NET_MODEL_KS ? 2 : 4); ++k) {
        int32_t rc = l2_encode_tmap(h, &h->tmap[k], src[k], g, HX, P, 2 * sizeof(T));
        if (rc) return rc;
    }
    return NET_OK;
}

template <class T, int MODEL, int P, int NOPS>
static int32_t l2_launch_n(net* h, const Lat2Args& a, int which_map) {
    typedef L2Shape<T, P> S;
    auto kern = lattice3d_v2_kernel<T, MODEL, P, S::X, S::TY, NOPS, S::MAXT>;
    kern<<<h->lat2_grid, h->lat2_threads, h->lat2_smem, h->stream>>>(h->tmap[which_map], a, h->mp, h->lat2);
    h->launches += 1;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

template <class T, int MODEL, int P>
static int32_t l2_launch(net* h, const Lat2Args& a, int nops, int which_map) {
    switch (nops) {
        case 0: return l2_launch_n<T, MODEL, P, 0>(h, a, which_map);
        case 1: return l2_launch_n<T, MODEL, P, 1>(h, a, which_map);
        case 2:
            if constexpr (MODEL == NET_MODEL_FHN) return l2_launch_n<T, MODEL, P, 2>(h, a, which_map);
            break;
        case 3:
            if constexpr (MODEL == NET_MODEL_KS) return l2_launch_n<T, MODEL, P, 3>(h, a, which_map);
            break;
        default: break;
    }
    return NET_ERR_INVALID;
}

// entry point of one dtype: configure (a == nullptr) or launch
template <class T>
static int32_t l2_entry(net* h, const Lat2Args* a, int nops, int which_map) {
    const int P = h->tv.P;
    const bool ks = h->desc.model == NET_MODEL_KS;
#define L2_DISPATCH(PP)                                                                    \
    if (P == PP) {                                                                         \
        if (ks) return a ? l2_launch<T, NET_MODEL_KS, PP>(h, *a, nops, which_map)          \
                         : l2_configure<T, NET_MODEL_KS, PP>(h);                           \
        return a ? l2_launch<T, NET_MODEL_FHN, PP>(h, *a, nops, which_map)                 \
                 : l2_configure<T, NET_MODEL_FHN, PP>(h);                                  \
    }
    L2_DISPATCH(2)
    L2_DISPATCH(4)
#undef L2_DISPATCH
    return NET_ERR_UNSUPPORTED;
}

}  // namespace oscnet
