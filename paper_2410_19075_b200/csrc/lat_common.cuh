// Helpers shared by the tiled 3D lattice kernels: packed pair adds, the x-run geometry of the
// ball of PAPER.md:313, mbarrier / TMA PTX wrappers, vector global loads and stores.
#pragma once
#include <cuda.h>

#include <type_traits>

#include "models.cuh"

namespace oscnet {

// ------------------------------------------------------------------ pairs
template <class T> struct PairOf;
template <> struct PairOf<float> { typedef float2 type; };
template <> struct PairOf<double> { typedef double2 type; };

__device__ __forceinline__ float2 padd(float2 a, float2 b) {
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;"
        : "=l"(r)
        : "l"(*reinterpret_cast<unsigned long long*>(&a)), "l"(*reinterpret_cast<unsigned long long*>(&b)));
    return *reinterpret_cast<float2*>(&r);
}
__device__ __forceinline__ double2 padd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }

// half-width of the x-run at (|dz|, |dy|), -1 if the row does not meet the ball
__host__ __device__ constexpr int l2_isqrt(int v) { int r = 0; while ((r + 1) * (r + 1) <= v) ++r; return r; }
__host__ __device__ constexpr int l2_run_w(int P, int adz, int ady) {
    int r = P * P - adz * adz - ady * ady;
    return r < 0 ? -1 : l2_isqrt(r);
}

// ------------------------------------------------------------------ PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* tmap, int c0, int c1, int c2, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(smem_u32(dst)), "l"(tmap), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2) : "memory");
}

__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* tmap, int c0, int c1, int c2, int c3, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
        ::"r"(smem_u32(dst)), "l"(tmap), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}

// N contiguous scalars from / to 16-byte (8-byte when N*sizeof == 8) aligned global memory
template <int N>
__device__ __forceinline__ void ldg_vec(const float* p, float (&v)[N]) {
    if constexpr (N % 4 == 0) {
#pragma unroll
        for (int c = 0; c < N / 4; ++c) {
            const float4 w = reinterpret_cast<const float4*>(p)[c];
            v[4 * c] = w.x; v[4 * c + 1] = w.y; v[4 * c + 2] = w.z; v[4 * c + 3] = w.w;
        }
    } else if constexpr (N % 2 == 0) {
#pragma unroll
        for (int c = 0; c < N / 2; ++c) {
            const float2 w = reinterpret_cast<const float2*>(p)[c];
            v[2 * c] = w.x; v[2 * c + 1] = w.y;
        }
    } else {
#pragma unroll
        for (int c = 0; c < N; ++c) v[c] = p[c];
    }
}
template <int N>
__device__ __forceinline__ void ldg_vec(const double* p, double (&v)[N]) {
    if constexpr (N % 2 == 0) {
#pragma unroll
        for (int c = 0; c < N / 2; ++c) {
            const double2 w = reinterpret_cast<const double2*>(p)[c];
            v[2 * c] = w.x; v[2 * c + 1] = w.y;
        }
    } else {
#pragma unroll
        for (int c = 0; c < N; ++c) v[c] = p[c];
    }
}
template <int N>
__device__ __forceinline__ void stg_vec(float* p, const float (&v)[N]) {
    if constexpr (N % 4 == 0) {
#pragma unroll
        for (int c = 0; c < N / 4; ++c)
            reinterpret_cast<float4*>(p)[c] = make_float4(v[4 * c], v[4 * c + 1], v[4 * c + 2], v[4 * c + 3]);
    } else if constexpr (N % 2 == 0) {
#pragma unroll
        for (int c = 0; c < N / 2; ++c) reinterpret_cast<float2*>(p)[c] = make_float2(v[2 * c], v[2 * c + 1]);
    } else {
#pragma unroll
        for (int c = 0; c < N; ++c) p[c] = v[c];
    }
}
template <int N>
__device__ __forceinline__ void stg_vec(double* p, const double (&v)[N]) {
    if constexpr (N % 2 == 0) {
#pragma unroll
        for (int c = 0; c < N / 2; ++c) reinterpret_cast<double2*>(p)[c] = make_double2(v[2 * c], v[2 * c + 1]);
    } else {
#pragma unroll
        for (int c = 0; c < N; ++c) p[c] = v[c];
    }
}

template <class T> __host__ __device__ constexpr int l2_hx(int P) {
    // x halo in pairs, rounded up so that every staged row piece is a multiple of 16 bytes
    return sizeof(T) == 4 ? (P + 1) / 2 * 2 : P;
}

template <int J, int N, class F>
__device__ __forceinline__ void l2_static_for(F&& f) {
    if constexpr (J < N) {
        f(std::integral_constant<int, J>{});
        l2_static_for<J + 1, N>(f);
    }
}


__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

}  // namespace oscnet
