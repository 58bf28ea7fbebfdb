// Local vector fields of the three model classes (device functions, T = float | double).
// Equations: include/oscnet.h (net_*_params) and PAPER.md eq. (1)-(3).
#pragma once
#include "oscnet_internal.cuh"

namespace oscnet {

template <class T> struct Math;
template <> struct Math<double> {
    static __device__ __forceinline__ double exp(double x) { return ::exp(x); }
    static __device__ __forceinline__ double expm1(double x) { return ::expm1(x); }
    static __device__ __forceinline__ double sin(double x) { return ::sin(x); }
    static __device__ __forceinline__ void sincos(double x, double* s, double* c) { ::sincos(x, s, c); }
    static __device__ __forceinline__ double abs(double x) { return ::fabs(x); }
};
template <> struct Math<float> {
    static __device__ __forceinline__ float exp(float x) { return ::expf(x); }
    static __device__ __forceinline__ float expm1(float x) { return ::expm1f(x); }
    static __device__ __forceinline__ float sin(float x) { return ::sinf(x); }
    static __device__ __forceinline__ void sincos(float x, float* s, float* c) { ::sincosf(x, s, c); }
    static __device__ __forceinline__ float abs(float x) { return ::fabsf(x); }
};

// (sin, cos) of an unwrapped fp32 phase on the SFU: two-term Cody-Waite reduction to [-pi, pi]
// (k = rint(x / 2 pi), r = x - k * 2 pi with 2 pi split hi + lo), then MUFU.SIN / MUFU.COS.
// Absolute error about 5e-7 for |x| up to a few 1e4 (sin.approx is 2^-20.9 on [-pi, pi]); the
// north star lets the sin/cos pair go to the SFU "with the error of that choice measured":
// tests/test_gpu_parity.py::test_fast_rewrite_error_against_direct_on_gpu does.  The fp64 path
// keeps the library sincos.
__device__ __forceinline__ void sincos_sfu(float x, float* s, float* c) {
    const float k = rintf(x * 0.15915494309189535f);
    float r = fmaf(k, -6.2831854820251465f, x);          // 2 pi rounded to fp32
    r = fmaf(k, 1.7484555e-7f, r);                       // minus (2 pi - fl(2 pi))
    *s = __sinf(r);
    *c = __cosf(r);
}
template <class T> __device__ __forceinline__ void sincos_stage(T x, T* s, T* c) { Math<T>::sincos(x, s, c); }
template <> __device__ __forceinline__ void sincos_stage<float>(float x, float* s, float* c) { sincos_sfu(x, s, c); }

// ----------------------------------------------------------------- Kuramoto
// Direct form: f = omega + (K/Omega) * sum_j sin(phi_j - phi_i - alpha); `sum` is that sum.
template <class T>
__device__ __forceinline__ T ks_rhs_direct(const ModelParams& mp, T omega, T sum, T inv_deg) {
    return omega + T(mp.K) * inv_deg * sum;
}
// Factorised form: with C = sum_j cos phi_j, S = sum_j sin phi_j and (ci, si) = (cos, sin) phi_i,
//   sum_j sin(phi_j - phi_i - alpha) = S cos(phi_i+alpha) - C sin(phi_i+alpha).
template <class T>
__device__ __forceinline__ T ks_rhs_factorised(const ModelParams& mp, T omega, T C, T S, T ci,
                                               T si, T inv_deg) {
    T ca = T(mp.cos_a), sa = T(mp.sin_a);
    T cia = ci * ca - si * sa;  // cos(phi_i + alpha)
    T sia = si * ca + ci * sa;  // sin(phi_i + alpha)
    return omega + T(mp.K) * inv_deg * (S * cia - C * sia);
}

// ---------------------------------------------------------- FitzHugh-Nagumo
// Cu = sum_j (u_j - u_i), Cv = sum_j (v_j - v_i).
template <class T>
__device__ __forceinline__ void fhn_rhs(const ModelParams& mp, T u, T v, T Cu, T Cv, T inv_deg,
                                        T* fu, T* fv) {
    T s = T(mp.sigma) * inv_deg;
    *fu = (u - u * u * u * T(1.0 / 3.0) - v + s * (T(mp.buu) * Cu + T(mp.buv) * Cv)) * T(mp.inv_eps);
    *fv = u + T(mp.a) + s * (T(mp.bvu) * Cu + T(mp.bvv) * Cv);
}

// ----------------------------------------------------------- Hodgkin-Huxley
// x/(1-exp(-x/10)) with the removable singularity at 0 (reading R10).
template <class T>
__device__ __forceinline__ T hh_vtrap(T x) {
    T r = x * T(0.1);
    if (Math<T>::abs(r) < T(1e-9)) return T(10);
    return -x / Math<T>::expm1(-r);
}

template <class T>
__device__ __forceinline__ void hh_rates(T V, T* am, T* bm, T* ah, T* bh, T* an, T* bn) {
    *am = T(0.1) * hh_vtrap<T>(V + T(40));
    *bm = T(4) * Math<T>::exp(-(V + T(65)) * T(1.0 / 18.0));
    *ah = T(0.07) * Math<T>::exp(-(V + T(65)) * T(1.0 / 20.0));
    *bh = T(1) / (T(1) + Math<T>::exp(-(V + T(35)) * T(0.1)));
    *an = T(0.01) * hh_vtrap<T>(V + T(55));
    *bn = T(0.125) * Math<T>::exp(-(V + T(65)) * T(1.0 / 80.0));
}

template <class T>
__device__ __forceinline__ T hh_syn_activation(const ModelParams& mp, T V) {
    return T(1) / (T(1) + Math<T>::exp(-(V - T(mp.theta_syn)) * T(mp.inv_k_syn)));
}

// ssum = sum_j S(V_j) over the in-neighbours.
template <class T>
__device__ __forceinline__ void hh_rhs(const ModelParams& mp, T V, T m, T h, T g, T Iext, T ssum,
                                       T inv_deg, T* fV, T* fm, T* fh, T* fg) {
    T am, bm, ah, bh, an, bn;
    hh_rates<T>(V, &am, &bm, &ah, &bh, &an, &bn);
    T INa = T(mp.gNa) * m * m * m * h * (V - T(mp.ENa));
    T g2 = g * g;
    T IK = T(mp.gK) * g2 * g2 * (V - T(mp.EK));
    T IL = T(mp.gL) * (V - T(mp.EL));
    T Isyn = T(mp.g_syn) * inv_deg * (T(mp.E_syn) - V) * ssum;
    *fV = (Iext - INa - IK - IL + Isyn) * T(mp.inv_C);
    *fm = am * (T(1) - m) - bm * m;
    *fh = ah * (T(1) - h) - bh * h;
    *fg = an * (T(1) - g) - bn * g;
}

// --------------------------------------------------------------- neighbours
// Calls f(j) for every in-neighbour j of element i, and returns the in-degree.
template <int TOPO, class F>
__device__ __forceinline__ int for_each_neighbor_local(const TopoView& tv, int64_t n, int64_t i, F&& f);

// A batch of B replicas of a net of rn elements is ONE net of B * rn elements whose coupling matrix is
// block diagonal: element i belongs to replica i / rn, its neighbours are
// those of its local index inside that replica.  The topology arrays describe ONE replica.
template <int TOPO, class F>
__device__ __forceinline__ int for_each_neighbor(const TopoView& tv, int64_t n, int64_t i, F&& f) {
    const int64_t rn = tv.ring_n;
    if (TOPO == NET_TOPO_RING || rn == n) return for_each_neighbor_local<TOPO>(tv, n, i, f);
    const int64_t base = i / rn * rn;
    return for_each_neighbor_local<TOPO>(tv, rn, i - base, [&](int64_t j) { f(base + j); });
}

template <int TOPO, class F>
__device__ __forceinline__ int for_each_neighbor_local(const TopoView& tv, int64_t n, int64_t i, F&& f) {
    if (TOPO == NET_TOPO_RING) {
        int P = tv.P;
        const int64_t rn = tv.ring_n, base = i / rn * rn;    // a batch is block diagonal: rings of rn elements
        for (int d = -P; d <= P; ++d) {
            if (d == 0 && !tv.include_self) continue;
            int64_t j = i - base + d;
            if (j < 0) j += rn;
            if (j >= rn) j -= rn;
            f(base + j);
        }
        return 2 * P + (tv.include_self ? 1 : 0);
    } else if (TOPO == NET_TOPO_LATTICE) {
        int nx = tv.nx, ny = tv.ny, nz = tv.nz;
        int x = (int)(i % nx);
        int64_t r = i / nx;
        int y = (int)(r % ny);
        int z = (int)(r / ny);
        for (int q = 0; q < tv.noff; ++q) {
            int xx = x + tv.off[3 * q], yy = y + tv.off[3 * q + 1], zz = z + tv.off[3 * q + 2];
            xx += (xx < 0) ? nx : 0; xx -= (xx >= nx) ? nx : 0;
            yy += (yy < 0) ? ny : 0; yy -= (yy >= ny) ? ny : 0;
            zz += (zz < 0) ? nz : 0; zz -= (zz >= nz) ? nz : 0;
            f(((int64_t)zz * ny + yy) * nx + xx);
        }
        return tv.noff;
    } else if (TOPO == NET_TOPO_COMPRESSED) {
        // EXTRACT of Alg. 2: row i = (p + i) mod n for p in XOR(V, D[C_i])
        const int c = tv.cmp_c[i];
        int64_t b = tv.cmp_dptr[c];
        const int64_t be = tv.cmp_dptr[c + 1];
        const int ae = tv.cmp_vlen;
        if (b == be) {                      // empty difference: the common pattern shifted by i
            for (int a = 0; a < ae; ++a) {
                int64_t j = i + tv.cmp_v[a];
                if (j >= n) j -= n;
                f(j);
            }
            return ae;
        }
        int a = 0, deg = 0;                 // symmetric difference of two sorted position lists
        while (a < ae || b < be) {
            const int32_t pv = a < ae ? tv.cmp_v[a] : 0x7fffffff;
            const int32_t pd = b < be ? tv.cmp_dpos[b] : 0x7fffffff;
            if (pv == pd) { ++a; ++b; continue; }
            int64_t j = i + (pv < pd ? pv : pd);
            if (pv < pd) ++a; else ++b;
            if (j >= n) j -= n;
            f(j);
            ++deg;
        }
        return deg;
    } else if (TOPO == NET_TOPO_CSR) {
        int64_t b = tv.row_ptr[i], e = tv.row_ptr[i + 1];
        for (int64_t q = b; q < e; ++q) f((int64_t)tv.col_idx[q]);
        return (int)(e - b);
    } else {
        int k = tv.k_uniform;
        const int32_t* row = tv.col_idx + i * (int64_t)k;
        for (int q = 0; q < k; ++q) f((int64_t)row[q]);
        return k;
    }
}

}  // namespace oscnet
