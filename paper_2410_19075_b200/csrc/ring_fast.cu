// FAST method for rings (configs 1 and 2): one persistent cooperative kernel integrates all
// n_steps; the coupling window sum over |j-i| <= P is a difference of
// prefix sums, exact in real arithmetic.
//
// Both ring models reduce to the window sum of NF = 2 fields: FHN (eq. (2))
// is linear, sum_j (u_j - u_i) = W_u(i) - (2P+1) u_i; for KS (eq. (3)) the sine is
// factorised, sum_j sin(phi_j - phi_i - a) = S_i cos(phi_i + a) - C_i sin(phi_i + a) with
// (C, S) the window sums of (cos phi, sin phi) -- one sincos per element per stage instead of
// one sine per link.
//
// These nets are latency-bound (2 KB / 1 MB of state), so the whole run is one launch: every
// thread keeps its E elements (base state, stage state, RK4 accumulator) in registers for all
// steps.  CTA b owns the contiguous chunk [b*chunk, (b+1)*chunk).  Per stage:
//   A. fields of the stage state -> inclusive prefix inside the chunk (thread-serial, warp
//      shuffles, warp totals) -> Sloc[f][i] and the chunk total tot[f][b] to global memory (L2);
//   B. ONE grid barrier (monotonic counter in L2; co-residency guaranteed by the cooperative
//      launch); single-CTA nets (config 1) use shared memory and __syncthreads instead;
//   C. every CTA scans the G chunk totals (double) into exclusive block offsets BT, and each
//      element forms W(i) = Pref(i+P) - Pref(i-P-1), Pref(j) = BT[blk(j)] + Sloc[j], with the
//      ring wrap taken as one extra full-ring term; local vector field; RK4 update in registers.
// Sloc/tot are double-buffered over consecutive stages, so one barrier per stage suffices.
// The cancellation of the prefix differences is bounded by (chunk length) x ulp x max|field| on
// Sloc plus G x ulp(double) on BT; the RHS divides it by Omega (measured: tests).
#include <cooperative_groups.h>
#include <stdlib.h>

#include "models.cuh"

namespace oscnet {

constexpr int RING_THREADS = 256;
constexpr int RING_GMAX = RING_THREADS;   // the chunk totals are scanned in one pass by one CTA
constexpr int RING_NT_SINGLE = 256;       // threads of a single-CTA ring / of every ring of a batch unless OSCNET_RING_NT
constexpr int RING_NT_BATCH = 128;        // says otherwise (measured, see ring_plan)

struct RingArgs {
    const void* y_in;        // [nvar][ld] state the run starts from / RHS is evaluated on
    void* y_out;             // integrate: final state (may alias y_in); rhs_only: f(y_in)
    const void* elem_param;  // omega_i (KS)
    void* S[2];              // 2 x [2][npad] prefix buffers (T)
    double* tot[2];          // 2 x [2][RING_GMAX] chunk totals
    unsigned int* bar;       // grid barrier counter (zeroed before the launch)
    int64_t n, ld, npad;     // n: elements per ring (a batch holds several rings back to back)
    int32_t P, include_self, chunk, G, chunk_shift;
    int32_t barrier_flags;   // 1: flag-array grid barrier, 0: shared counter
    int64_t n_steps;
    double dt;
    int32_t rhs_only;
    // phase models: order-parameter samples taken inside the launch (net_integrate_observed).  The
    // block totals of (cos phi, sin phi) that stage 0 of a step scans anyway ARE the sums of the
    // global order parameter of the state at that step, so a sample costs one 16-byte store.
    int64_t obs_every;       // 0: no sampling; else the state at steps obs_first, obs_first + obs_every, ... < n_steps
    int64_t obs_first;
    double* obs_cs;          // [sample][ring][2] = sum cos phi, sum sin phi over the ring
    double* obs_ref;         // phi of every element at step obs_first (start of the velocity window)
};

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_add_u32(unsigned* p, unsigned v) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

__device__ __forceinline__ void st_release_u32(unsigned* p, unsigned v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// Grid barrier over G co-resident CTAs (cooperative launch), G <= RING_THREADS.
// Counter form (default): one red.release.add per CTA on a shared counter, thread 0 polls it.
// Flag form (OSCNET_RING_BARRIER=flags, tried in round 2 to avoid the read-modify-write that L2
// serialises over G arrivals): CTA b publishes the epoch in its own word flags[b] (one release
// store); thread t < G of every CTA polls flags[t] (acquire), all G words in parallel.  Measured
// over 128 CTAs (net_probe_latency): 5.47 us against 1.21 us for the counter -- 16 384 polling
// threads with acquire loads cost far more than 128 serialised reds; config 2 2.3e9 against 5.7e9
// osc-steps/s.  Kept only as the record of that measurement.
__device__ __forceinline__ void grid_barrier(unsigned* bar, unsigned epoch, int G, int flags_form) {
    __syncthreads();
    if (flags_form) {
        if (threadIdx.x == 0) st_release_u32(bar + blockIdx.x, epoch);
        if ((int)threadIdx.x < G) while (ld_acquire_u32(bar + threadIdx.x) < epoch) {}
    } else if (threadIdx.x == 0) {
        red_release_add_u32(bar, 1u);
        while (ld_acquire_u32(bar) < epoch * (unsigned)G) {}
    }
    __syncthreads();
}

template <class T> __device__ __forceinline__ T ld_l2(const T* p) { return __ldcg(p); }
template <class T> __device__ __forceinline__ void st_l2(T* p, T v) { __stcg(p, v); }

// Inclusive block scan of two values per thread (a, b); returns the block totals through
// (ta, tb).  wsum: shared scratch [2][RING_THREADS/32].  TAIL_SYNC = false: the caller has a CTA
// barrier of its own before wsum is written again.  (A radix-4 warp scan with a tree over the
// warp totals -- fewer dependent levels, more shuffles -- was measured slower: 0.35 against
// 0.34 us per scan, config 1b 2.29e10 against 2.51e10.)
template <class A, bool TAIL_SYNC, int NT = RING_THREADS>
__device__ __forceinline__ void block_scan2(A& a, A& b, A& ta, A& tb, A (*wsum)[NT / 32]) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        A ua = __shfl_up_sync(0xffffffffu, a, o), ub = __shfl_up_sync(0xffffffffu, b, o);
        if (lane >= o) { a += ua; b += ub; }
    }
    if (lane == 31) { wsum[0][warp] = a; wsum[1][warp] = b; }
    __syncthreads();
    A oa = 0, ob = 0, sa = 0, sb = 0;
#pragma unroll
    for (int w = 0; w < NT / 32; ++w) {
        const A va = wsum[0][w], vb = wsum[1][w];
        if (w < warp) { oa += va; ob += vb; }
        sa += va; sb += vb;
    }
    a += oa; b += ob;
    ta = sa; tb = sb;
    if (TAIL_SYNC) __syncthreads();
}

// NT: threads per CTA.  Multi-CTA rings always run RING_THREADS; single-CTA rings (config 1 and the
// batches) may run fewer, wider threads: fewer warps shorten the scan over the warp totals and the
// CTA barriers, more elements per thread lengthen the serial part (sincos, thread-local prefix).
// OBS: the launch takes order-parameter samples (a separate instance: the plain kernel carries none
// of it -- the first version, with the test inside the one kernel, cost config 1 20 %).
template <class T, int MODEL, int E, bool SINGLE, int NT = RING_THREADS, bool OBS = false>
__global__ void __launch_bounds__(NT) ring_persistent_kernel(RingArgs a, ModelParams mp) {
    // KS: phi | FHN: (u, v) | KS with inertia (eq. (3) in full): (phi, psi = dphi/dt), fields as for KS
    constexpr int NV = MODEL == NET_MODEL_KS ? 1 : 2;
    constexpr bool PHASE = MODEL == NET_MODEL_KS || MODEL == NET_MODEL_KSI;
    extern __shared__ __align__(16) unsigned char ring_smem[];
    static_assert(SINGLE || NT == RING_THREADS, "multi-CTA rings scan the chunk totals with RING_THREADS threads");
    __shared__ T wsumT[2][NT / 32];
    __shared__ double wsumD[2][NT / 32];
    __shared__ double BT[2][RING_GMAX + 1];

    const int64_t n = a.n, ld = a.ld;
    const int chunk = a.chunk, G = a.G, P = a.P;
    // single-CTA rings: CTA = one ring of the batch; otherwise CTA = one chunk of the one ring
    const int b = SINGLE ? 0 : blockIdx.x;
    const int64_t goff = SINGLE ? (int64_t)blockIdx.x * n : 0;   // first element of this CTA's ring
    const int64_t cbeg = (int64_t)b * chunk;
    const int64_t i0 = cbeg + (int64_t)threadIdx.x * E;      // first element of this thread (inside its ring)
    const T* __restrict__ yin = (const T*)a.y_in + goff;
    const T* __restrict__ ep = (const T*)a.elem_param + goff;
    const T dt = (T)a.dt;
    const int deg = 2 * P + (a.include_self ? 1 : 0);
    const T inv_deg = deg > 0 ? T(1) / T(deg) : T(0);
    const T nwin = T(2 * P + 1);

    T y0[E][NV], x[E][NV], acc[E][NV], om[E];
    bool ok[E];
#pragma unroll
    for (int e = 0; e < E; ++e) {
        ok[e] = i0 + e < n && threadIdx.x * E + e < chunk;
        om[e] = (PHASE && ok[e]) ? ep[i0 + e] : T(0);
#pragma unroll
        for (int v = 0; v < NV; ++v) {
            y0[e][v] = ok[e] ? yin[v * ld + i0 + e] : T(0);
            x[e][v] = y0[e][v];
            acc[e][v] = T(0);
        }
    }

    const int64_t n_stage = a.rhs_only ? 1 : 4 * a.n_steps;
    [[maybe_unused]] int64_t next_sample = a.obs_first, n_sampled = 0;
    for (int64_t q = 0; q < n_stage; ++q) {
        const int stage = (int)(q & 3);
        const int buf = (int)(q & 1);
        T* Sg = SINGLE ? reinterpret_cast<T*>(ring_smem) : (T*)a.S[buf];
        const int64_t sstride = SINGLE ? (int64_t)chunk : a.npad;
        // ---- A: fields and their inclusive prefix inside the chunk
        T f0[E], f1[E];
#pragma unroll
        for (int e = 0; e < E; ++e) {
            if (PHASE) {
                T s, c;
                Math<T>::sincos(x[e][0], &s, &c);
                f0[e] = ok[e] ? c : T(0);
                f1[e] = ok[e] ? s : T(0);
            } else {
                // padding lanes of a ragged last chunk carry no field: their registers drift away
                // from zero under the RK4 update (fhn_rhs(0,0) = (0, a)), so mask like the phase models
                f0[e] = ok[e] ? x[e][0] : T(0);
                f1[e] = ok[e] ? x[e][NV - 1] : T(0);
            }
        }
        T p0[E], p1[E];
        p0[0] = f0[0]; p1[0] = f1[0];
#pragma unroll
        for (int e = 1; e < E; ++e) { p0[e] = p0[e - 1] + f0[e]; p1[e] = p1[e - 1] + f1[e]; }
        T s0 = p0[E - 1], s1 = p1[E - 1], t0, t1;
        block_scan2<T, false, NT>(s0, s1, t0, t1, wsumT);   // a CTA barrier follows before wsumT is reused
        const T ex0 = s0 - p0[E - 1], ex1 = s1 - p1[E - 1];   // exclusive offset of this thread
        // order-parameter sample of the state this step starts from
        [[maybe_unused]] bool sample_now = false;
        [[maybe_unused]] int64_t sample_k = 0;
        if constexpr (OBS && PHASE) {
            if (stage == 0 && (q >> 2) == next_sample) {
                const int64_t sidx = q >> 2;
                sample_now = true;
                sample_k = n_sampled++;
                next_sample += a.obs_every;
                if (SINGLE && threadIdx.x == 0) {
                    double* o = a.obs_cs + (sample_k * (int64_t)gridDim.x + blockIdx.x) * 2;
                    o[0] = (double)t0; o[1] = (double)t1;
                }
                if (sidx == a.obs_first) {
#pragma unroll
                    for (int e = 0; e < E; ++e)
                        if (ok[e]) a.obs_ref[goff + i0 + e] = (double)y0[e][0];
                }
            }
        }
#pragma unroll
        for (int e = 0; e < E; ++e) {
            if (ok[e]) {
                const int64_t at = SINGLE ? (int64_t)(threadIdx.x * E + e) : i0 + e;
                if (SINGLE) { Sg[at] = ex0 + p0[e]; Sg[sstride + at] = ex1 + p1[e]; }
                else { st_l2(Sg + at, ex0 + p0[e]); st_l2(Sg + sstride + at, ex1 + p1[e]); }
            }
        }
        if (!SINGLE && threadIdx.x == 0) {
            st_l2(a.tot[buf] + b, (double)t0);
            st_l2(a.tot[buf] + RING_GMAX + b, (double)t1);
        }
        // ---- B: every chunk's prefix is visible
        if (SINGLE) __syncthreads();
        else grid_barrier(a.bar, (unsigned)(q + 1), G, a.barrier_flags);
        // the chunk totals and the 4 E prefix values of this thread are requested together: both
        // are in flight during the same L2 round trip
        double c0 = 0.0, c1 = 0.0;
        if (!SINGLE && threadIdx.x < G) { c0 = ld_l2(a.tot[buf] + threadIdx.x); c1 = ld_l2(a.tot[buf] + RING_GMAX + threadIdx.x); }
        int64_t jh[E], jl[E];
        int nwrap[E];
        bool has_lo[E];
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int64_t i = ok[e] ? i0 + e : 0;
            int64_t hi = i + P, lo = i - P - 1;
            int w = 0;
            if (hi >= n) { hi -= n; ++w; }
            if (lo < -1) { lo += n; ++w; }
            has_lo[e] = lo >= 0;
            jh[e] = hi; jl[e] = has_lo[e] ? lo : 0;
            nwrap[e] = w;
        }
        T h0[E], h1[E], l0[E], l1[E];
#pragma unroll
        for (int e = 0; e < E; ++e) {
            h0[e] = SINGLE ? Sg[jh[e]] : ld_l2(Sg + jh[e]);
            h1[e] = SINGLE ? Sg[sstride + jh[e]] : ld_l2(Sg + sstride + jh[e]);
            l0[e] = SINGLE ? Sg[jl[e]] : ld_l2(Sg + jl[e]);
            l1[e] = SINGLE ? Sg[sstride + jl[e]] : ld_l2(Sg + sstride + jl[e]);
        }
        // ---- C: block offsets
        if (!SINGLE) {
            const double v0 = c0, v1 = c1;
            double u0, u1;
            block_scan2<double, false, NT>(c0, c1, u0, u1, wsumD);  // the __syncthreads after BT
            if (threadIdx.x < G) { BT[0][threadIdx.x] = c0 - v0; BT[1][threadIdx.x] = c1 - v1; }
            if (threadIdx.x == 0) { BT[0][G] = u0; BT[1][G] = u1; }
            if constexpr (OBS)
                if (sample_now && blockIdx.x == 0 && threadIdx.x == 0) { a.obs_cs[sample_k * 2] = u0; a.obs_cs[sample_k * 2 + 1] = u1; }
            __syncthreads();
        }
        // window sums, local field, RK4 update.  W(i) = Pref(i+P) - Pref(i-P-1) with the ring wrap
        // taken as one extra full-ring term (the total = BT[G], no load).  All 4 E prefix loads
        // of a thread are issued together, branch-free: one L2 round trip per stage, not one per
        // term (the serial form cost 1.4 us per element and stage on config 2).
        T k[E][NV];
        T W0v[E], W1v[E];
        {
#pragma unroll
            for (int e = 0; e < E; ++e) {
                double bt0 = 0.0, bt1 = 0.0;
                T sl0 = h0[e], sl1 = h1[e];
                if (!SINGLE) {
                    const int bh = (int)(jh[e] >> a.chunk_shift);   // chunk = 256 E is a power of two
                    bt0 = BT[0][bh]; bt1 = BT[1][bh];
                }
                if (has_lo[e]) {
                    sl0 -= l0[e]; sl1 -= l1[e];
                    if (!SINGLE) {
                        const int bl = (int)(jl[e] >> a.chunk_shift);
                        bt0 -= BT[0][bl]; bt1 -= BT[1][bl];
                    }
                }
                // full-ring terms: Pref(n-1) = total of the ring
                T tot0, tot1;
                if (SINGLE) { tot0 = Sg[n - 1]; tot1 = Sg[sstride + n - 1]; }
                else { tot0 = T(0); tot1 = T(0); bt0 += (double)nwrap[e] * BT[0][G]; bt1 += (double)nwrap[e] * BT[1][G]; }
                if (SINGLE) { sl0 += T(nwrap[e]) * tot0; sl1 += T(nwrap[e]) * tot1; }
                W0v[e] = ok[e] ? (T)bt0 + sl0 : T(0);
                W1v[e] = ok[e] ? (T)bt1 + sl1 : T(0);
            }
        }
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const T W0 = W0v[e], W1 = W1v[e];
            if (PHASE) {
                T C = W0, S = W1;
                if (!a.include_self) { C -= f0[e]; S -= f1[e]; }
                const T torque = ks_rhs_factorised<T>(mp, om[e], C, S, f0[e], f1[e], inv_deg);
                if (MODEL == NET_MODEL_KS) k[e][0] = torque;
                else {      // m phi'' + eps phi' = torque
                    k[e][0] = x[e][NV - 1];
                    k[e][NV - 1] = (torque - T(mp.damp) * x[e][NV - 1]) * T(mp.inv_m);
                }
            } else {
                const T Cu = W0 - nwin * f0[e], Cv = W1 - nwin * f1[e];
                fhn_rhs<T>(mp, f0[e], f1[e], Cu, Cv, inv_deg, &k[e][0], &k[e][NV - 1]);
            }
        }
        if (a.rhs_only) {
            T* out = (T*)a.y_out + goff;
#pragma unroll
            for (int e = 0; e < E; ++e)
                if (ok[e])
#pragma unroll
                    for (int v = 0; v < NV; ++v) out[v * ld + i0 + e] = k[e][v];
            return;
        }
        // textbook RK4 in registers: acc = k1 + 2 k2 + 2 k3 (+ k4)
#pragma unroll
        for (int e = 0; e < E; ++e)
#pragma unroll
            for (int v = 0; v < NV; ++v) {
                const T kv = k[e][v];
                if (stage == 0) { acc[e][v] = kv; x[e][v] = y0[e][v] + (T(0.5) * dt) * kv; }
                else if (stage == 1) { acc[e][v] += T(2) * kv; x[e][v] = y0[e][v] + (T(0.5) * dt) * kv; }
                else if (stage == 2) { acc[e][v] += T(2) * kv; x[e][v] = y0[e][v] + dt * kv; }
                else { y0[e][v] += (dt * T(1.0 / 6.0)) * (acc[e][v] + kv); x[e][v] = y0[e][v]; }
            }
        if (SINGLE) __syncthreads();   // the shared prefix buffer is rewritten by the next stage
    }
    T* out = (T*)a.y_out + goff;
#pragma unroll
    for (int e = 0; e < E; ++e)
        if (ok[e])
#pragma unroll
            for (int v = 0; v < NV; ++v) out[v * ld + i0 + e] = y0[e][v];
}

// ------------------------------------------------------------------ host side
struct RingPlan { int E, G, chunk, nt; bool single; size_t smem; };

// gmax: CTAs that can be co-resident (one per SM always can; two per SM when the occupancy
// query at launch agrees -- fewer elements per thread shorten the dependent chain of a stage)
static bool ring_plan(int64_t n, size_t esize, RingPlan* p, int gmax = 148) {
    int emin = 1;
    if (const char* e = getenv("OSCNET_RING_E")) {      // tuning aid: the chunk must stay a power of two
        const int v = atoi(e);
        if (v == 1 || v == 2 || v == 4 || v == 8) emin = v;
    }
    for (int E = emin; E <= 8; E *= 2) {
        const int64_t chunk = (int64_t)RING_THREADS * E;
        const int64_t G = (n + chunk - 1) / chunk;
        if (G <= gmax && G <= RING_GMAX) {
            p->E = E; p->G = (int)G; p->chunk = (int)chunk; p->single = G == 1; p->nt = RING_THREADS;
            // single-CTA rings: fewer, wider threads where the ring fits (instantiated: 32 x 8,
            // 64 x {4, 8}, 128 x {2, 4, 8}).  Default RING_NT_SINGLE, OSCNET_RING_NT overrides.
            if (p->single) {
                // measured on B200 (OSCNET_RING_NT sweep, bench configs 1 / 1b, osc-steps/s):
                //   threads      256      128      64       32 (one warp, 8 elements per lane)
                //   one ring   1.08e8   9.3e7    6.3e7    2.7e7   -- the fp64 sincos of 8 elements per lane is
                //                                                   issue-bound in one warp; more warps win
                //   1184 rings 2.51e10  3.42e10  3.44e10  1.83e10 -- the batch is bound by instruction issue:
                //                                                   fewer warps = less scan work per element
                int want = gmax == 1 ? RING_NT_BATCH : RING_NT_SINGLE;
                if (const char* e = getenv("OSCNET_RING_NT")) want = atoi(e);
                if (want == 32 || want == 64 || want == 128) {
                    const int emin_nt = want == 32 ? 8 : want == 64 ? 4 : 2;
                    for (int E2 = emin_nt; E2 <= 8; E2 *= 2)
                        if ((int64_t)want * E2 >= n) { p->nt = want; p->E = E2; p->chunk = want * E2; break; }
                }
            }
            p->smem = p->single ? 2 * (size_t)p->chunk * esize : 0;
            return true;
        }
    }
    return false;
}

// d->n is the total over the batch (api.cu: normalise); batches need rings that fit one CTA
bool ring_supported(const net_desc* d) {
    RingPlan p;
    const int batch = d->batch > 0 ? d->batch : 1;
    return d->topo.kind == NET_TOPO_RING &&
           (d->model == NET_MODEL_KS || d->model == NET_MODEL_FHN || d->model == NET_MODEL_KSI) &&
           ring_plan(d->n / batch, d->dtype == NET_F32 ? 4 : 8, &p, batch > 1 ? 1 : 148);
}

constexpr size_t RING_OBS_BYTES = 32u << 20;     // order-parameter samples taken inside a launch (16 bytes per sample and ring)

static size_t ring_work_bytes(int64_t n_total, size_t es) {
    const size_t npad = (size_t)round_up(n_total, 64);
    return (2 * (2 * npad * es) + 2 * (2 * RING_GMAX * sizeof(double)) + 256 + 1024 + 255) / 256 * 256;
}

size_t ring_scratch_bytes(const net_desc* d) {
    return ring_work_bytes(d->n, d->dtype == NET_F32 ? 4 : 8) + RING_OBS_BYTES;
}

template <class T, int MODEL, int E, bool SINGLE, int NT = RING_THREADS>
static int32_t ring_launch_t(net* h, RingArgs& a, const RingPlan& p) {
    constexpr bool PHASE = MODEL == NET_MODEL_KS || MODEL == NET_MODEL_KSI;
    auto kern = ring_persistent_kernel<T, MODEL, E, SINGLE, NT, false>;
    if constexpr (PHASE)
        if (a.obs_every > 0) kern = ring_persistent_kernel<T, MODEL, E, SINGLE, NT, true>;
    if (p.smem > 48 * 1024)
        OSC_CUDA(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.smem));
    if (!SINGLE && p.G > 148) {      // more than one CTA per SM: must all be resident
        int dev = 0, sms = 148, occ = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        OSC_CUDA(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, RING_THREADS, p.smem));
        if ((int64_t)occ * sms < p.G) return NET_ERR_UNSUPPORTED;
    }
    if (!SINGLE) OSC_CUDA(h, cudaMemsetAsync(a.bar, 0, sizeof(unsigned) * RING_GMAX, h->stream));
    void* params[] = {&a, &h->mp};
    if (SINGLE)      // one CTA per ring of the batch
        OSC_CUDA(h, cudaLaunchKernel((const void*)kern, dim3((unsigned)h->desc.batch), dim3(NT), params, p.smem, h->stream));
    else
        OSC_CUDA(h, cudaLaunchCooperativeKernel((const void*)kern, dim3(p.G), dim3(RING_THREADS), params, p.smem, h->stream));
    h->launches += 1;
    return NET_OK;
}

template <class T, int MODEL>
static int32_t ring_launch_e(net* h, RingArgs& a, const RingPlan& p) {
    if (p.single && p.nt == 32) return ring_launch_t<T, MODEL, 8, true, 32>(h, a, p);
    if (p.single && p.nt == 64)
        return p.E == 4 ? ring_launch_t<T, MODEL, 4, true, 64>(h, a, p) : ring_launch_t<T, MODEL, 8, true, 64>(h, a, p);
    if (p.single && p.nt == 128)
        return p.E == 2 ? ring_launch_t<T, MODEL, 2, true, 128>(h, a, p)
             : p.E == 4 ? ring_launch_t<T, MODEL, 4, true, 128>(h, a, p) : ring_launch_t<T, MODEL, 8, true, 128>(h, a, p);
    if (p.single) {
        switch (p.E) {
            case 1: return ring_launch_t<T, MODEL, 1, true>(h, a, p);
            case 2: return ring_launch_t<T, MODEL, 2, true>(h, a, p);
            case 4: return ring_launch_t<T, MODEL, 4, true>(h, a, p);
            default: return ring_launch_t<T, MODEL, 8, true>(h, a, p);
        }
    }
    switch (p.E) {
        case 1: return ring_launch_t<T, MODEL, 1, false>(h, a, p);
        case 2: return ring_launch_t<T, MODEL, 2, false>(h, a, p);
        case 4: return ring_launch_t<T, MODEL, 4, false>(h, a, p);
        default: return ring_launch_t<T, MODEL, 8, false>(h, a, p);
    }
}

static int ring_barrier_flags() {
    const char* e = getenv("OSCNET_RING_BARRIER");
    return e && e[0] == 'f';
}

// y_in -> y_out over n_steps RK4 steps (rhs_only: y_out = f(y_in))
static int32_t ring_run_plan(net* h, const RingPlan& p, const void* y_in, void* y_out, int64_t n_steps, double dt, int rhs_only,
                             int64_t obs_every = 0, int64_t obs_first = 0) {
    RingArgs a;
    memset(&a, 0, sizeof(a));
    a.obs_every = obs_every; a.obs_first = obs_first;
    a.barrier_flags = ring_barrier_flags();
    a.obs_cs = (double*)((char*)h->b.scratch + ring_work_bytes(h->n, h->esize));
    a.obs_ref = h->b.obs_ref;
    a.y_in = y_in; a.y_out = y_out; a.elem_param = h->b.elem_param;
    a.n = h->tv.ring_n; a.ld = h->ld; a.npad = round_up(h->n, 64);
    a.P = h->tv.P; a.include_self = h->tv.include_self; a.chunk = p.chunk; a.G = p.G;
    a.chunk_shift = 0;
    while ((1 << a.chunk_shift) < p.chunk) ++a.chunk_shift;
    a.n_steps = n_steps; a.dt = dt; a.rhs_only = rhs_only;
    char* s = (char*)h->b.scratch;
    const size_t sbytes = 2 * (size_t)a.npad * h->esize;
    a.S[0] = s; a.S[1] = s + sbytes;
    a.tot[0] = (double*)(s + 2 * sbytes);
    a.tot[1] = a.tot[0] + 2 * RING_GMAX;
    a.bar = (unsigned*)(a.tot[1] + 2 * RING_GMAX);
    const bool f32 = h->desc.dtype == NET_F32;
    if (h->desc.model == NET_MODEL_KS)
        return f32 ? ring_launch_e<float, NET_MODEL_KS>(h, a, p) : ring_launch_e<double, NET_MODEL_KS>(h, a, p);
    if (h->desc.model == NET_MODEL_KSI)
        return f32 ? ring_launch_e<float, NET_MODEL_KSI>(h, a, p) : ring_launch_e<double, NET_MODEL_KSI>(h, a, p);
    return f32 ? ring_launch_e<float, NET_MODEL_FHN>(h, a, p) : ring_launch_e<double, NET_MODEL_FHN>(h, a, p);
}

// ------------------------------------------------------------------ latency probes
// The ring configs are bound by the dependent chain of one stage, not by bytes or flops
// (SURVEY.md 8(d)): block scan -> grid barrier -> one L2 round trip -> scan of the totals ->
// local field (KS: one fp64 sincos).  These kernels time exactly those primitives, as the ring
// kernel uses them, so that bench.py can quote the stage time against a measured floor.
__global__ void __launch_bounds__(RING_THREADS) probe_barrier_kernel(unsigned* bar, int iters, int G, int flags_form) {
    for (int it = 0; it < iters; ++it) grid_barrier(bar, (unsigned)(it + 1), G, flags_form);
}
__global__ void probe_ring_init_kernel(unsigned* ring, unsigned n, unsigned stride) {
    for (unsigned i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) ring[i] = (i + stride) % n;
}
__global__ void probe_l2_kernel(const unsigned* ring, int iters, unsigned* sink) {
    unsigned j = 0;
    for (int it = 0; it < iters; ++it) j = __ldcg(ring + j);      // dependent loads served by L2
    *sink = j;
}
__global__ void __launch_bounds__(RING_THREADS) probe_scan_kernel(int iters, double* sink) {
    __shared__ double wsum[2][RING_THREADS / 32];
    double a = 1.0 + threadIdx.x, b = 2.0, ta = 0, tb = 0;
    for (int it = 0; it < iters; ++it) {
        block_scan2<double, true>(a, b, ta, tb, wsum);
        a = a * 1e-9 + ta * 1e-9; b = b * 1e-9 + tb * 1e-9;         // the next scan depends on this one
    }
    if (threadIdx.x == 0) *sink = a + b;
}
__global__ void probe_sincos_kernel(int iters, double x, double* sink) {
    for (int it = 0; it < iters; ++it) {
        double s, c;
        sincos(x, &s, &c);
        x += 1e-3 * s + 1e-3 * c;                                   // dependent chain
    }
    *sink = x;
}

// out[0] grid barrier over the CTAs of this net's ring plan (1 CTA: 0), out[1] dependent L2 load,
// out[2] block scan of two doubles (256 threads), out[3] dependent fp64 sincos; microseconds each.
int32_t ring_probe_latency(net* h, double* out) {
    RingPlan p;
    // only nets served by the persistent ring kernel: their scratch is rewritten by every launch
    // (the scratch of a lattice net holds its exchange fields)
    if (!(h->fast_kind == FAST_RING_KS || h->fast_kind == FAST_RING_FHN) ||
        !ring_plan(h->tv.ring_n, h->esize, &p, h->desc.batch > 1 ? 1 : 148))
        return set_err(h, NET_ERR_UNSUPPORTED, "latency probes: ring nets on the FAST path only");
    const int G = p.G;
    char* s = (char*)h->b.scratch;
    const unsigned N = 1u << 20;                                     // 4 MB ring of indices, L2 resident
    if (h->b.scratch_bytes < (size_t)N * 4 + 4096) return set_err(h, NET_ERR_SIZE, "scratch too small for the probes");
    unsigned* ring = (unsigned*)s;
    unsigned* bar = (unsigned*)(s + (size_t)N * 4);
    double* sink = (double*)(s + (size_t)N * 4 + 2048);      // past the RING_GMAX barrier words
    cudaStream_t st = h->stream;
    cudaEvent_t e0, e1;
    OSC_CUDA(h, cudaEventCreate(&e0));
    OSC_CUDA(h, cudaEventCreate(&e1));
    const int iters = 2000;
    auto timed = [&](auto&& launch, double* us) -> int32_t {
        float ms = 0.f;
        for (int rep = 0; rep < 2; ++rep) {                          // rep 0 warms up
            cudaEventRecord(e0, st);
            int32_t rc = launch();
            if (rc) return rc;
            cudaEventRecord(e1, st);
            OSC_CUDA(h, cudaEventSynchronize(e1));
            OSC_CUDA(h, cudaEventElapsedTime(&ms, e0, e1));
        }
        *us = (double)ms * 1e3 / iters;
        return NET_OK;
    };
    int32_t rc = NET_OK;
    out[0] = 0.0;
    if (G > 1) {
        rc = timed([&]() -> int32_t {
            OSC_CUDA(h, cudaMemsetAsync(bar, 0, sizeof(unsigned) * RING_GMAX, st));
            int it = iters, g = G, ff = ring_barrier_flags();
            void* params[] = {&bar, &it, &g, &ff};
            OSC_CUDA(h, cudaLaunchCooperativeKernel((const void*)probe_barrier_kernel, dim3(G), dim3(RING_THREADS), params, 0, st));
            return NET_OK;
        }, &out[0]);
    }
    if (rc == NET_OK) {
        probe_ring_init_kernel<<<296, 256, 0, st>>>(ring, N, 16411u);
        rc = timed([&]() -> int32_t { probe_l2_kernel<<<1, 1, 0, st>>>(ring, iters, (unsigned*)sink); OSC_CUDA(h, cudaGetLastError()); return NET_OK; }, &out[1]);
    }
    if (rc == NET_OK)
        rc = timed([&]() -> int32_t { probe_scan_kernel<<<1, RING_THREADS, 0, st>>>(iters, sink); OSC_CUDA(h, cudaGetLastError()); return NET_OK; }, &out[2]);
    if (rc == NET_OK)
        rc = timed([&]() -> int32_t { probe_sincos_kernel<<<1, 1, 0, st>>>(iters, 0.3, sink); OSC_CUDA(h, cudaGetLastError()); return NET_OK; }, &out[3]);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    h->launches += 9;
    return rc;
}

// sum R, sum R^2 and the count of the samples a launch took, added to the statistics accumulators
// (observables.cu: acc[0], acc[1], acc[2]); R = |sum over the rings of (C, S)| / n_total
__global__ void __launch_bounds__(256) ring_obs_accumulate_kernel(const double* __restrict__ cs, int64_t samples, int rings, double inv_n, double* acc) {
    __shared__ double red[2][256];
    double s1 = 0.0, s2 = 0.0;
    for (int64_t k = threadIdx.x; k < samples; k += 256) {
        double C = 0.0, S = 0.0;
        for (int r = 0; r < rings; ++r) { C += cs[(k * rings + r) * 2]; S += cs[(k * rings + r) * 2 + 1]; }
        const double R = sqrt(C * C + S * S) * inv_n;
        s1 += R; s2 += R * R;
    }
    red[0][threadIdx.x] = s1; red[1][threadIdx.x] = s2;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) { red[0][threadIdx.x] += red[0][threadIdx.x + o]; red[1][threadIdx.x] += red[1][threadIdx.x + o]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) { acc[0] += red[0][0]; acc[1] += red[1][0]; acc[2] += (double)samples; }
}

// net_integrate_observed of a phase model on the persistent ring kernel: ONE launch for all steps;
// the samples at steps s_a, s_a + obs_every, ... < n_steps are taken inside it.  *handled = false:
// this net / run does not qualify (the caller samples between launches as before).
int32_t ring_run_observed(net* h, int64_t n_steps, double dt, int64_t obs_every, int64_t s_a, bool* handled) {
    *handled = false;
    RingPlan p;
    if (!(h->method == NET_METHOD_FAST && h->fast_kind == FAST_RING_KS) || n_steps > (1 << 20)) return NET_OK;
    if (!ring_plan(h->tv.ring_n, h->esize, &p, h->desc.batch > 1 ? 1 : 148)) return NET_OK;
    const int64_t samples = (n_steps - s_a) / obs_every;          // steps s_a ... n_steps - obs_every
    const int rings = p.single ? h->desc.batch : 1;
    if ((size_t)samples * rings * 16 > RING_OBS_BYTES || getenv("OSCNET_NO_FAST_OBS")) return NET_OK;
    int32_t rc = ring_run_plan(h, p, h->b.y, h->b.y, n_steps, dt, 0, obs_every, s_a);
    if (rc) return rc;
    if (samples > 0) {
        const double* cs = (const double*)((char*)h->b.scratch + ring_work_bytes(h->n, h->esize));
        ring_obs_accumulate_kernel<<<1, 256, 0, h->stream>>>(cs, samples, rings, 1.0 / (double)h->n, h->b.obs_acc);
        h->launches += 1;
        OSC_CUDA(h, cudaGetLastError());
    }
    *handled = true;
    return NET_OK;
}

int32_t ring_run(net* h, const void* y_in, void* y_out, int64_t n_steps, double dt, int rhs_only) {
    RingPlan p;
    // (two CTAs per SM -- gmax = 296, half the elements per thread -- measured slower on config 2:
    // 4.8e9 against 5.0e9 osc-steps/s; the 256-way barrier costs more than the shorter chain saves)
    if (!ring_plan(h->tv.ring_n, h->esize, &p, h->desc.batch > 1 ? 1 : 148)) return set_err(h, NET_ERR_UNSUPPORTED, "ring too large for the persistent kernel");
    return ring_run_plan(h, p, y_in, y_out, n_steps, dt, rhs_only);
}

}  // namespace oscnet
