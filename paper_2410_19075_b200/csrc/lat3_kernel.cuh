// FAST method for 3D periodic lattices, third generation (configs 3 and 5): warp-decoupled
// z-marching ball sums fed entirely by TMA.
//
// Mathematics as before (x-run decomposition of the ball of PAPER.md:313, register accumulators
// for the 2P+1 open output planes; exact in real arithmetic).  This file holds the pair form --
// both fields of the ball sum as one packed pair per thread -- that FitzHugh-Nagumo lattices run;
// Kuramoto-Sakaguchi lattices run the field-split form (lat3s_kernel.cuh), which shares the
// operand-tile table, the parameter block and the producer protocol defined here.  What
// changed is what the second generation was bound by on B200 (profiles/r01_baseline_ncu.md:
// 17 % occupancy, one CTA-wide barrier per plane, operand loads exposed once per plane, 93
// instructions per element):
//   * a dedicated PRODUCER warp issues, D planes ahead, one TMA tensor load for the staged
//     stencil plane (tile + halo, from the ghost-padded pair array) AND one per pointwise operand
//     tile of the output plane that iteration finishes (y, Y2, Z, omega ...).  Everything a
//     consumer touches arrives in shared memory on one `full` mbarrier per iteration: there is no
//     global load in the compute warps, and the bytes in flight are set by D, not by occupancy;
//   * CONSUMER warps never meet at a CTA barrier: each warp waits on `full[i]`, computes, stores
//     its outputs straight from registers and arrives on `done[i]`, which is all the producer
//     needs to recycle the slots.  Warps of one CTA drift up to D planes apart and several small
//     CTAs share an SM, so stalls of one warp are covered by the others;
//   * the stage is a template parameter and the model constants arrive pre-converted to the
//     arithmetic type of the net (no F2F / branches on the stage in the inner loop).
// RK4 in the "Z form" (lattice_v2.cuh / DESIGN.md section 4), 13 records per element and step.
#pragma once
#include "lat_common.cuh"

namespace oscnet {

// L3_LOC: not a stage of the integrator -- the local order parameter of reading R9 through the same
// ball-sum machinery: the stencil source is the unit phasor field
// (cos theta, sin theta), the finisher writes |ball sum incl. the centre| / n_ball.
enum { L3_S0 = 0, L3_S1 = 1, L3_S2 = 2, L3_S3 = 3, L3_RHS = 4, L3_LOC = 5 };

// operand tiles per finished plane.  FHN (pair tiles): stage 0: - | 1: y | 2: y, Y2 | 3: Z | RHS: -
// KS (scalar tiles, omega last): stage 0, 1: y, omega | 2: y, Y2, Y3, omega | 3: Z, omega | RHS: omega
template <int MODEL, int STAGE> struct L3Ops {
    static constexpr int N = STAGE == L3_LOC ? 0 : MODEL == NET_MODEL_FHN
        ? (STAGE == L3_S1 || STAGE == L3_S3 ? 1 : STAGE == L3_S2 ? 2 : 0)
        : (STAGE == L3_S2 ? 4 : STAGE == L3_RHS ? 1 : 2);
};

template <class T> struct L3Params {   // model constants in the arithmetic type of the net
    T h;                       // stage weight: dt/2, dt/2, dt, dt/6
    T nb;                      // FHN: lattice points of the ball including the centre
    T cuu, cuv, cvu, cvv;      // FHN: (sigma/Omega) b, the u row also divided by eps
    T ie, ie3, a;              // FHN: 1/eps, -1/(3 eps), a
    T kd, ca, sa;              // KS: K/Omega, cos alpha, sin alpha
    T inv_nb;                  // L3_LOC: 1 / (lattice points of the ball including the centre)
    int include_self;
};

__device__ __forceinline__ float2 pfma(float2 a, float2 b, float2 c) {
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;"
        : "=l"(r)
        : "l"(*reinterpret_cast<unsigned long long*>(&a)), "l"(*reinterpret_cast<unsigned long long*>(&b)),
          "l"(*reinterpret_cast<unsigned long long*>(&c)));
    return *reinterpret_cast<float2*>(&r);
}
__device__ __forceinline__ double2 pfma(double2 a, double2 b, double2 c) {
    return make_double2(fma(a.x, b.x, c.x), fma(a.y, b.y, c.y));
}

// Work distribution.  The first tiles * nchunks CTAs each take one chunk of Lz planes of one tile
// column, chunk-major, so that all of them march through the same planes at the same time: the halo
// rows and columns a tile shares with its neighbours are then fetched from HBM once and served from L2
// to the others (measured on cfg 3a: 296 equal spans cut tile-major, every SM busy, run 28 % SLOWER
// than 250 aligned half columns that leave 46 SMs with one CTA instead of two).  Where the chunks do not
// fill the grid's last wave, they are shortened (nchunks * Lz < nz) and the planes left at the top of
// every column, linearised tile-major, are cut into equal spans for the remaining CTAs of the wave; a
// span that crosses into the next column is run as segments, each with its own 2P lead-in planes, the
// pipeline state carrying over.  nchunks = 0: the whole space as equal spans.
struct L3Span { long long begin, end; int r, zbase; };   // positions u: tile u / r, plane zbase + u % r
struct L3Seg { int x0, y0, z0, len; };
__device__ __forceinline__ L3Span l3_span(const L3Geom& g, int nz) {
    const int tiles = g.tiles_x * g.tiles_y;
    const int m = tiles * g.nchunks;
    const int bid = (int)blockIdx.x;
    if (bid < m) {
        const int tile = bid % tiles, k = bid / tiles;
        const int zb = k * g.Lz;
        const int len = min(g.Lz, nz - zb);
        const long long begin = (long long)tile * nz + zb;
        return L3Span{begin, begin + len, nz, 0};
    }
    const int zbase = g.nchunks * g.Lz, r = nz - zbase;
    const long long U = (long long)tiles * r;
    const long long c = bid - m, gt = (long long)gridDim.x - m;
    return L3Span{U * c / gt, U * (c + 1) / gt, r, zbase};
}
__device__ __forceinline__ L3Seg l3_segment(const L3Geom& g, const L3Span& sp, long long u) {
    const int tile = (int)(u / sp.r);
    const int dz = (int)(u - (long long)tile * sp.r);
    const long long left = sp.end - u;
    const int len = left < (long long)(sp.r - dz) ? (int)left : sp.r - dz;
    return L3Seg{(tile % g.tiles_x) * g.TXt, (tile / g.tiles_x) * g.TYt, sp.zbase + dz, len};
}

// ROT = 0: the accumulators of the open output planes are addressed by a compile-time phase J modulo
// 2P + 1, which needs 2P + 1 copies of the plane body: for P = 4 those copies (130 KB of SASS) overflow
// the instruction cache once the decoupled warps drift apart (profiles/r01_lat3_ncu.md, cfg 3a:
// no_instruction).  ROT = 1: one body, the accumulators shifted down one slot after every plane (2P
// register moves per accumulator row and plane).  ROT = G > 1: G bodies with phases 0 .. G-1 indexing
// G - 1 slots past 2P + 1, one shift by G slots after every G planes (the moves of ROT = 1 divided by G).
template <int ROT, int NACC> __host__ __device__ constexpr int l3_slot(int j) { return ROT > 0 ? j : j % NACC; }
template <class T, int MODEL, int P, int STAGE, int X, int TY, int MAXT, int MINB, int ROT>
__global__ void __launch_bounds__(MAXT, MINB)
lat3_kernel(const __grid_constant__ CUtensorMap tm_st, const __grid_constant__ CUtensorMap tm_op0,
            const __grid_constant__ CUtensorMap tm_op1, const __grid_constant__ CUtensorMap tm_op2,
            const __grid_constant__ CUtensorMap tm_op3, L3Ptrs a, L3Params<T> mp, L3Geom g) {
    typedef typename PairOf<T>::type Pr;
    static_assert(MODEL == NET_MODEL_FHN, "pair form: FHN; KS lattices run lat3s_kernel");
    constexpr int HX = l2_hx<T>(P);           // x ghost width of the padded pair arrays
    constexpr int NCOL = X + 2 * HX;          // pairs a thread reads per staged row
    constexpr int OFF = HX - P;
    constexpr int NACC = 2 * P + 1;
    constexpr int NSLOT = NACC + (ROT > 1 ? ROT - 1 : 0);   // accumulator slots (ROT > 1: the group's phases index past NACC)
    constexpr int NT = L3Ops<MODEL, STAGE>::N;
    constexpr int U8 = (int)sizeof(Pr) / 8;   // 8-byte TMA elements per pair
    constexpr int EW = 2 * X;                 // scalars per thread-row of an operand / output tile

    extern __shared__ __align__(128) unsigned char l3_smem[];
    const int D = g.D, NB = D + 1, NS = P + 1 + D;
    uint64_t* full = reinterpret_cast<uint64_t*>(l3_smem);      // NB barriers
    uint64_t* done = full + NB;                                  // NB barriers
    unsigned char* st_ring = l3_smem + 256;
    unsigned char* op_ring = st_ring + (size_t)NS * g.st_stride;

    const int nx = g.nx, ny = g.ny, nz = g.nz;
    const int tid = threadIdx.x;
    const L3Span sp = l3_span(g, nz);         // this CTA's share of the (tile, z) space

    if (tid == 0) {
        for (int s = 0; s < NB; ++s) { mbar_init(full + s, 1); mbar_init(done + s, (unsigned)g.ncw); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // ------------------------------------------------------------------ producer warp
    if ((tid >> 5) == g.ncw) {
        if ((tid & 31) == 0) {
            asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_st) : "memory");
            if (NT >= 1) asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_op0) : "memory");
            if (NT >= 2) asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_op1) : "memory");
            int b = 0, ss = 0;
            unsigned round = 0;                     // iterations so far / NB
            for (long long s = sp.begin; s < sp.end;) {
                const L3Seg sg = l3_segment(g, sp, s);
                const int x0 = sg.x0, y0 = sg.y0, z0 = sg.z0, nplanes = sg.len + 2 * P;
                for (int j = 0; j < nplanes; ++j) {
                    // slot reuse: every consumer warp has finished the iteration NB before this one (phase round-1 of done[b])
                    if (round > 0) mbar_wait(done + b, (round & 1u) ^ 1u);
                    const bool ops = NT > 0 && j >= 2 * P;
                    mbar_expect_tx(full + b, g.st_bytes + (ops ? NT * g.op_bytes : 0u));
                    int zz = (z0 - P + j) % nz; if (zz < 0) zz += nz;
                    tma_load_3d(st_ring + (size_t)ss * g.st_stride, &tm_st, x0 * U8, y0, zz, full + b);
                    if (ops) {
                        const int zo = z0 - 2 * P + j;
                        unsigned char* ob = op_ring + (size_t)b * NT * g.op_stride;
                        // operands: centre boxes of the padded pair arrays
                        const int cx = (x0 + HX) * U8, cy = y0 + P;
                        if (NT >= 1) tma_load_3d(ob, &tm_op0, cx, cy, zo, full + b);
                        if (NT >= 2) tma_load_3d(ob + g.op_stride, &tm_op1, cx, cy, zo, full + b);
                        if (NT >= 3) tma_load_3d(ob + 2 * (size_t)g.op_stride, &tm_op2, cx, cy, zo, full + b);
                        if (NT >= 4) tma_load_3d(ob + 3 * (size_t)g.op_stride, &tm_op3, cx, cy, zo, full + b);
                    }
                    ss = ss + 1 == NS ? 0 : ss + 1;
                    if (++b == NB) { b = 0; ++round; }
                }
                s += sg.len;
            }
        }
        return;
    }

    // ------------------------------------------------------------------ consumer warps
    const int PW = g.PW;
    const int q = tid % g.QX, st = tid / g.QX;
    const int nxp = nx + 2 * HX, nyp = ny + 2 * P;
    const int64_t pxy = (int64_t)nxp * nyp;
    // per segment (set in the loop at the end of the kernel)
    int z0 = 0, x = 0, yrow0 = 0, gxs = 0;
    bool owner = false;

    Pr acc[NSLOT][TY][X];
#pragma unroll
    for (int k = 0; k < NSLOT; ++k)
#pragma unroll
        for (int r = 0; r < TY; ++r)
#pragma unroll
            for (int i = 0; i < X; ++i) acc[k][r][i] = Pr{T(0), T(0)};

    int slot = 0, cslot = NS - P, b = 0;      // ring slots of planes i and i - P; barrier index
    unsigned phase = 0;

    auto do_plane = [&](int i, auto Jc) {
        constexpr int J = decltype(Jc)::value;
        const int zo = z0 - 2 * P + i;            // output plane completed by this iteration
        mbar_wait(full + b, phase);
        if (owner) {
            const Pr* sb = reinterpret_cast<const Pr*>(st_ring + (size_t)slot * g.st_stride) + (st * TY) * PW + q * X;
            Pr A[P > 1 ? P - 1 : 1][TY][X];
            bool Aset[P > 1 ? P - 1 : 1][TY];
#pragma unroll
            for (int k = 0; k < (P > 1 ? P - 1 : 1); ++k)
#pragma unroll
                for (int r = 0; r < TY; ++r) Aset[k][r] = false;
#pragma unroll
            for (int rr = 0; rr < TY + 2 * P; ++rr) {           // staged row rr <-> y = yrow0 - P + rr
                const int dist = rr < P ? P - rr : (rr >= TY + P ? rr - (TY + P - 1) : 0);
                const int wmax = l2_run_w(P, 0, dist);
                Pr v[NCOL];
                const Pr* row = sb + rr * PW;
                if constexpr (sizeof(T) == 4) {
#pragma unroll
                    for (int c = 0; c < NCOL / 2; ++c) {
                        float4 w4 = *reinterpret_cast<const float4*>(row + 2 * c);
                        v[2 * c] = make_float2(w4.x, w4.y);
                        v[2 * c + 1] = make_float2(w4.z, w4.w);
                    }
                } else {
#pragma unroll
                    for (int c = 0; c < NCOL; ++c) v[c] = row[c];
                }
                Pr R[P + 1][X];
#pragma unroll
                for (int e = 0; e < X; ++e) {
                    R[0][e] = v[OFF + P + e];
#pragma unroll
                    for (int w = 1; w <= P; ++w)
                        if (w <= wmax) R[w][e] = padd(R[w - 1][e], padd(v[OFF + P + e - w], v[OFF + P + e + w]));
                }
#pragma unroll
                for (int r = 0; r < TY; ++r) {
                    const int ady = rr - P - r < 0 ? -(rr - P - r) : rr - P - r;
                    if (ady > P) continue;
                    {   // |dz| = 0: straight into the accumulator of output plane i
                        const int w = l2_run_w(P, 0, ady);
#pragma unroll
                        for (int e = 0; e < X; ++e) acc[l3_slot<ROT, NACC>(J + P)][r][e] = padd(acc[l3_slot<ROT, NACC>(J + P)][r][e], R[w][e]);
                    }
#pragma unroll
                    for (int k = 1; k < P; ++k) {    // 0 < |dz| < P: in-plane partial sums
                        const int w = l2_run_w(P, k, ady);
                        if (w >= 0) {
#pragma unroll
                            for (int e = 0; e < X; ++e)
                                A[k - 1][r][e] = Aset[k - 1][r] ? padd(A[k - 1][r][e], R[w][e]) : R[w][e];
                            Aset[k - 1][r] = true;
                        }
                    }
                    if (ady == 0) {                  // |dz| = P: the centre alone (first / last contribution)
#pragma unroll
                        for (int e = 0; e < X; ++e) {
                            acc[l3_slot<ROT, NACC>(J + 2 * P)][r][e] = R[0][e];
                            acc[l3_slot<ROT, NACC>(J)][r][e] = padd(acc[l3_slot<ROT, NACC>(J)][r][e], R[0][e]);
                        }
                    }
                }
            }
#pragma unroll
            for (int k = 1; k < P; ++k)
#pragma unroll
                for (int r = 0; r < TY; ++r)
#pragma unroll
                    for (int e = 0; e < X; ++e) {
                        acc[l3_slot<ROT, NACC>(J + P - k)][r][e] = padd(acc[l3_slot<ROT, NACC>(J + P - k)][r][e], A[k - 1][r][e]);
                        acc[l3_slot<ROT, NACC>(J + P + k)][r][e] = padd(acc[l3_slot<ROT, NACC>(J + P + k)][r][e], A[k - 1][r][e]);
                    }
        }
        // ---- finish output plane zo (accumulator J)
        if (owner && zo >= z0) {
            const Pr* cb = reinterpret_cast<const Pr*>(st_ring + (size_t)cslot * g.st_stride) + (st * TY + P) * PW + q * X + HX;
            const T* ob = reinterpret_cast<const T*>(op_ring + (size_t)b * NT * g.op_stride) + (st * TY) * (g.TXt * 2) + q * EW;
            const int ostride = g.op_stride / (int)sizeof(T);    // scalars between operand tiles
            const int orow = g.TXt * 2;                          // scalars per tile row
#pragma unroll
            for (int r = 0; r < TY; ++r) {
                const int yy = yrow0 + r;
                if (yy >= ny) continue;
                if constexpr (STAGE == L3_LOC) {     // |sum of the unit phasors over the ball| / n_ball, plain scalar array
                    T lo[X];
#pragma unroll
                    for (int e = 0; e < X; ++e) {
                        const Pr W = acc[l3_slot<ROT, NACC>(J)][r][e];
                        lo[e] = sqrt(W.x * W.x + W.y * W.y) * mp.inv_nb;
                    }
                    stg_vec<X>((T*)a.out + ((int64_t)zo * ny + yy) * nx + x, lo);
                    continue;
                }
                const int64_t ip = (int64_t)zo * pxy + (int64_t)(yy + P) * nxp + (x + HX);     // padded pair arrays
                const int gys = yy < P ? ny : (yy >= ny - P ? -ny : 0);
                auto store_pairs = [&](T* base, const T (&vals)[2 * X]) {    // with the periodic images
                    stg_vec<2 * X>(base + 2 * ip, vals);
                    if (gxs != 0) stg_vec<2 * X>(base + 2 * (ip + gxs), vals);
                    if (gys != 0) {
                        stg_vec<2 * X>(base + 2 * (ip + (int64_t)gys * nxp), vals);
                        if (gxs != 0) stg_vec<2 * X>(base + 2 * (ip + (int64_t)gys * nxp + gxs), vals);
                    }
                };
                // operand tiles of this thread-row: shared memory, 16-byte vectors where X allows
                T o0[EW], o1[EW];
                if (NT >= 1) ldg_vec<EW>(ob + r * orow, o0);
                if (NT >= 2) ldg_vec<EW>(ob + ostride + r * orow, o1);
                T ov[EW];
                [[maybe_unused]] T zv[EW];
                // centre pairs of the row: one 16-byte load for the two f32 pairs of a thread (two 8-byte
                // loads at a 16-byte lane stride take twice the wavefronts)
                Pr cpair[X];
                if constexpr (sizeof(T) == 4 && X == 2) {
                    const float4 c4 = *reinterpret_cast<const float4*>(cb + r * PW);
                    cpair[0] = Pr{c4.x, c4.y};
                    cpair[1] = Pr{c4.z, c4.w};
                } else {
#pragma unroll
                    for (int e = 0; e < X; ++e) cpair[e] = cb[r * PW + e];
                }
#pragma unroll
                for (int e = 0; e < X; ++e) {
                    const Pr c = cpair[e];
                    const Pr W = acc[l3_slot<ROT, NACC>(J)][r][e];
                    // sum_j (u_j - u_i) over the ball = W - n_ball c whether or not the centre counts
                    const Pr Cc = pfma(c, Pr{-mp.nb, -mp.nb}, W);
                    const T u = c.x, v = c.y;
                    const T rr_ = fma(u * u, mp.ie3, mp.ie);      // (1 - u^2/3)/eps
                    T gu = fma(mp.cuu, Cc.x, mp.cuv * Cc.y);
                    gu = fma(-mp.ie, v, gu);
                    const T ku = fma(u, rr_, gu);
                    const T kv = fma(mp.cvu, Cc.x, fma(mp.cvv, Cc.y, u + mp.a));
                    T ou, ovv;
                    if constexpr (STAGE == L3_RHS) { ou = ku; ovv = kv; }
                    else if constexpr (STAGE == L3_S0) { ou = fma(mp.h, ku, u); ovv = fma(mp.h, kv, v); }
                    else { ou = fma(mp.h, ku, o0[2 * e]); ovv = fma(mp.h, kv, o0[2 * e + 1]); }
                    if constexpr (STAGE == L3_S2) {
                        zv[2 * e] = (o1[2 * e] + T(2) * u + ou - o0[2 * e]) * T(1.0 / 3.0);
                        zv[2 * e + 1] = (o1[2 * e + 1] + T(2) * v + ovv - o0[2 * e + 1]) * T(1.0 / 3.0);
                    }
                    ov[2 * e] = ou; ov[2 * e + 1] = ovv;
                }
                store_pairs((T*)a.out, ov);
                if constexpr (STAGE == L3_S2) stg_vec<EW>((T*)a.out2 + 2 * ip, zv);   // Z is never a stencil source
            }
        }
        // this warp is done with barrier b: stencil plane i - P and operand slot b may be refilled
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(done + b);
        slot = slot + 1 == NS ? 0 : slot + 1;
        cslot = cslot + 1 == NS ? 0 : cslot + 1;
        if (++b == NB) { b = 0; phase ^= 1u; }
    };

    // The accumulator of an output plane is ASSIGNED by the first plane that reaches it (|dz| = P), so
    // what the previous segment left in the registers never enters an output of this one.
#pragma unroll 1
    for (long long s = sp.begin; s < sp.end;) {
        const L3Seg sg = l3_segment(g, sp, s);
        const int nplanes = sg.len + 2 * P;
        z0 = sg.z0;
        x = sg.x0 + q * X;
        owner = st < g.SY && x < nx;
        yrow0 = sg.y0 + st * TY;
        gxs = x < HX ? nx : (x >= nx - HX ? -nx : 0);   // periodic image this thread also writes
        constexpr int GSZ = ROT > 0 ? ROT : NACC;       // plane bodies in the loop
#pragma unroll 1
        for (int base = 0; base < nplanes; base += GSZ) {
            l2_static_for<0, GSZ>([&](auto Jc) {
                if (base + decltype(Jc)::value < nplanes) do_plane(base + decltype(Jc)::value, Jc);
            });
            if constexpr (ROT > 0) {
#pragma unroll
                for (int k = 0; k + 1 < NACC; ++k)
#pragma unroll
                    for (int r = 0; r < TY; ++r)
#pragma unroll
                        for (int e = 0; e < X; ++e) acc[k][r][e] = acc[k + ROT][r][e];
            }
        }
        s += sg.len;
    }
}

}  // namespace oscnet
