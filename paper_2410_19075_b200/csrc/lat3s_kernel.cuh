// Field-split variant of the third-generation 3D lattice kernel for Kuramoto-Sakaguchi lattices
// (configs 3a and 3b).
//
// Same mathematics and the same producer / mbarrier pipeline as lat3_kernel.cuh (x-run
// decomposition of the ball of PAPER.md:313, z-marching register accumulators, factorised sine
// of Alg. 1).  What the ncu capture of lat3_kernel on cfg 3b showed
// (profiles/r01_final_ncu.md): with both fields of the ball sum, (cos phi, sin phi), carried as a
// pair by every thread, the fp64 accumulators of the 2P + 1 open planes leave room for only
// X x TY = 2 x 1 outputs per thread, so every thread loads and run-sums 2P + 1 staged rows for
// ONE output row -- 45 LDS.128 and 164 DADD per output, two thirds of the kernel time in
// shared-memory wavefronts.
// Here the two lanes  l  and  l ^ 16  of a warp share one 2 x 2 block of outputs and each carries
// ONE field (lanes 0-15 the cos plane, lanes 16-31 the sin plane): the same 72 accumulator
// registers now cover 2 x 2 outputs of one field, the staged rows are shared by two output rows
// (25 LDS.128 and 114 DADD per output), and the two partial results meet once per finished plane
// through a warp shuffle; lane f then finishes output row f of the block.
// fp32 (cfg 3a): the same split halves the registers a thread needs for its accumulators (the two
// x-adjacent columns of one field form the packed f32x2 operand instead of the (cos, sin) pair), so
// twice as many warps are resident -- that kernel was bound by dependent-issue latency at 12 warps
// per SM, not by a pipe (add.f32x2 moves as many lanes per clock as add.f32: measured 64 vs 128
// thread-instructions per clock and SM).
#pragma once
#include "lat3_kernel.cuh"

namespace oscnet {

template <class T, int P, int STAGE, int TY, int MAXT, int MINB, int ROT>
__global__ void __launch_bounds__(MAXT, MINB)
lat3s_kernel(const __grid_constant__ CUtensorMap tm_st, const __grid_constant__ CUtensorMap tm_op0,
             const __grid_constant__ CUtensorMap tm_op1, const __grid_constant__ CUtensorMap tm_op2,
             const __grid_constant__ CUtensorMap tm_op3, L3Ptrs a, L3Params<T> mp, L3Geom g) {
    typedef typename PairOf<T>::type Pr;      // the two x-adjacent columns of a thread, one field
    static_assert(P % 2 == 0, "column pairs of even shifts are aligned register pairs");
    constexpr int MODEL = NET_MODEL_KS;
    constexpr int X = 2;
    static_assert(TY % 2 == 0, "the two lanes of a block split its rows");
    constexpr int HX = l2_hx<T>(P);           // x ghost width of the padded planes
    constexpr int OFF = HX - P;
    constexpr int NCOL = X + 2 * P;           // scalars a thread reads per staged row
    constexpr int NACC = 2 * P + 1;
    constexpr int NSLOT = NACC + (ROT > 1 ? ROT - 1 : 0);   // accumulator slots (ROT > 1: the group's phases index past NACC)
    constexpr int NT = L3Ops<MODEL, STAGE>::N;
    static_assert(OFF % 2 == 0 && NCOL % 2 == 0, "aligned column pairs");

    extern __shared__ __align__(128) unsigned char l3_smem[];
    const int D = g.D, NB = D + 1, NS = P + 1 + D;
    uint64_t* full = reinterpret_cast<uint64_t*>(l3_smem);      // NB barriers
    uint64_t* done = full + NB;                                  // NB barriers
    unsigned char* st_ring = l3_smem + 256;
    unsigned char* op_ring = st_ring + (size_t)NS * g.st_stride;

    const int nx = g.nx, ny = g.ny, nz = g.nz;
    const int tid = threadIdx.x;
    const L3Span sp = l3_span(g, nz);         // this CTA's share of the (tile, z) space (lat3_kernel.cuh)

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
            unsigned round = 0;
            for (long long s = sp.begin; s < sp.end;) {
                const L3Seg sg = l3_segment(g, sp, s);
                const int x0 = sg.x0, y0 = sg.y0, z0 = sg.z0, nplanes = sg.len + 2 * P;
                for (int j = 0; j < nplanes; ++j) {
                    if (round > 0) mbar_wait(done + b, (round & 1u) ^ 1u);
                    const bool ops = NT > 0 && j >= 2 * P;
                    mbar_expect_tx(full + b, g.st_bytes + (ops ? NT * g.op_bytes : 0u));
                    int zz = (z0 - P + j) % nz; if (zz < 0) zz += nz;
                    tma_load_4d(st_ring + (size_t)ss * g.st_stride, &tm_st, x0, y0, zz, 0, full + b);
                    if (ops) {
                        const int zo = z0 - 2 * P + j;
                        unsigned char* ob = op_ring + (size_t)b * NT * g.op_stride;
                        if (NT >= 1) tma_load_3d(ob, &tm_op0, x0, y0, zo, full + b);
                        if (NT >= 2) tma_load_3d(ob + g.op_stride, &tm_op1, x0, y0, zo, full + b);
                        if (NT >= 3) tma_load_3d(ob + 2 * (size_t)g.op_stride, &tm_op2, x0, y0, zo, full + b);
                        if (NT >= 4) tma_load_3d(ob + 3 * (size_t)g.op_stride, &tm_op3, x0, y0, zo, full + b);
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
    // lanes l and l ^ 16 own the same 2 x 2 block of outputs ("unit"), one field each
    const int PW = g.PW;
    const int lane = tid & 31;
    const int f = lane >> 4;                              // 0: cos plane, 1: sin plane
    const int unit = (tid >> 5) * 16 + (lane & 15);
    const int q = unit % g.QX, st = unit / g.QX;
    const int nxp = nx + 2 * HX, nyp = ny + 2 * P;
    const int64_t nxy = (int64_t)nx * ny;
    const int64_t pxy = (int64_t)nxp * nyp;
    const int splane = PW * g.PH;                             // scalars between the staged cos and sin boxes
    // per segment (set in the loop at the end of the kernel)
    int z0 = 0, x = 0, yrow0 = 0, gxs = 0;
    bool owner = false;

    Pr acc[NSLOT][TY];
#pragma unroll
    for (int k = 0; k < NSLOT; ++k)
#pragma unroll
        for (int r = 0; r < TY; ++r) acc[k][r] = Pr{T(0), T(0)};

    int slot = 0, cslot = NS - P, b = 0;      // ring slots of planes i and i - P; barrier index
    unsigned phase = 0;

    auto do_plane = [&](int i, auto Jc) {
        constexpr int J = decltype(Jc)::value;
        const int zo = z0 - 2 * P + i;            // output plane completed by this iteration
        mbar_wait(full + b, phase);
        if (owner) {
            const T* sb = reinterpret_cast<const T*>(st_ring + (size_t)slot * g.st_stride) + f * splane + (st * TY) * PW + q * X + OFF;
            Pr A[P > 1 ? P - 1 : 1][TY];
            bool Aset[P > 1 ? P - 1 : 1][TY];
#pragma unroll
            for (int k = 0; k < (P > 1 ? P - 1 : 1); ++k)
#pragma unroll
                for (int r = 0; r < TY; ++r) Aset[k][r] = false;
#pragma unroll
            for (int rr = 0; rr < TY + 2 * P; ++rr) {           // staged row rr <-> y = yrow0 - P + rr
                const int dist = rr < P ? P - rr : (rr >= TY + P ? rr - (TY + P - 1) : 0);
                const int wmax = l2_run_w(P, 0, dist);
                Pr v[NCOL / 2];                                  // v[c] = columns (2c, 2c + 1) of the row piece
                const Pr* row = reinterpret_cast<const Pr*>(sb + rr * PW);
#pragma unroll
                for (int c = 0; c < NCOL / 2; ++c) {
                    if (2 * c + 1 < P - wmax || 2 * c > P + X - 1 + wmax) continue;     // columns no run of this row reaches
                    v[c] = row[c];
                }
                auto col = [&](int j) -> T { return (j & 1) ? v[j / 2].y : v[j / 2].x; };
                Pr R[P + 1];
                R[0] = v[P / 2];
#pragma unroll
                for (int w = 1; w <= P; ++w)
                    if (w <= wmax) {
                        Pr side;
                        if (w % 2 == 0) side = padd(v[(P - w) / 2], v[(P + w) / 2]);
                        else side = Pr{col(P - w) + col(P + w), col(P + 1 - w) + col(P + 1 + w)};
                        R[w] = padd(R[w - 1], side);
                    }
#pragma unroll
                for (int r = 0; r < TY; ++r) {
                    const int ady = rr - P - r < 0 ? -(rr - P - r) : rr - P - r;
                    if (ady > P) continue;
                    {   // |dz| = 0: straight into the accumulator of output plane i
                        const int w = l2_run_w(P, 0, ady);
                        acc[l3_slot<ROT, NACC>(J + P)][r] = padd(acc[l3_slot<ROT, NACC>(J + P)][r], R[w]);
                    }
#pragma unroll
                    for (int k = 1; k < P; ++k) {    // 0 < |dz| < P: in-plane partial sums
                        const int w = l2_run_w(P, k, ady);
                        if (w >= 0) {
                            A[k - 1][r] = Aset[k - 1][r] ? padd(A[k - 1][r], R[w]) : R[w];
                            Aset[k - 1][r] = true;
                        }
                    }
                    if (ady == 0) {                  // |dz| = P: the centre alone (first / last contribution)
                        acc[l3_slot<ROT, NACC>(J + 2 * P)][r] = R[0];
                        acc[l3_slot<ROT, NACC>(J)][r] = padd(acc[l3_slot<ROT, NACC>(J)][r], R[0]);
                    }
                }
            }
#pragma unroll
            for (int k = 1; k < P; ++k)
#pragma unroll
                for (int r = 0; r < TY; ++r) {
                    acc[l3_slot<ROT, NACC>(J + P - k)][r] = padd(acc[l3_slot<ROT, NACC>(J + P - k)][r], A[k - 1][r]);
                    acc[l3_slot<ROT, NACC>(J + P + k)][r] = padd(acc[l3_slot<ROT, NACC>(J + P + k)][r], A[k - 1][r]);
                }
        }
        // ---- finish output plane zo (accumulator J): lane f takes the output rows 2m + f of the block
        if (zo >= z0) {                                   // uniform over the CTA
#pragma unroll
          for (int m = 0; m < TY / 2; ++m) {              // rows 2m, 2m + 1: lane f finishes row 2m + f
            const Pr send = f ? acc[l3_slot<ROT, NACC>(J)][2 * m] : acc[l3_slot<ROT, NACC>(J)][2 * m + 1];    // the row the partner finishes
            const T other[X] = {__shfl_xor_sync(0xffffffffu, send.x, 16), __shfl_xor_sync(0xffffffffu, send.y, 16)};
            const Pr ownp = f ? acc[l3_slot<ROT, NACC>(J)][2 * m + 1] : acc[l3_slot<ROT, NACC>(J)][2 * m];
            const T ownv[X] = {ownp.x, ownp.y};
            const int r = 2 * m + f;
            const int yy = yrow0 + r;
            if (owner && yy < ny) {
                const T* cc = reinterpret_cast<const T*>(st_ring + (size_t)cslot * g.st_stride) + (st * TY + P + r) * PW + q * X + HX;
                const T* ob = reinterpret_cast<const T*>(op_ring + (size_t)b * NT * g.op_stride) + (st * TY + r) * g.TXt + q * X;
                const int ostride = g.op_stride / (int)sizeof(T);    // scalars between operand tiles
                const int64_t il = (int64_t)zo * nxy + (int64_t)yy * nx + x;                    // plain scalar arrays
                const int64_t ip = (int64_t)zo * pxy + (int64_t)(yy + P) * nxp + (x + HX);     // padded planes
                [[maybe_unused]] const int gys = yy < P ? ny : (yy >= ny - P ? -ny : 0);
                T o0[X], o1[X], o2[X], o3[X];
                if (NT >= 1) ldg_vec<X>(ob, o0);
                if (NT >= 2) ldg_vec<X>(ob + ostride, o1);
                if (NT >= 3) ldg_vec<X>(ob + 2 * ostride, o2);
                if (NT >= 4) ldg_vec<X>(ob + 3 * ostride, o3);
                T cx[X], cy[X];
                ldg_vec<X>(cc, cx);
                ldg_vec<X>(cc + splane, cy);
                [[maybe_unused]] T ov[X], zv[X], cv[X], sv[X];
                if constexpr (STAGE == L3_LOC) {      // local order parameter: |ball sum incl. the centre| / n_ball
#pragma unroll
                    for (int e = 0; e < X; ++e) ov[e] = sqrt(ownv[e] * ownv[e] + other[e] * other[e]) * mp.inv_nb;
                    stg_vec<X>((T*)a.out + il, ov);
                    continue;
                }
#pragma unroll
                for (int e = 0; e < X; ++e) {
                    const T own = ownv[e];
                    T C = f ? other[e] : own, S = f ? own : other[e];
                    if (!mp.include_self) { C -= cx[e]; S -= cy[e]; }
                    const T cia = cx[e] * mp.ca - cy[e] * mp.sa;      // cos(phi_i + alpha)
                    const T sia = cy[e] * mp.ca + cx[e] * mp.sa;      // sin(phi_i + alpha)
                    const T om = NT == 4 ? o3[e] : NT == 2 ? o1[e] : o0[e];
                    const T k = om + mp.kd * (S * cia - C * sia);
                    T o;
                    if constexpr (STAGE == L3_RHS) o = k;
                    else o = o0[e] + mp.h * k;                   // y (stages 0-2) or Z (stage 3)
                    if constexpr (STAGE == L3_S2) zv[e] = (o1[e] + T(2) * o2[e] + o - o0[e]) * T(1.0 / 3.0);
                    ov[e] = o;
                    if constexpr (STAGE != L3_RHS) sincos_stage<T>(o, &sv[e], &cv[e]);
                }
                stg_vec<X>((T*)a.out + il, ov);
                if constexpr (STAGE == L3_S2) stg_vec<X>((T*)a.out2 + il, zv);
                if constexpr (STAGE != L3_RHS) {
                    T* Ec = (T*)a.Eout;
                    T* Es = Ec + g.plane;
                    auto store_planes = [&](int64_t at) { stg_vec<X>(Ec + at, cv); stg_vec<X>(Es + at, sv); };
                    store_planes(ip);
                    if (gxs != 0) store_planes(ip + gxs);
                    if (gys != 0) {
                        store_planes(ip + (int64_t)gys * nxp);
                        if (gxs != 0) store_planes(ip + (int64_t)gys * nxp + gxs);
                    }
                }
            }
          }
        }
        // this warp is done with barrier b: stencil plane i - P and operand slot b may be refilled
        __syncwarp();
        if (lane == 0) mbar_arrive(done + b);
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
                    for (int r = 0; r < TY; ++r) acc[k][r] = acc[k + ROT][r];
            }
        }
        s += sg.len;
    }
}

}  // namespace oscnet
