// FAST method for 3D periodic lattices, second generation (configs 3 and 5).
//
// Same mathematics as lattice_fast.cu (x-run decomposition of the ball of PAPER.md:313, z-marching
// CTA, register accumulators for the 2P+1 open output planes; exact in real arithmetic), rebuilt
// around what bounds it on B200:
//   * the two fields of the ball sum -- (u, v) for FHN, (cos phi, sin phi) for KS -- are stored
//     INTERLEAVED as pairs, in global memory and in shared memory, so every add of the ball sum is
//     one packed FADD2 (add.rn.f32x2) on an aligned register pair and every shared-memory access
//     is a 16-byte LDS;
//   * the pair fields live in GHOST-PADDED arrays (x padded by GX = halo rounded to 16 bytes, y by
//     GY = P on both sides; the producer of a field also writes the periodic images), so every
//     staged plane -- tile plus halo -- is ONE TMA tensor load (cp.async.bulk.tensor.3d,
//     UTMALDG) completing on an mbarrier, issued D planes ahead of the compute by one thread:
//     no register staging and no address arithmetic in the inner loop;
//   * KS: the producing stage writes E = (cos phi, sin phi) of its output next to phi, so the
//     sincos is paid exactly once per element per stage and halos are plain copies;
//   * RK4 in the "Z form" (13 state records per step, at most two pointwise operands per stage):
//       stage 0: Y2 = y + dt/2 f(y)        stage 1: Y3 = y + dt/2 f(Y2)
//       stage 2: Y4 = y + dt f(Y3),  Z = (Y2 + 2 Y3 + Y4 - y)/3   (Z overwrites Y2)
//       stage 3: y  = Z + dt/6 f(Y4)
//     which is y + dt/6 (k1 + 2 k2 + 2 k3 + k4) with k_s recovered from the stage states.
// Thread = X consecutive columns x TY rows; CTA = QX x SY threads; tile = (QX X) x (SY TY).
#pragma once
#include "lat_common.cuh"

namespace oscnet {

// ------------------------------------------------------------------ kernel
// NOPS = number of pointwise operand arrays of this stage:
//   FHN  stage 0: 0 (y is the centre of the staged plane) | 1: y | 2: y, Y2 | 3: Z | RHS: 0
//   KS   stage 0, 1: y | 2: y, Y2, Y3 | 3: Z | RHS: 0
template <class T, int MODEL, int P, int X, int TY, int NOPS, int MAXT, int MINB = 1>
__global__ void __launch_bounds__(MAXT, MINB) lattice3d_v2_kernel(const __grid_constant__ CUtensorMap tmap,
                                                                   Lat2Args a, ModelParams mp, Lat2 g) {
    typedef typename PairOf<T>::type Pr;
    constexpr int HX = l2_hx<T>(P);           // = GX, the x ghost width of the padded arrays
    constexpr int NCOL = X + 2 * HX;          // pairs loaded per staged row by one thread
    constexpr int OFF = HX - P;               // loaded index of column x - P
    constexpr int NACC = 2 * P + 1;
    constexpr int NVS = MODEL == NET_MODEL_KS ? 1 : 2;   // scalars per element of the state arrays
    constexpr int EW = X * NVS;               // scalars per thread-row of a state array
    constexpr int U8 = (int)sizeof(Pr) / 8;   // 8-byte TMA elements per pair

    extern __shared__ __align__(128) unsigned char l2_smem[];
    const int PW = g.PW, PH = g.PH, NS = g.NS, D = g.D;
    uint64_t* full = reinterpret_cast<uint64_t*>(l2_smem);                       // NS barriers
    const unsigned box_bytes = (unsigned)(PW * PH * sizeof(Pr));
    const unsigned plane_bytes = (box_bytes + 127u) / 128u * 128u;
    unsigned char* ring = l2_smem + 128;

    const int nx = g.nx, ny = g.ny, nz = g.nz;
    const int nxp = nx + 2 * HX, nyp = ny + 2 * P;
    const int64_t nxy = (int64_t)nx * ny;           // unpadded plane (KS scalar arrays)
    const int64_t pxy = (int64_t)nxp * nyp;         // padded plane (pair arrays)
    int bid = blockIdx.x;
    const int tix = bid % g.tiles_x; bid /= g.tiles_x;
    const int tiy = bid % g.tiles_y; bid /= g.tiles_y;
    const int x0 = tix * g.TXt, y0 = tiy * g.TYt;
    const int z0 = bid * g.Lz;
    const int z1 = min(nz, z0 + g.Lz);
    const int tid = threadIdx.x;
    const int q = tid % g.QX, st = tid / g.QX;
    const int x = x0 + q * X;
    const bool owner = st < g.SY && x < nx && q * X < g.TXt;
    const int yrow0 = y0 + st * TY;
    // periodic images this thread also writes: column shift (pairs) and row shift (rows), 0 = none
    const int gxs = x < HX ? nx : (x >= nx - HX ? -nx : 0);

    const T* op0 = (const T*)a.op0;     // op1 may alias out2 (Z overwrites Y2 element by element)
    const T* op1 = (const T*)a.op1;
    const T* op2 = (const T*)a.op2;
    const int stage = a.stage;
    const T dt = (T)a.dt;

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) mbar_init(full + s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmap) : "memory");
    }
    __syncthreads();

    // plane idx of this chunk (lattice plane z0 - P + idx, periodic) -> ring slot idx mod NS.
    // The box starts at padded coordinates (x0, y0) = lattice (x0 - GX, y0 - P).
    auto issue_plane = [&](int idx, int slot) {          // one thread
        int zz = (z0 - P + idx) % nz; if (zz < 0) zz += nz;
        mbar_expect_tx(full + slot, box_bytes);
        tma_load_3d(ring + (size_t)slot * plane_bytes, &tmap, x0 * U8, y0, zz, full + slot);
    };

    const int nplanes = (z1 - z0) + 2 * P;
    if (tid == 0)
        for (int idx = 0; idx <= D && idx < nplanes; ++idx) issue_plane(idx, idx);

    Pr acc[NACC][TY][X];
#pragma unroll
    for (int k = 0; k < NACC; ++k)
#pragma unroll
        for (int r = 0; r < TY; ++r)
#pragma unroll
            for (int i = 0; i < X; ++i) acc[k][r][i] = Pr{T(0), T(0)};

    const int deg = g.n_ball - (g.include_self ? 0 : 1);
    const T inv_deg = deg > 0 ? T(1) / T(deg) : T(0);

    // One plane.  J = idx mod NACC selects, at compile time, which accumulator is which open
    // output plane: accumulator (J + P + dz) mod NACC collects output plane p + dz.
    int slot = 0, cslot = NS - P, islot = (D + 1) % NS;   // ring slots of planes idx, idx - P, idx + D + 1
    unsigned phase = 0;
    auto do_plane = [&](int idx, auto Jc) {
        constexpr int J = decltype(Jc)::value;
        const int zo = z0 - 2 * P + idx;          // output plane completed by this iteration
        const bool finishing = owner && zo >= z0;
        // pointwise operands of the plane finished in this iteration: issued before the wait
        T o0[TY][EW], o1[TY][EW], o2[TY][EW], om[TY][X];
        if (finishing) {
#pragma unroll
            for (int r = 0; r < TY; ++r) {
                const int yy = yrow0 + r;
                if (yy < ny) {
                    // state arrays: FHN padded pairs, KS plain scalars
                    const int64_t i = MODEL == NET_MODEL_KS
                        ? (int64_t)zo * nxy + (int64_t)yy * nx + x
                        : ((int64_t)zo * pxy + (int64_t)(yy + P) * nxp + (x + HX)) * 2;
                    if (NOPS >= 1) ldg_vec<EW>(op0 + i, o0[r]);
                    if (NOPS >= 2) ldg_vec<EW>(op1 + i, o1[r]);
                    if (NOPS >= 3) ldg_vec<EW>(op2 + i, o2[r]);
                    if (MODEL == NET_MODEL_KS) ldg_vec<X>((const T*)a.omega + i, om[r]);
                }
            }
        }
        mbar_wait(full + slot, phase);
        if (owner) {
            const Pr* b = reinterpret_cast<const Pr*>(ring + (size_t)slot * plane_bytes) + (st * TY) * PW + q * X;
            Pr A[P > 1 ? P - 1 : 1][TY][X];      // in-plane sums of |dz| = 1 .. P-1
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
                const Pr* row = b + rr * PW;
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
                for (int i = 0; i < X; ++i) {
                    R[0][i] = v[OFF + P + i];
#pragma unroll
                    for (int w = 1; w <= P; ++w)
                        if (w <= wmax) R[w][i] = padd(R[w - 1][i], padd(v[OFF + P + i - w], v[OFF + P + i + w]));
                }
#pragma unroll
                for (int r = 0; r < TY; ++r) {
                    const int ady = rr - P - r < 0 ? -(rr - P - r) : rr - P - r;
                    if (ady > P) continue;
                    // |dz| = 0: straight into the accumulator of output plane p
                    {
                        const int w = l2_run_w(P, 0, ady);
#pragma unroll
                        for (int i = 0; i < X; ++i) acc[(J + P) % NACC][r][i] = padd(acc[(J + P) % NACC][r][i], R[w][i]);
                    }
                    // 0 < |dz| < P: in-plane partial sums
#pragma unroll
                    for (int k = 1; k < P; ++k) {
                        const int w = l2_run_w(P, k, ady);
                        if (w >= 0) {
#pragma unroll
                            for (int i = 0; i < X; ++i)
                                A[k - 1][r][i] = Aset[k - 1][r] ? padd(A[k - 1][r][i], R[w][i]) : R[w][i];
                            Aset[k - 1][r] = true;
                        }
                    }
                    // |dz| = P: the centre point alone.  Output plane p + P sees its first
                    // contribution (assignment), output plane p - P its last.
                    if (ady == 0) {
#pragma unroll
                        for (int i = 0; i < X; ++i) {
                            acc[(J + 2 * P) % NACC][r][i] = R[0][i];
                            acc[J % NACC][r][i] = padd(acc[J % NACC][r][i], R[0][i]);
                        }
                    }
                }
            }
#pragma unroll
            for (int k = 1; k < P; ++k)
#pragma unroll
                for (int r = 0; r < TY; ++r)
#pragma unroll
                    for (int i = 0; i < X; ++i) {
                        acc[(J + P - k) % NACC][r][i] = padd(acc[(J + P - k) % NACC][r][i], A[k - 1][r][i]);
                        acc[(J + P + k) % NACC][r][i] = padd(acc[(J + P + k) % NACC][r][i], A[k - 1][r][i]);
                    }
        }
        // ---- finish output plane zo (accumulator J)
        if (finishing) {
            const Pr* cb = reinterpret_cast<const Pr*>(ring + (size_t)cslot * plane_bytes) + (st * TY + P) * PW + q * X + HX;
#pragma unroll
            for (int r = 0; r < TY; ++r) {
                const int yy = yrow0 + r;
                if (yy < ny) {
                    const int64_t il = (int64_t)zo * nxy + (int64_t)yy * nx + x;                    // plain scalar arrays
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
                    T ov[EW], zv[EW], ev[2 * X];
#pragma unroll
                    for (int e = 0; e < X; ++e) {
                        const Pr c = cb[r * PW + e];
                        const Pr W = acc[J % NACC][r][e];
                        T k[NVS], yv[NVS], y2[NVS], y3[NVS];
                        if (MODEL == NET_MODEL_KS) {
                            T C = W.x, S = W.y;
                            if (!g.include_self) { C -= c.x; S -= c.y; }
                            k[0] = ks_rhs_factorised<T>(mp, om[r][e], C, S, c.x, c.y, inv_deg);
                            yv[0] = NOPS >= 1 ? o0[r][e] : T(0);
                            y2[0] = NOPS >= 2 ? o1[r][e] : T(0);
                            y3[0] = NOPS >= 3 ? o2[r][e] : T(0);
                        } else {
                            const T nb = T(g.n_ball);
                            const T Cu = W.x - nb * c.x, Cv = W.y - nb * c.y;
                            fhn_rhs<T>(mp, c.x, c.y, Cu, Cv, inv_deg, &k[0], &k[NVS - 1]);
                            // stage 0: y is the stage input itself; stage 2: Y3 is
                            yv[0] = NOPS >= 1 ? o0[r][2 * e] : c.x;
                            yv[NVS - 1] = NOPS >= 1 ? o0[r][2 * e + 1] : c.y;
                            y2[0] = NOPS >= 2 ? o1[r][2 * e] : T(0);
                            y2[NVS - 1] = NOPS >= 2 ? o1[r][2 * e + 1] : T(0);
                            y3[0] = c.x; y3[NVS - 1] = c.y;
                        }
#pragma unroll
                        for (int vv = 0; vv < NVS; ++vv) {
                            T o;
                            if (stage <= 1) o = yv[vv] + (T(0.5) * dt) * k[vv];
                            else if (stage == 2) {
                                o = yv[vv] + dt * k[vv];
                                zv[e * NVS + vv] = (y2[vv] + T(2) * y3[vv] + o - yv[vv]) * T(1.0 / 3.0);
                            } else if (stage == 3) o = yv[vv] + (dt * T(1.0 / 6.0)) * k[vv];   // yv = Z
                            else o = k[vv];
                            ov[e * NVS + vv] = o;
                        }
                        if (MODEL == NET_MODEL_KS && stage != STAGE_RHS_ONLY) {
                            T s_, c_;
                            Math<T>::sincos(ov[e], &s_, &c_);
                            ev[2 * e] = c_; ev[2 * e + 1] = s_;
                        }
                    }
                    if constexpr (MODEL == NET_MODEL_KS) {
                        stg_vec<EW>((T*)a.out + il, ov);
                        if (stage == 2) stg_vec<EW>((T*)a.out2 + il, zv);
                        if (stage != STAGE_RHS_ONLY) store_pairs((T*)a.Eout, ev);
                    } else {
                        store_pairs((T*)a.out, ov);
                        if (stage == 2) stg_vec<EW>((T*)a.out2 + 2 * ip, zv);    // Z is never a stencil source
                    }
                }
            }
        }
        __syncthreads();
        // the slot of plane idx - P is free: refill it with plane idx + D + 1
        if (tid == 0 && idx + D + 1 < nplanes) issue_plane(idx + D + 1, islot);
        slot = slot + 1 == NS ? 0 : slot + 1;
        cslot = cslot + 1 == NS ? 0 : cslot + 1;
        islot = islot + 1 == NS ? 0 : islot + 1;
        if (slot == 0) phase ^= 1u;
    };

    // planes in groups of NACC so that the accumulator roles are compile-time constants
    for (int base = 0; base < nplanes; base += NACC)
        l2_static_for<0, NACC>([&](auto Jc) {
            if (base + decltype(Jc)::value < nplanes) do_plane(base + decltype(Jc)::value, Jc);
        });
}

}  // namespace oscnet
