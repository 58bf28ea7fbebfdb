// FAST method for 3D periodic lattices (configs 3 and 5): tiled, z-marching ball sums.
//
// The coupling of eq. (2)/(3) over the ball (i-i')^2+(j-j')^2+(k-k')^2 <= P^2 is
// linear in the neighbours' exchange variables once the sine is factorised
//   sum_j sin(phi_j - phi_i - a) = S_i cos(phi_i + a) - C_i sin(phi_i + a),  (C,S) = sum_j (cos,sin) phi_j
// (FHN: sum_j (u_j - u_i) = U_i - Omega u_i), so every stage needs the ball sum of NF = 2 fields.
// The ball is decomposed into x-runs: for every (dz, dy) the points |dx| <= w(|dz|,|dy|),
// w = floor(sqrt(P^2 - dz^2 - dy^2)).  A CTA owns an xy tile (TX columns x S*TY rows) and marches
// along z over a chunk of planes.  Each plane (with its xy halo; periodic wrap resolved at load
// time) is staged once in shared memory -- for KS as (cos phi, sin phi), so the sincos is paid
// once per loaded element, not once per link -- and every thread, owning one column x and a
// strip of TY rows, forms the x-run sums R_w by sliding, the in-plane partial sums
// A_k(y) = sum_dy R_{w(k,dy)}(y+dy), k = |dz|, and adds A_|dz| into 2P+1 register accumulators
// of the output planes z-P..z+P.  The plane whose accumulator is complete is finished in
// registers: local vector field + fused RK4 stage update, coalesced store.
// Exact in real arithmetic; the rounding differs from the direct sum only by the order of the adds.
#include "models.cuh"

namespace oscnet {

constexpr int LAT_NLMAX = 8;   // staged-plane elements per thread per field (upper bound)

__host__ __device__ constexpr int lat_isqrt(int v) {
    int r = 0;
    while ((r + 1) * (r + 1) <= v) ++r;
    return r;
}
// half-width of the x-run at (|dz|, |dy|), -1 if the row does not meet the ball
__host__ __device__ constexpr int lat_run_w(int P, int adz, int ady) {
    int r = P * P - adz * adz - ady * ady;
    return r < 0 ? -1 : lat_isqrt(r);
}
// widest run any output of the strip needs from the staged row at distance `dist` (>= 0) from it
__host__ __device__ constexpr int lat_row_wmax(int P, int dist) { return lat_run_w(P, 0, dist); }

template <class T> __device__ __forceinline__ T ldg_stream(const T* p) { return __ldcs(p); }

template <class T, int MODEL, int P, int TY>
__global__ void __launch_bounds__(sizeof(T) == 8 ? 256 : 512) lattice3d_stage_kernel(StageArgs a, ModelParams mp, Lat3 g) {
    constexpr int NF = 2;                      // fields in the ball sum
    constexpr int NIN = MODEL == NET_MODEL_KS ? 1 : 2;   // state variables loaded per element
    constexpr int NB = P + 2;                  // staged planes kept: p+1 (being filled), p .. p-P
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* smem = reinterpret_cast<T*>(smem_raw);
    const int PW = g.PW, PH = g.PH;
    const int plane_elems = PW * PH;           // per field
    const int nx = g.nx, ny = g.ny, nz = g.nz;
    const int64_t ld = a.ld;
    const int64_t nxy = (int64_t)nx * ny;

    int bid = blockIdx.x;
    const int tix = bid % g.tiles_x; bid /= g.tiles_x;
    const int tiy = bid % g.tiles_y; bid /= g.tiles_y;
    const int x0 = tix * g.TX, y0 = tiy * (g.S * TY);
    const int z0 = bid * g.Lz;
    const int z1 = min(nz, z0 + g.Lz);
    const int tid = threadIdx.x;
    const int lx = tid % g.TX, st = tid / g.TX;
    const bool owner = st < g.S && x0 + lx < nx;
    const int yrow0 = y0 + st * TY;            // first row of the strip

    const T* __restrict__ in = (const T*)a.in;
    const T* __restrict__ yb = (const T*)a.y;
    const T* __restrict__ Y2 = (const T*)a.Y2;
    const T* __restrict__ Y3 = (const T*)a.Y3;
    const T* __restrict__ ep = (const T*)a.elem_param;
    T* __restrict__ out = (T*)a.out;
    const int stage = a.stage;
    const T dt = (T)a.dt;

    // ---- load slots of this thread inside a staged plane (z independent)
    int goff[LAT_NLMAX];
#pragma unroll
    for (int k = 0; k < LAT_NLMAX; ++k) {
        const int e = tid + k * blockDim.x;
        if (e < plane_elems) {
            const int row = e / PW, col = e - row * PW;
            int gx = x0 - P + col, gy = y0 - P + row;
            gx %= nx; if (gx < 0) gx += nx;
            gy %= ny; if (gy < 0) gy += ny;
            goff[k] = gy * nx + gx;
        } else goff[k] = -1;
    }
    T pre[NIN][LAT_NLMAX];
    auto plane_issue = [&](int p) {            // global -> registers
        int zz = p % nz; if (zz < 0) zz += nz;
        const T* base = in + (int64_t)zz * nxy;
#pragma unroll
        for (int k = 0; k < LAT_NLMAX; ++k)
#pragma unroll
            for (int v = 0; v < NIN; ++v)
                pre[v][k] = goff[k] >= 0 ? base[v * ld + goff[k]] : T(0);
    };
    auto plane_commit = [&](int slot) {        // registers -> shared (KS: as cos, sin)
        T* b = smem + (size_t)slot * NF * plane_elems;
#pragma unroll
        for (int k = 0; k < LAT_NLMAX; ++k) {
            const int e = tid + k * blockDim.x;
            if (goff[k] >= 0) {
                if (MODEL == NET_MODEL_KS) {
                    T s, c;
                    Math<T>::sincos(pre[0][k], &s, &c);
                    b[e] = c;
                    b[plane_elems + e] = s;
                } else {
                    b[e] = pre[0][k];
                    b[plane_elems + e] = pre[NIN - 1][k];
                }
            }
        }
    };

    T acc[2 * P + 1][NF][TY];
#pragma unroll
    for (int k = 0; k <= 2 * P; ++k)
#pragma unroll
        for (int f = 0; f < NF; ++f)
#pragma unroll
            for (int r = 0; r < TY; ++r) acc[k][f][r] = T(0);

    const T inv_deg = T(1) / T(g.n_ball - (g.include_self ? 0 : 1));
    int slot = 0;                               // slot of plane p
    plane_issue(z0 - P);
    plane_commit(0);
    __syncthreads();
    const int p_last = z1 - 1 + P;
    for (int p = z0 - P; p <= p_last; ++p) {
        const int slot_next = slot + 1 == NB ? 0 : slot + 1;
        if (p < p_last) plane_issue(p + 1);
        const int zo = p - P;                   // output plane completed by this iteration
        // ---- in-plane partial sums of plane p, added to the 2P+1 open output planes
        if (owner) {
            const T* b = smem + (size_t)slot * NF * plane_elems + (st * TY) * PW + lx;
#pragma unroll
            for (int f = 0; f < NF; ++f) {
                T A[P + 1][TY];
#pragma unroll
                for (int k = 0; k <= P; ++k)
#pragma unroll
                    for (int r = 0; r < TY; ++r) A[k][r] = T(0);
#pragma unroll
                for (int rr = 0; rr < TY + 2 * P; ++rr) {       // staged row rr <-> y = yrow0 - P + rr
                    // distance of this row from the strip, widest run needed from it
                    const int dist = rr < P ? P - rr : (rr >= TY + P ? rr - (TY + P - 1) : 0);
                    const int wmax = lat_row_wmax(P, dist);
                    const T* row = b + f * plane_elems + rr * PW + P;   // row[dx], dx = -P..P
                    T R[P + 1];
                    R[0] = row[0];
#pragma unroll
                    for (int w = 1; w <= P; ++w)
                        R[w] = w <= wmax ? R[w - 1] + (row[-w] + row[w]) : T(0);
#pragma unroll
                    for (int r = 0; r < TY; ++r) {
                        const int ady = rr - P - r < 0 ? -(rr - P - r) : rr - P - r;
                        if (ady <= P) {
#pragma unroll
                            for (int k = 0; k <= P; ++k) {
                                const int w = lat_run_w(P, k, ady);
                                if (w >= 0) A[k][r] += R[w];
                            }
                        }
                    }
                }
#pragma unroll
                for (int r = 0; r < TY; ++r) {
                    acc[P][f][r] += A[0][r];
#pragma unroll
                    for (int k = 1; k <= P; ++k) {
                        acc[P - k][f][r] += A[k][r];       // output planes p-P+(P-+k): |dz| = k
                        acc[P + k][f][r] += A[k][r];
                    }
                }
            }
        }
        // ---- finish output plane zo (accumulator 0)
        if (owner && zo >= z0) {
            int cslot = slot - P; if (cslot < 0) cslot += NB;    // staged plane zo (centre values)
            const T* cb = smem + (size_t)cslot * NF * plane_elems + (st * TY + P) * PW + lx + P;
#pragma unroll
            for (int r = 0; r < TY; ++r) {
                const int yy = yrow0 + r;
                if (yy < ny) {
                    const int64_t i = (int64_t)zo * nxy + (int64_t)yy * nx + (x0 + lx);
                    const T c0 = cb[r * PW], c1 = cb[plane_elems + r * PW];
                    constexpr int NV = MODEL == NET_MODEL_KS ? 1 : 2;
                    T k[NV], xin[NV];
                    if (MODEL == NET_MODEL_KS) {
                        T C = acc[0][0][r], Ssum = acc[0][1][r];
                        if (!g.include_self) { C -= c0; Ssum -= c1; }
                        k[0] = ks_rhs_factorised<T>(mp, ep[i], C, Ssum, c0, c1, inv_deg);
                        xin[0] = stage == 3 ? in[i] : T(0);
                    } else {
                        const T nb = T(g.n_ball);
                        const T Cu = acc[0][0][r] - nb * c0, Cv = acc[0][1][r] - nb * c1;
                        fhn_rhs<T>(mp, c0, c1, Cu, Cv, inv_deg, &k[0], &k[1]);
                        xin[0] = c0; xin[NV - 1] = c1;
                    }
#pragma unroll
                    for (int v = 0; v < NV; ++v) {
                        T y = 0, y2 = 0, y3 = 0;
                        if (stage != STAGE_RHS_ONLY) y = yb[v * ld + i];
                        if (stage == 3) { y2 = ldg_stream(Y2 + v * ld + i); y3 = ldg_stream(Y3 + v * ld + i); }
                        out[v * ld + i] = stage_combine<T>(stage, dt, k[v], y, y2, y3, xin[v]);
                    }
                }
            }
        }
        // ---- rotate the accumulators
#pragma unroll
        for (int k = 0; k < 2 * P; ++k)
#pragma unroll
            for (int f = 0; f < NF; ++f)
#pragma unroll
                for (int r = 0; r < TY; ++r) acc[k][f][r] = acc[k + 1][f][r];
#pragma unroll
        for (int f = 0; f < NF; ++f)
#pragma unroll
            for (int r = 0; r < TY; ++r) acc[2 * P][f][r] = T(0);
        if (p < p_last) plane_commit(slot_next);
        __syncthreads();
        slot = slot_next;
    }
}

// ------------------------------------------------------------------ host side
template <class T, int MODEL, int P, int TY>
static int32_t lat_configure(net* h) {
    Lat3& g = h->lat;
    const TopoView& tv = h->tv;
    g.nx = tv.nx; g.ny = tv.ny; g.nz = tv.nz;
    g.include_self = tv.include_self;
    g.n_ball = tv.noff + (tv.include_self ? 0 : 1);
    g.tiles_x = (g.nx + 127) / 128;
    g.TX = (g.nx + g.tiles_x - 1) / g.tiles_x;
    int strips = (g.ny + TY - 1) / TY;
    const int max_threads = sizeof(T) == 8 ? 256 : 512;   // = __launch_bounds__ of the kernel
    g.S = max_threads / g.TX < strips ? max_threads / g.TX : strips;
    if (g.S < 1) g.S = 1;
    g.tiles_y = (g.ny + g.S * TY - 1) / (g.S * TY);
    g.PW = g.TX + 2 * P;
    g.PH = g.S * TY + 2 * P;
    h->lat_threads = (g.TX * g.S + 31) / 32 * 32;
    if (g.PW * g.PH > LAT_NLMAX * h->lat_threads) return NET_ERR_UNSUPPORTED;
    h->lat_smem = sizeof(T) * (size_t)(P + 2) * 2 * g.PW * g.PH;
    if (h->lat_smem > 220 * 1024) return NET_ERR_UNSUPPORTED;
    auto kern = lattice3d_stage_kernel<T, MODEL, P, TY>;
    OSC_CUDA(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->lat_smem));
    int occ = 0;
    OSC_CUDA(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, h->lat_threads, h->lat_smem));
    if (occ < 1) return NET_ERR_UNSUPPORTED;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int64_t slots = (int64_t)occ * sms, tiles = (int64_t)g.tiles_x * g.tiles_y;
    // planes per chunk: fewest (waves x planes marched per CTA, halo included)
    int64_t best_cost = -1;
    for (int nch = 1; nch <= g.nz; ++nch) {
        const int Lz = (g.nz + nch - 1) / nch;
        const int chunks = (g.nz + Lz - 1) / Lz;
        const int64_t waves = (tiles * chunks + slots - 1) / slots;
        const int64_t cost = waves * (Lz + 2 * P + 1);
        if (best_cost < 0 || cost < best_cost) { best_cost = cost; g.Lz = Lz; g.nchunks = chunks; }
    }
    h->lat_grid = (unsigned)(tiles * g.nchunks);
    return NET_OK;
}

template <class T, int MODEL, int P, int TY>
static int32_t lat_launch(net* h, const StageArgs& a) {
    lattice3d_stage_kernel<T, MODEL, P, TY><<<h->lat_grid, h->lat_threads, h->lat_smem, h->stream>>>(a, h->mp, h->lat);
    h->launches += 1;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

// dispatch over (dtype, model, P); TY = 4 rows per thread for P <= 2, 2 above (register budget)
template <class T, int MODEL>
static int32_t lat_dispatch(net* h, const StageArgs* a) {
    switch (h->tv.P) {
        case 1: return a ? lat_launch<T, MODEL, 1, 4>(h, *a) : lat_configure<T, MODEL, 1, 4>(h);
        case 2: return a ? lat_launch<T, MODEL, 2, 4>(h, *a) : lat_configure<T, MODEL, 2, 4>(h);
        case 3: return a ? lat_launch<T, MODEL, 3, 2>(h, *a) : lat_configure<T, MODEL, 3, 2>(h);
        case 4: return a ? lat_launch<T, MODEL, 4, 2>(h, *a) : lat_configure<T, MODEL, 4, 2>(h);
        default: return NET_ERR_UNSUPPORTED;
    }
}

static int32_t lat_entry(net* h, const StageArgs* a) {
    const bool f32 = h->desc.dtype == NET_F32;
    if (h->desc.model == NET_MODEL_KS)
        return f32 ? lat_dispatch<float, NET_MODEL_KS>(h, a) : lat_dispatch<double, NET_MODEL_KS>(h, a);
    return f32 ? lat_dispatch<float, NET_MODEL_FHN>(h, a) : lat_dispatch<double, NET_MODEL_FHN>(h, a);
}

bool lattice3d_supported(const net_desc* d) {
    const net_topology& t = d->topo;
    return t.kind == NET_TOPO_LATTICE && t.ndim == 3 && t.radius >= 1 && t.radius <= 4 &&
           (d->model == NET_MODEL_KS || d->model == NET_MODEL_FHN);
}
int32_t lattice3d_prepare(net* h) { return lat_entry(h, nullptr); }
int32_t lattice3d_stage(net* h, const StageArgs& a) { return lat_entry(h, &a); }

}  // namespace oscnet
