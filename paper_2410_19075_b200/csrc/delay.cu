// NET_MODEL_FHN2: FitzHugh-Nagumo exactly as eq. (2) of the paper -- x-only
// coupling with delay tau, applied current, additive noise on y -- under the fixed-step RK4 of
// net_integrate (reading R17):
//   tau = delay_steps * dt.  The workspace keeps x_j and dx_j/dt (= the k1 of that step) at the last
//   delay_steps + 2 step times, slot of step q = q mod (delay_steps + 2) ("maintaining data from
//   previous time steps and performing interpolation").  The four RK4 stages of step n
//   read x_j(t - tau) as
//       stage 0 (t_n):          H[n - m]
//       stages 1, 2 (t_n+dt/2): cubic Hermite midpoint of H[n - m], H[n - m + 1]
//                               (the constant initial value while n < m: dx/dt jumps at t = 0)
//       stage 3 (t_n + dt):     H[n - m + 1]
//   and stage 0 records (x, k1_x) of step n.  m = 0: the stage values themselves.
//   Noise: after the last stage y_i += D sqrt(dt) xi(seed, i, n), xi = sqrt(-2 ln u1) cos(2 pi u2)
//   with u1, u2 from the splitmix64 finaliser of reading R8 keyed by (seed, i, 2n+1 / 2n+2).
// One thread per element, one term per link (the form of Alg. 1), every topology kind.
#include "models.cuh"

namespace oscnet {

namespace {

struct DelayArgs {
    const void* xa;      // H[n - m]      x
    const void* da;      //               dx/dt
    const void* xb;      // H[n - m + 1]  x
    const void* db;
    void* rec_x;         // stage 0: slot of step n
    void* rec_d;
    int mode;            // 0: xa, 1: Hermite midpoint, 2: xb, 3: the stage input itself (no delay), 4: xa (constant history)
    double dt8;          // dt / 8
    double noise_amp;    // D sqrt(dt) (stage 3), else 0
    long long step;      // n
};

__device__ __forceinline__ unsigned long long dl_mix64(unsigned long long z) {
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27; z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}

__device__ __forceinline__ double dl_gauss(unsigned long long seed, long long i, long long n) {
    const unsigned long long G = 0x9E3779B97F4A7C15ULL;
    const unsigned long long hi = dl_mix64(seed + G * (unsigned long long)(i + 1));
    const unsigned long long a = dl_mix64(hi + G * (unsigned long long)(2 * n + 1));
    const unsigned long long b = dl_mix64(hi + G * (unsigned long long)(2 * n + 2));
    const double u1 = ((double)(a >> 11) + 1.0) * (1.0 / 9007199254740992.0);
    const double u2 = (double)(b >> 11) * (1.0 / 9007199254740992.0);
    return sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925286766559 * u2);
}

template <class T, int TOPO>
__global__ void __launch_bounds__(256) fhn2_stage_kernel(StageArgs a, ModelParams mp, TopoView tv, DelayArgs d) {
    const int64_t n = a.n, ld = a.ld;
    const T* __restrict__ in = (const T*)a.in;
    const T* __restrict__ xa = (const T*)d.xa;
    const T* __restrict__ da = (const T*)d.da;
    const T* __restrict__ xb = (const T*)d.xb;
    const T* __restrict__ db = (const T*)d.db;
    const int stage = a.stage, mode = d.mode;
    const T dt = (T)a.dt, dt8 = (T)d.dt8;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const T x = in[i], y = in[ld + i];
        T Cx = 0;
        const int deg = for_each_neighbor<TOPO>(tv, n, i, [&](int64_t j) {
            T xd;
            if (mode == 3) xd = in[j];
            else if (mode == 1) xd = T(0.5) * (xa[j] + xb[j]) + dt8 * (da[j] - db[j]);
            else if (mode == 2) xd = xb[j];
            else xd = xa[j];
            Cx += xd - x;
        });
        const T s = deg > 0 ? T(mp.sigma) / T(deg) : T(0);
        T k[2];
        k[0] = (x - x * x * x * T(1.0 / 3.0) - y + s * Cx + T(mp.I_app)) * T(mp.inv_eps);
        k[1] = x + T(mp.a);
        if (d.rec_x) { ((T*)d.rec_x)[i] = x; ((T*)d.rec_d)[i] = k[0]; }
        const T xin[2] = {x, y};
#pragma unroll
        for (int v = 0; v < 2; ++v) {
            T yb = 0, y2 = 0, y3 = 0;
            if (stage != STAGE_RHS_ONLY) yb = ((const T*)a.y)[v * ld + i];
            if (stage == 3) { y2 = ((const T*)a.Y2)[v * ld + i]; y3 = ((const T*)a.Y3)[v * ld + i]; }
            T o = stage_combine<T>(stage, dt, k[v], yb, y2, y3, xin[v]);
            if (v == 1 && d.noise_amp != 0.0) o += (T)(d.noise_amp * dl_gauss(mp.noise_seed, i, d.step));
            ((T*)a.out)[v * ld + i] = o;
        }
    }
}

template <class T>
__global__ void fhn2_reset_kernel(const T* __restrict__ x, T* __restrict__ hx, T* __restrict__ hd, int64_t n, int64_t ld, int slots) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        for (int q = 0; q < slots; ++q) { hx[(int64_t)q * ld + i] = x[i]; hd[(int64_t)q * ld + i] = T(0); }
}

template <class T>
int32_t launch(net* h, const StageArgs& a, const DelayArgs& d) {
    int64_t blocks = (a.n + 255) / 256;
    if (blocks > 148 * 64) blocks = 148 * 64;
    dim3 g((unsigned)blocks), b(256);
    switch (h->tv.kind) {
        case NET_TOPO_RING: fhn2_stage_kernel<T, NET_TOPO_RING><<<g, b, 0, h->stream>>>(a, h->mp, h->tv, d); break;
        case NET_TOPO_LATTICE: fhn2_stage_kernel<T, NET_TOPO_LATTICE><<<g, b, 0, h->stream>>>(a, h->mp, h->tv, d); break;
        case NET_TOPO_CSR: fhn2_stage_kernel<T, NET_TOPO_CSR><<<g, b, 0, h->stream>>>(a, h->mp, h->tv, d); break;
        case NET_TOPO_COMPRESSED: fhn2_stage_kernel<T, NET_TOPO_COMPRESSED><<<g, b, 0, h->stream>>>(a, h->mp, h->tv, d); break;
        default: fhn2_stage_kernel<T, NET_TOPO_RANDOM_INDEGREE><<<g, b, 0, h->stream>>>(a, h->mp, h->tv, d); break;
    }
    h->launches += 1;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

}  // namespace

// every slot of the history ring <- the current x, derivative 0 (constant initial function)
int32_t delay_reset_history(net* h) {
    const int slots = h->desc.delay_steps + 2;
    int64_t blocks = (h->n + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    if (h->desc.dtype == NET_F32)
        fhn2_reset_kernel<float><<<(unsigned)blocks, 256, 0, h->stream>>>((const float*)h->b.y, (float*)h->b.hist_x, (float*)h->b.hist_d, h->n, h->ld, slots);
    else
        fhn2_reset_kernel<double><<<(unsigned)blocks, 256, 0, h->stream>>>((const double*)h->b.y, (double*)h->b.hist_x, (double*)h->b.hist_d, h->n, h->ld, slots);
    h->launches += 1;
    h->hist_step = 0;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

int32_t delay_stage(net* h, const StageArgs& a) {
    const int64_t m = h->desc.delay_steps, S = m + 2, st = h->hist_step;
    const size_t slot = (size_t)h->ld * h->esize;
    auto sx = [&](int64_t q) { return (char*)h->b.hist_x + (size_t)(((q % S) + S) % S) * slot; };
    auto sd = [&](int64_t q) { return (char*)h->b.hist_d + (size_t)(((q % S) + S) % S) * slot; };
    DelayArgs d;
    memset(&d, 0, sizeof(d));
    d.xa = sx(st - m); d.da = sd(st - m); d.xb = sx(st - m + 1); d.db = sd(st - m + 1);
    d.dt8 = a.dt * 0.125;
    d.step = st;
    if (a.stage == STAGE_RHS_ONLY || m == 0) d.mode = 3;
    else if (a.stage == 0) d.mode = 0;
    else if (a.stage == 3) d.mode = 2;
    else d.mode = st < m ? 4 : 1;
    if (a.stage == 0) { d.rec_x = sx(st); d.rec_d = sd(st); }
    if (a.stage == 3 && h->mp.noise_D != 0.0) d.noise_amp = h->mp.noise_D * sqrt(a.dt);
    return h->desc.dtype == NET_F32 ? launch<float>(h, a, d) : launch<double>(h, a, d);
}

}  // namespace oscnet
