// Observable kernels: phase maps, global / local Kuramoto order parameter, mean phase
// velocity and the long-run statistics window (reading R9; the paper names the
// analyses -- PAPER.md:301 average frequencies, :325 coherent/incoherent regions, :416
// "synchronization analysis at each output" -- without formulas).  All in double, all
// reductions in a fixed order (deterministic).
#include "models.cuh"

namespace oscnet {

constexpr int RED_BLOCKS = 592;  // 4 per SM
constexpr int RED_THREADS = 256;

template <class T>
__global__ void phase_kernel(const T* __restrict__ y, int64_t n, int64_t ld, int model,
                             ModelParams mp, double* __restrict__ theta) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
        double th;
        if (model == NET_MODEL_KS || model == NET_MODEL_KSI) th = (double)y[i];
        else if (model == NET_MODEL_FHN || model == NET_MODEL_FHN2) th = atan2((double)y[ld + i], (double)y[i]);
        else th = atan2((double)y[3 * ld + i] - mp.n_c, ((double)y[i] - mp.V_c) * mp.inv_V_s);
        theta[i] = th;
    }
}

__device__ __forceinline__ double block_sum(double v, double* sh) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) sh[w] = v;
    __syncthreads();
    double r = 0;
    if (threadIdx.x == 0)
        for (int q = 0; q < (int)(blockDim.x >> 5); ++q) r += sh[q];
    __syncthreads();
    return r;  // valid in thread 0
}

// mode 0: partial[2b..] = sum (cos th, sin th); mode 1: sum (x, 0); mode 2: sum ((x-mean)^2, 0)
__global__ void reduce_partial_kernel(const double* __restrict__ x, int64_t n, int mode,
                                      const double* __restrict__ mean_ptr, double* __restrict__ partial) {
    __shared__ double sh[8];
    double a = 0, b = 0;
    const double mean = (mode == 2) ? mean_ptr[0] : 0.0;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
        double v = x[i];
        if (mode == 0) { double s, c; sincos(v, &s, &c); a += c; b += s; }
        else if (mode == 1) a += v;
        else { double d = v - mean; a += d * d; }
    }
    double ra = block_sum(a, sh);
    double rb = block_sum(b, sh);
    if (threadIdx.x == 0) { partial[2 * blockIdx.x] = ra; partial[2 * blockIdx.x + 1] = rb; }
}

// finish modes: 0 -> out[0]=R, out[1]=Psi (and acc[0]+=R, acc[1]+=R^2, acc[2]+=1 if acc);
//               1 -> out[0] = sum/n ; 2 -> out[0] = sqrt(sum/n)
__global__ void reduce_finish_kernel(const double* __restrict__ partial, int nb, int64_t n, int mode,
                                     double* __restrict__ out, double* __restrict__ acc) {
    __shared__ double sh[8];
    double a = 0, b = 0;
    for (int q = threadIdx.x; q < nb; q += blockDim.x) { a += partial[2 * q]; b += partial[2 * q + 1]; }
    double ra = block_sum(a, sh);
    double rb = block_sum(b, sh);
    if (threadIdx.x == 0) {
        if (mode == 0) {
            double c = ra / (double)n, s = rb / (double)n;
            double R = sqrt(c * c + s * s);
            out[0] = R;
            out[1] = atan2(s, c);
            if (acc) { acc[0] += R; acc[1] += R * R; acc[2] += 1.0; }
        } else if (mode == 1) out[0] = ra / (double)n;
        else out[0] = sqrt(ra / (double)n);
    }
}

// Order parameter of every replica of a batch: CTA r reduces elements [r*rn, (r+1)*rn) in a fixed
// order; out[2r] = R_r, out[2r+1] = Psi_r.
__global__ void replica_order_kernel(const double* __restrict__ theta, int64_t rn, double* __restrict__ out) {
    __shared__ double sh[8];
    const double* th = theta + (int64_t)blockIdx.x * rn;
    double a = 0, b = 0;
    for (int64_t i = threadIdx.x; i < rn; i += blockDim.x) {
        double s, c;
        sincos(th[i], &s, &c);
        a += c; b += s;
    }
    const double ra = block_sum(a, sh);
    const double rb = block_sum(b, sh);
    if (threadIdx.x == 0) {
        const double c = ra / (double)rn, s = rb / (double)rn;
        out[2 * blockIdx.x] = sqrt(c * c + s * s);
        out[2 * blockIdx.x + 1] = atan2(s, c);
    }
}

__global__ void cossin_kernel(const double* __restrict__ theta, int64_t n, double* __restrict__ cs) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
        double s, c;
        sincos(theta[i], &s, &c);
        cs[i] = c;
        cs[n + i] = s;
    }
}

template <int TOPO>
__global__ void local_order_kernel(TopoView tv, int64_t n, const double* __restrict__ cs,
                                   double* __restrict__ out) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
        double c = 0, s = 0;
        bool has_self = false;
        int deg = for_each_neighbor<TOPO>(tv, n, i, [&](int64_t j) {
            if (j == i) has_self = true;
            c += cs[j];
            s += cs[n + j];
        });
        if (!has_self) { c += cs[i]; s += cs[n + i]; ++deg; }
        out[i] = sqrt(c * c + s * s) / (double)deg;
    }
}

static unsigned grid_for(int64_t items) {
    int64_t b = (items + 255) / 256;
    if (b < 1) b = 1;
    if (b > 148 * 16) b = 148 * 16;
    return (unsigned)b;
}

int32_t obs_phase(net* h, const void* state, double* d_theta) {
    if (h->pairs) {   // padded pair layout: through Y3 (dead between steps) as SoA
        int32_t rc = pairs_unpack(h, state, h->b.Y3);
        if (rc) return rc;
        state = h->b.Y3;
    }
    if (h->desc.dtype == NET_F32)
        phase_kernel<float><<<grid_for(h->n), 256, 0, h->stream>>>((const float*)state, h->n, h->ld, h->desc.model, h->mp, d_theta);
    else
        phase_kernel<double><<<grid_for(h->n), 256, 0, h->stream>>>((const double*)state, h->n, h->ld, h->desc.model, h->mp, d_theta);
    h->launches += 1;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

static int32_t reduce(net* h, const double* x, int mode, const double* mean, double* out, double* acc) {
    reduce_partial_kernel<<<RED_BLOCKS, RED_THREADS, 0, h->stream>>>(x, h->n, mode, mean, h->b.obs_partial);
    reduce_finish_kernel<<<1, RED_THREADS, 0, h->stream>>>(h->b.obs_partial, RED_BLOCKS, h->n, mode, out, acc);
    h->launches += 2;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

int32_t obs_global_order(net* h, const double* d_theta, double* d_out2) {
    return reduce(h, d_theta, 0, nullptr, d_out2, nullptr);
}

int32_t obs_replica_order(net* h, const double* d_theta, double* d_out) {
    const int batch = h->desc.batch > 0 ? h->desc.batch : 1;
    replica_order_kernel<<<batch, RED_THREADS, 0, h->stream>>>(d_theta, h->n / batch, d_out);
    h->launches += 1;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

// Rings: the window sum of (cos, sin) theta over |j - i| <= P is a difference of prefix sums -- the
// same machinery as the ring stage kernel.  In-place inclusive scan of the two
// rows of cs (one CTA; the rings are small), then one thread per element.
__global__ void __launch_bounds__(1024) ring_prefix_kernel(double* __restrict__ cs, int64_t n) {
    __shared__ double wsum[2][32];
    __shared__ double carry[2];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x < 2) carry[threadIdx.x] = 0.0;
    __syncthreads();
    for (int64_t base = 0; base < n; base += 1024) {
        const int64_t i = base + threadIdx.x;
        double a = i < n ? cs[i] : 0.0, b = i < n ? cs[n + i] : 0.0;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const double ua = __shfl_up_sync(0xffffffffu, a, o), ub = __shfl_up_sync(0xffffffffu, b, o);
            if (lane >= o) { a += ua; b += ub; }
        }
        if (lane == 31) { wsum[0][warp] = a; wsum[1][warp] = b; }
        __syncthreads();
        double oa = carry[0], ob = carry[1];
        for (int w = 0; w < warp; ++w) { oa += wsum[0][w]; ob += wsum[1][w]; }
        a += oa; b += ob;
        if (i < n) { cs[i] = a; cs[n + i] = b; }
        __syncthreads();
        if (threadIdx.x == 1023) { carry[0] = a; carry[1] = b; }
        __syncthreads();
    }
}

// pre = inclusive prefix of (cos | sin) over all rings back to back; ring r = elements [r rn, (r+1) rn)
__global__ void ring_local_order_kernel(const double* __restrict__ pre, int64_t n, int64_t rn, int P, double* __restrict__ out) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t base = i / rn * rn, il = i - base;
        auto pref = [&](const double* p, int64_t j) { return j < 0 ? 0.0 : p[j]; };     // Pref(-1) = 0
        double w[2];
#pragma unroll
        for (int f = 0; f < 2; ++f) {
            const double* p = pre + (int64_t)f * n;
            const double before = pref(p, base - 1), total = p[base + rn - 1] - before;   // this ring alone
            int64_t lo = il - P, hi = il + P;                                             // window [lo, hi], self included
            double s = 0.0;
            if (lo < 0) { s += total - (p[base + lo + rn - 1] - before); lo = 0; }        // tail of the ring
            if (hi >= rn) { s += p[base + hi - rn] - before; hi = rn - 1; }               // head of the ring
            s += p[base + hi] - pref(p, base + lo - 1);
            w[f] = s;
        }
        out[i] = sqrt(w[0] * w[0] + w[1] * w[1]) / (double)(2 * P + 1);
    }
}

int32_t obs_local_order(net* h, const double* d_theta, double* d_out) {
    // 3D lattices on the tiled kernels: the ball-sum instance of the stage kernel (lattice_v2.cu)
    if (lattice_v3_has_local_order(h)) return lattice_v3_local_order(h, d_out);
    cossin_kernel<<<grid_for(h->n), 256, 0, h->stream>>>(d_theta, h->n, h->b.obs_tmp);
    if (h->tv.kind == NET_TOPO_RING && 2 * (int64_t)h->tv.P + 1 <= h->tv.ring_n) {
        ring_prefix_kernel<<<1, 1024, 0, h->stream>>>(h->b.obs_tmp, h->n);
        ring_local_order_kernel<<<grid_for(h->n), 256, 0, h->stream>>>(h->b.obs_tmp, h->n, h->tv.ring_n, h->tv.P, d_out);
        h->launches += 3;
        OSC_CUDA(h, cudaGetLastError());
        return NET_OK;
    }
    unsigned g = grid_for(h->n);
    switch (h->tv.kind) {
        case NET_TOPO_RING: local_order_kernel<NET_TOPO_RING><<<g, 256, 0, h->stream>>>(h->tv, h->n, h->b.obs_tmp, d_out); break;
        case NET_TOPO_LATTICE: local_order_kernel<NET_TOPO_LATTICE><<<g, 256, 0, h->stream>>>(h->tv, h->n, h->b.obs_tmp, d_out); break;
        case NET_TOPO_CSR: local_order_kernel<NET_TOPO_CSR><<<g, 256, 0, h->stream>>>(h->tv, h->n, h->b.obs_tmp, d_out); break;
        case NET_TOPO_COMPRESSED: local_order_kernel<NET_TOPO_COMPRESSED><<<g, 256, 0, h->stream>>>(h->tv, h->n, h->b.obs_tmp, d_out); break;
        default: local_order_kernel<NET_TOPO_RANDOM_INDEGREE><<<g, 256, 0, h->stream>>>(h->tv, h->n, h->b.obs_tmp, d_out); break;
    }
    h->launches += 2;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

// ------------------------------------------------------------ statistics window
// acc layout (doubles): 0 sum R, 1 sum R^2, 2 samples, 3..4 scratch {R,Psi}, 5 mean Rloc,
//                       6 mean vel, 7 std vel
template <class T>
__global__ void window_begin_kernel(const double* __restrict__ theta, const T* __restrict__ y,
                                    int64_t n, double* __restrict__ prev, double* __restrict__ wind,
                                    double* __restrict__ ref) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
        prev[i] = theta[i];
        wind[i] = 0.0;
        ref[i] = (double)y[i];
    }
}

__global__ void window_accum_kernel(const double* __restrict__ theta, int64_t n,
                                    double* __restrict__ prev, double* __restrict__ wind) {
    const double TWO_PI = 6.283185307179586476925286766559;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
        double d = theta[i] - prev[i];
        wind[i] += d - TWO_PI * rint(d / TWO_PI);
        prev[i] = theta[i];
    }
}

template <class T>
__global__ void window_velocity_kernel(const T* __restrict__ y, const double* __restrict__ ref,
                                       const double* __restrict__ wind, int64_t n, int is_ks,
                                       double inv_T, double* __restrict__ vel) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x)
        vel[i] = is_ks ? ((double)y[i] - ref[i]) * inv_T : wind[i] * inv_T;
}

int32_t obs_window_begin(net* h) {
    OSC_CUDA(h, cudaMemsetAsync(h->b.obs_acc, 0, 16 * sizeof(double), h->stream));
    return NET_OK;
}

// Called at every sample inside the window.  `first` = first sample of the window (t_a).
int32_t obs_window_sample(net* h, int first) {
    double* theta = h->b.obs_loc;  // reuse as theta scratch during the window
    int32_t rc = obs_phase(h, h->b.y, theta);
    if (rc) return rc;
    rc = reduce(h, theta, 0, nullptr, h->b.obs_acc + 3, h->b.obs_acc);
    if (rc) return rc;
    unsigned g = grid_for(h->n);
    if (first) {
        if (h->desc.dtype == NET_F32)
            window_begin_kernel<float><<<g, 256, 0, h->stream>>>(theta, (const float*)h->b.y, h->n, h->b.obs_theta_prev, h->b.obs_wind, h->b.obs_ref);
        else
            window_begin_kernel<double><<<g, 256, 0, h->stream>>>(theta, (const double*)h->b.y, h->n, h->b.obs_theta_prev, h->b.obs_wind, h->b.obs_ref);
    } else {
        window_accum_kernel<<<g, 256, 0, h->stream>>>(theta, h->n, h->b.obs_theta_prev, h->b.obs_wind);
    }
    h->launches += 1;
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

int32_t obs_window_finish(net* h, double t_a, double t_b, int64_t n_samples) {
    double T = t_b - t_a;
    double inv_T = T > 0 ? 1.0 / T : 0.0;
    unsigned g = grid_for(h->n);
    int is_ks = h->desc.model == NET_MODEL_KS || h->desc.model == NET_MODEL_KSI;
    if (h->desc.dtype == NET_F32)
        window_velocity_kernel<float><<<g, 256, 0, h->stream>>>((const float*)h->b.y, h->b.obs_ref, h->b.obs_wind, h->n, is_ks, inv_T, h->b.obs_vel);
    else
        window_velocity_kernel<double><<<g, 256, 0, h->stream>>>((const double*)h->b.y, h->b.obs_ref, h->b.obs_wind, h->n, is_ks, inv_T, h->b.obs_vel);
    h->launches += 1;
    OSC_CUDA(h, cudaGetLastError());
    int32_t rc;
    if ((rc = reduce(h, h->b.obs_vel, 1, nullptr, h->b.obs_acc + 6, nullptr))) return rc;
    if ((rc = reduce(h, h->b.obs_vel, 2, h->b.obs_acc + 6, h->b.obs_acc + 7, nullptr))) return rc;
    // local order at the last sample (theta of the final state is still in obs_theta_prev)
    if ((rc = obs_local_order(h, h->b.obs_theta_prev, h->b.obs_loc))) return rc;
    if ((rc = reduce(h, h->b.obs_loc, 1, nullptr, h->b.obs_acc + 5, nullptr))) return rc;
    double acc[8];
    OSC_CUDA(h, cudaMemcpyAsync(acc, h->b.obs_acc, sizeof(acc), cudaMemcpyDeviceToHost, h->stream));
    OSC_CUDA(h, cudaStreamSynchronize(h->stream));
    double m = acc[2] > 0 ? acc[0] / acc[2] : 0.0;
    double var = acc[2] > 0 ? acc[1] / acc[2] - m * m : 0.0;
    h->stats[0] = m;
    h->stats[1] = var > 0 ? sqrt(var) : 0.0;
    h->stats[2] = acc[5];
    h->stats[3] = acc[6];
    h->stats[4] = acc[7];
    h->stats[5] = (double)n_samples;
    h->stats[6] = t_a;
    h->stats[7] = t_b;
    h->stats_valid = 1;
    return NET_OK;
}

}  // namespace oscnet
