// Adaptive Dormand-Prince 5(4) on the device (the solver the paper names first,
// PAPER.md:99).  Tableau and controller: the textbook DOPRI5 of the paper's reference [22]
// (reading R15):
//   k_s = f(y + h sum_{j<s} a_sj k_j), y5 = y + h sum b_j k_j (b = a_7.), first-same-as-last,
//   err = sqrt(mean((h sum e_j k_j / (atol + rtol max(|y|, |y5|)))^2)), accept iff err <= 1,
//   h <- h min(facmax, max(0.2, 0.9 err^-1/5)), facmax 10 (1 right after a rejection),
//   last step cut to land on t_end.
// Every right-hand side is the net's own fused RHS kernel family (whatever net_eval_rhs runs:
// field-split lattice kernels, ring prefix sums, blocked CSR, ...).  The step size, the time, the
// accept / reject decision and the counters live in device memory: the error norm is reduced by
// the last block of dp5_error_kernel, which also takes the decision and sets the next step, and
// dp5_commit_kernel applies it, so the host enqueues attempts blindly, DP5_BATCH at a time, and
// reads the control block back once per batch (no round trip per step).  Attempts enqueued after
// t_end was reached leave every vector untouched.
#include <math.h>

#include "oscnet_internal.cuh"

namespace oscnet {

namespace {

constexpr int DP5_BATCH = 8;         // attempts per host read-back
constexpr int DP5_THREADS = 256;
constexpr int DP5_MAXBLOCKS = 1184;

struct Dp5Ctrl {
    double t, h, t_end, rtol, atol, err, h_used;
    long long accepted, rejected, attempts, max_attempts;
    int done, after_reject, last, accept;
    unsigned ticket;
    int pad_;
};

__constant__ double DP5_A[7][6] = {
    {0, 0, 0, 0, 0, 0},
    {1.0 / 5.0, 0, 0, 0, 0, 0},
    {3.0 / 40.0, 9.0 / 40.0, 0, 0, 0, 0},
    {44.0 / 45.0, -56.0 / 15.0, 32.0 / 9.0, 0, 0, 0},
    {19372.0 / 6561.0, -25360.0 / 2187.0, 64448.0 / 6561.0, -212.0 / 729.0, 0, 0},
    {9017.0 / 3168.0, -355.0 / 33.0, 46732.0 / 5247.0, 49.0 / 176.0, -5103.0 / 18656.0, 0},
    {35.0 / 384.0, 0.0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 11.0 / 84.0}};
__constant__ double DP5_E[7] = {71.0 / 57600.0, 0.0, -71.0 / 16695.0, 71.0 / 1920.0,
                                -17253.0 / 339200.0, 22.0 / 525.0, -1.0 / 40.0};

struct Dp5Vecs {
    void* y;
    void* y5;
    void* tmp;
    void* k[7];
};

// start of an attempt: the last step is cut to land on t_end
__global__ void dp5_begin_kernel(Dp5Ctrl* c) {
    if (c->done) return;
    if (c->attempts >= c->max_attempts) { c->done = 2; return; }
    c->last = 0;
    if (c->t + 1.01 * c->h >= c->t_end) { c->h = c->t_end - c->t; c->last = 1; }
}

// dst = y + h sum_{j<s} a_sj k_j   (s = 1..6; s = 6 writes y5)
template <class T>
__global__ void __launch_bounds__(DP5_THREADS) dp5_stage_kernel(const Dp5Ctrl* c, Dp5Vecs v, int s, int64_t len) {
    if (c->done) return;
    const double h = c->h;
    const T* y = (const T*)v.y;
    T* dst = (T*)(s == 6 ? v.y5 : v.tmp);
    for (int64_t q = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; q < len; q += (int64_t)gridDim.x * blockDim.x) {
        double acc = 0.0;
        for (int j = 0; j < s; ++j) acc += DP5_A[s][j] * (double)((const T*)v.k[j])[q];
        dst[q] = (T)((double)y[q] + h * acc);
    }
}

// error norm (block partials; the last block to finish sums them in index order, decides, and sets
// the next step and time)
template <class T>
__global__ void __launch_bounds__(DP5_THREADS) dp5_error_kernel(Dp5Ctrl* c, Dp5Vecs v, int64_t len, double* partial) {
    if (c->done) return;
    __shared__ double red[DP5_THREADS];
    __shared__ bool is_last;
    const double h = c->h, rtol = c->rtol, atol = c->atol;
    const T* y = (const T*)v.y;
    const T* y5 = (const T*)v.y5;
    double s2 = 0.0;
    for (int64_t q = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; q < len; q += (int64_t)gridDim.x * blockDim.x) {
        double acc = 0.0;
#pragma unroll
        for (int j = 0; j < 7; ++j) acc += DP5_E[j] * (double)((const T*)v.k[j])[q];
        const double sc = atol + rtol * fmax(fabs((double)y[q]), fabs((double)y5[q]));
        const double r = h * acc / sc;
        s2 += r * r;
    }
    red[threadIdx.x] = s2;
    __syncthreads();
    for (int o = DP5_THREADS / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        partial[blockIdx.x] = red[0];
        __threadfence();
        is_last = atomicAdd(&c->ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    double tot = 0.0;
    for (unsigned b = threadIdx.x; b < gridDim.x; b += DP5_THREADS) tot += __ldcg(partial + b);
    red[threadIdx.x] = tot;
    __syncthreads();
    for (int o = DP5_THREADS / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        c->ticket = 0;
        const double err = sqrt(red[0] / (double)len);
        const double facmax = c->after_reject ? 1.0 : 10.0;
        double fac = err > 0.0 ? 0.9 * pow(err, -0.2) : facmax;
        fac = fmin(facmax, fmax(0.2, fac));
        c->err = err;
        c->attempts += 1;
        if (err <= 1.0) {           // (a NaN error is a rejection with the smallest factor)
            c->accept = 1;
            c->t = c->last ? c->t_end : c->t + c->h;
            c->h_used = c->h;
            c->accepted += 1;
            c->after_reject = 0;
        } else {
            c->accept = 0;
            c->rejected += 1;
            c->after_reject = 1;
            if (!(err == err)) fac = 0.2;
        }
        c->h *= fac;
    }
}

// accepted: y <- y5, k1 <- k7 (first same as last); reached t_end: done
template <class T>
__global__ void __launch_bounds__(DP5_THREADS) dp5_commit_kernel(Dp5Ctrl* c, Dp5Vecs v, int64_t len) {
    if (c->done) return;
    if (c->accept) {
        T* y = (T*)v.y;
        const T* y5 = (const T*)v.y5;
        T* k1 = (T*)v.k[0];
        const T* k7 = (const T*)v.k[6];
        for (int64_t q = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; q < len; q += (int64_t)gridDim.x * blockDim.x) {
            y[q] = y5[q];
            k1[q] = k7[q];
        }
    }
}

// after every block of the commit kernel has run (next kernel on the stream)
__global__ void dp5_end_kernel(Dp5Ctrl* c) {
    if (c->done) return;
    if (c->accept && !(c->t < c->t_end)) c->done = 1;
    c->accept = 0;
}

size_t dp5_vec_bytes(const net* h) { return (size_t)round_up((int64_t)h->nvar * h->n * h->esize, 256); }

}  // namespace

size_t adaptive_workspace_bytes(const net* h) {
    return 10 * dp5_vec_bytes(h) + 256 + sizeof(double) * DP5_MAXBLOCKS + 256;
}

template <class T>
static int32_t dp5_run(net* h, double t_end, double rtol, double atol, double h0, int64_t max_attempts,
                       char* work, double* out5) {
    const size_t vb = dp5_vec_bytes(h);
    Dp5Vecs v;
    v.y = work; v.y5 = work + vb; v.tmp = work + 2 * vb;
    for (int j = 0; j < 7; ++j) v.k[j] = work + (3 + j) * vb;
    Dp5Ctrl* d_c = (Dp5Ctrl*)(work + 10 * vb);
    double* partial = (double*)(work + 10 * vb + 256);
    const int64_t len = (int64_t)h->nvar * h->n;
    cudaStream_t st = h->stream;
    int64_t nb = (len + DP5_THREADS - 1) / DP5_THREADS;
    const unsigned grid = (unsigned)(nb > DP5_MAXBLOCKS ? DP5_MAXBLOCKS : nb);
    Dp5Ctrl c;
    memset(&c, 0, sizeof(c));
    c.t = h->t; c.h = h0; c.t_end = t_end; c.rtol = rtol; c.atol = atol; c.max_attempts = max_attempts;
    OSC_CUDA(h, cudaMemcpyAsync(d_c, &c, sizeof(c), cudaMemcpyHostToDevice, st));
    int32_t rc;
    if ((rc = state_to_external(h, v.y))) return rc;              // y (caller layout [nvar][n]) <- the net's state
    if ((rc = rhs_at(h, v.y, v.k[0]))) return rc;                 // k1 = f(y)
    while (true) {
        for (int a = 0; a < DP5_BATCH; ++a) {
            dp5_begin_kernel<<<1, 1, 0, st>>>(d_c);
            for (int s = 1; s < 7; ++s) {
                dp5_stage_kernel<T><<<grid, DP5_THREADS, 0, st>>>(d_c, v, s, len);
                if ((rc = rhs_at(h, s == 6 ? v.y5 : v.tmp, v.k[s]))) return rc;
            }
            dp5_error_kernel<T><<<grid, DP5_THREADS, 0, st>>>(d_c, v, len, partial);
            dp5_commit_kernel<T><<<grid, DP5_THREADS, 0, st>>>(d_c, v, len);
            dp5_end_kernel<<<1, 1, 0, st>>>(d_c);
            h->launches += 10;
        }
        OSC_CUDA(h, cudaGetLastError());
        OSC_CUDA(h, cudaMemcpyAsync(&c, d_c, sizeof(c), cudaMemcpyDeviceToHost, st));
        OSC_CUDA(h, cudaStreamSynchronize(st));
        if (c.done) break;
    }
    if ((rc = state_from_external(h, v.y))) return rc;            // the net's state <- y
    h->t = c.t;
    h->step += c.accepted;
    out5[0] = (double)c.accepted; out5[1] = (double)c.rejected; out5[2] = c.h_used; out5[3] = c.h; out5[4] = c.t;
    if (c.done == 2) return set_err(h, NET_ERR_INVALID, "net_integrate_adaptive: max_attempts (%lld) exhausted at t = %.17g", (long long)max_attempts, c.t);
    return NET_OK;
}

int32_t adaptive_integrate(net* h, double t_end, double rtol, double atol, double h0, int64_t max_attempts,
                           void* d_work, size_t work_bytes, double* out5) {
    if (!(h0 > 0.0) || !(rtol >= 0.0) || !(atol >= 0.0) || !(rtol + atol > 0.0) || !(t_end >= h->t) || max_attempts < 1)
        return set_err(h, NET_ERR_INVALID, "net_integrate_adaptive: need h0 > 0, rtol, atol >= 0 (not both 0), t_end >= t, max_attempts >= 1");
    if (!d_work || ((uintptr_t)d_work & 255) != 0 || work_bytes < adaptive_workspace_bytes(h))
        return set_err(h, NET_ERR_SIZE, "net_integrate_adaptive: work buffer missing, misaligned or smaller than net_adaptive_workspace_bytes");
    if (t_end == h->t) { out5[0] = out5[1] = out5[2] = 0.0; out5[3] = h0; out5[4] = h->t; return NET_OK; }
    return h->desc.dtype == NET_F32 ? dp5_run<float>(h, t_end, rtol, atol, h0, max_attempts, (char*)d_work, out5)
                                    : dp5_run<double>(h, t_end, rtol, atol, h0, max_attempts, (char*)d_work, out5);
}

}  // namespace oscnet
