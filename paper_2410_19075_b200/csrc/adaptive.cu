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
#include <stdlib.h>

#include "oscnet_internal.cuh"

namespace oscnet {

namespace {

constexpr int DP5_BATCH = 8;         // attempts per host read-back
constexpr int DP5_THREADS = 256;
constexpr int DP5_MAXBLOCKS = 1184;

struct Dp5Ctrl {
    double t, h, t_end, rtol, atol, err, h_used, t_prev;
    long long accepted, rejected, attempts, max_attempts, next_out;
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
// continuous extension CONTD5 of the paper's reference [22] (dense output)
__constant__ double DP5_D[7] = {-12715105075.0 / 11282082432.0, 0.0, 87487479700.0 / 32700410799.0,
                                -10690763975.0 / 1880347072.0, 701980252875.0 / 199316789632.0,
                                -1453857185.0 / 822651844.0, 69997945.0 / 29380423.0};
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
            c->t_prev = c->t;
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

// Dense output (runs between the decision and the commit of an accepted step): every requested time
// in (t_prev, t] gets the CONTD5 interpolant
//   y(t_prev + theta h) = r1 + theta (r2 + (1 - theta)(r3 + theta (r4 + (1 - theta) r5))),
//   r1 = y, r2 = y5 - y, r3 = h k1 - r2, r4 = r2 - h k7 - r3, r5 = h sum_j d_j k_j.
// All blocks walk the same list of pending times (read-only here); dp5_end_kernel advances next_out.
template <class T>
__global__ void __launch_bounds__(DP5_THREADS) dp5_dense_kernel(const Dp5Ctrl* c, Dp5Vecs v, int64_t len,
                                                                const double* __restrict__ t_out, long long n_out, T* out) {
    if (c->done || !c->accept) return;
    const double h = c->h_used, t0 = c->t_prev, t1 = c->t;
    for (long long o = c->next_out; o < n_out && t_out[o] <= t1; ++o) {
        const double th = (c->last && o == n_out - 1) ? 1.0 : (t_out[o] - t0) / h, th1 = 1.0 - th;
        T* dst = out + o * len;
        for (int64_t q = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; q < len; q += (int64_t)gridDim.x * blockDim.x) {
            const double y = (double)((const T*)v.y)[q], y5 = (double)((const T*)v.y5)[q];
            const double k1 = (double)((const T*)v.k[0])[q], k7 = (double)((const T*)v.k[6])[q];
            const double r2 = y5 - y, r3 = h * k1 - r2, r4 = r2 - h * k7 - r3;
            double r5 = 0.0;
#pragma unroll
            for (int j = 0; j < 7; ++j) r5 += DP5_D[j] * (double)((const T*)v.k[j])[q];
            r5 *= h;
            dst[q] = (T)(y + th * (r2 + th1 * (r3 + th * (r4 + th1 * r5))));
        }
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
__global__ void dp5_end_kernel(Dp5Ctrl* c, const double* __restrict__ t_out, long long n_out) {
    if (c->done) return;
    if (c->accept) {
        long long o = c->next_out;
        while (o < n_out && t_out[o] <= c->t) ++o;      // the outputs dp5_dense_kernel has just written
        c->next_out = o;
        if (!(c->t < c->t_end)) c->done = 1;
    }
    c->accept = 0;
}

size_t dp5_vec_bytes(const net* h) { return (size_t)round_up((int64_t)h->nvar * h->n * h->esize, 256); }

}  // namespace

size_t adaptive_workspace_bytes(const net* h) {
    return 10 * dp5_vec_bytes(h) + 256 + sizeof(double) * DP5_MAXBLOCKS + 256;
}

// t_out (device, ascending, n_out >= 0 entries, the last one = t_end) / d_out: dense output, or null
template <class T>
static int32_t dp5_run(net* h, double t_end, double rtol, double atol, double h0, int64_t max_attempts,
                       char* work, double* out5, const double* d_t_out, long long n_out, void* d_out) {
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
    // One batch of DP5_BATCH attempts.  Every kernel takes the step size, the time and the decision
    // from the device control block, so a batch is the same work whatever the state: it is captured
    // once into a CUDA graph and replayed (about 50 launches and 24 copies per attempt would
    // otherwise be bound by the host's launch rate: 0.41 ms against 0.35 ms per attempt on 10^6
    // elements).  The legacy default stream cannot be captured: plain launches there.
    auto enqueue_batch = [&]() -> int32_t {
        for (int a = 0; a < DP5_BATCH; ++a) {
            dp5_begin_kernel<<<1, 1, 0, st>>>(d_c);
            for (int s = 1; s < 7; ++s) {
                dp5_stage_kernel<T><<<grid, DP5_THREADS, 0, st>>>(d_c, v, s, len);
                int32_t r = rhs_at(h, s == 6 ? v.y5 : v.tmp, v.k[s]);
                if (r) return r;
            }
            dp5_error_kernel<T><<<grid, DP5_THREADS, 0, st>>>(d_c, v, len, partial);
            if (n_out > 0) dp5_dense_kernel<T><<<grid, DP5_THREADS, 0, st>>>(d_c, v, len, d_t_out, n_out, (T*)d_out);
            dp5_commit_kernel<T><<<grid, DP5_THREADS, 0, st>>>(d_c, v, len);
            dp5_end_kernel<<<1, 1, 0, st>>>(d_c, d_t_out, n_out);
            h->launches += n_out > 0 ? 11 : 10;
        }
        return NET_OK;
    };
    struct GraphHolder {
        cudaGraph_t g = nullptr;
        cudaGraphExec_t e = nullptr;
        ~GraphHolder() { if (e) cudaGraphExecDestroy(e); if (g) cudaGraphDestroy(g); }
    } gh;
    int64_t per_batch = 0;
    if (st != nullptr && st != cudaStreamLegacy && !getenv("OSCNET_DP5_NO_GRAPH")) {
        const int64_t before = h->launches;
        OSC_CUDA(h, cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal));
        rc = enqueue_batch();
        const cudaError_t e = cudaStreamEndCapture(st, &gh.g);
        per_batch = h->launches - before;
        h->launches = before;                      // the capture itself launched nothing
        if (rc) return rc;
        if (e != cudaSuccess) return cuda_err(h, e, "cudaStreamEndCapture(dp5)");
        OSC_CUDA(h, cudaGraphInstantiate(&gh.e, gh.g, 0));
    }
    while (true) {
        if (gh.e) {
            OSC_CUDA(h, cudaGraphLaunch(gh.e, st));
            h->launches += per_batch;
        } else if ((rc = enqueue_batch())) return rc;
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
    return h->desc.dtype == NET_F32 ? dp5_run<float>(h, t_end, rtol, atol, h0, max_attempts, (char*)d_work, out5, nullptr, 0, nullptr)
                                    : dp5_run<double>(h, t_end, rtol, atol, h0, max_attempts, (char*)d_work, out5, nullptr, 0, nullptr);
}

// Dense output: the states at the ascending host times t_out[0 .. n_out) (the last one ends the run)
// go to d_out [n_out][nvar][n] (device, dtype of the net).  The times travel to the tail of the work
// buffer; the steps are those of adaptive_integrate (outputs never shorten a step).
int32_t adaptive_integrate_dense(net* h, int64_t n_out, const double* t_out, void* d_out, double rtol, double atol, double h0,
                                 int64_t max_attempts, void* d_work, size_t work_bytes, double* out5) {
    if (n_out < 1 || !t_out || !d_out) return set_err(h, NET_ERR_INVALID, "net_integrate_adaptive_dense: need n_out >= 1, t_out and d_out");
    if (!(t_out[0] > h->t)) return set_err(h, NET_ERR_INVALID, "net_integrate_adaptive_dense: t_out[0] must lie after the net's time");
    for (int64_t q = 1; q < n_out; ++q)
        if (!(t_out[q] > t_out[q - 1])) return set_err(h, NET_ERR_INVALID, "net_integrate_adaptive_dense: t_out must ascend strictly");
    if (!(h0 > 0.0) || !(rtol >= 0.0) || !(atol >= 0.0) || !(rtol + atol > 0.0) || max_attempts < 1)
        return set_err(h, NET_ERR_INVALID, "net_integrate_adaptive_dense: need h0 > 0, rtol, atol >= 0 (not both 0), max_attempts >= 1");
    const size_t need = adaptive_workspace_bytes(h) + (size_t)round_up(n_out * (int64_t)sizeof(double), 256);
    if (!d_work || ((uintptr_t)d_work & 255) != 0 || work_bytes < need)
        return set_err(h, NET_ERR_SIZE, "net_integrate_adaptive_dense: work buffer missing, misaligned or smaller than net_adaptive_workspace_bytes + 8 n_out (rounded up to 256)");
    double* d_t = (double*)((char*)d_work + adaptive_workspace_bytes(h));
    OSC_CUDA(h, cudaMemcpyAsync(d_t, t_out, sizeof(double) * n_out, cudaMemcpyHostToDevice, h->stream));
    OSC_CUDA(h, cudaStreamSynchronize(h->stream));     // t_out is the caller's (pageable) memory
    const double t_end = t_out[n_out - 1];
    return h->desc.dtype == NET_F32 ? dp5_run<float>(h, t_end, rtol, atol, h0, max_attempts, (char*)d_work, out5, d_t, n_out, d_out)
                                    : dp5_run<double>(h, t_end, rtol, atol, h0, max_attempts, (char*)d_work, out5, d_t, n_out, d_out);
}

}  // namespace oscnet
