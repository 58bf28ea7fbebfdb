// net_order_parameter_noalloc: the global Kuramoto order parameter R e^{i Psi} = (1/N) sum_j e^{i theta_j}
// (reading R9; the paper's "synchronization analysis at each output") for
// callers that may not allocate: code under CUDA graph capture, tight serving loops, harnesses that
// forbid cudaMalloc.  The existing path (net_observables(NET_OBS_GLOBAL_ORDER): reduce_partial_kernel
// + reduce_finish_kernel in observables.cu) keeps its block partials in the net's workspace; this
// variant keeps them in a file-scope device array that every GPU loading the library holds until exit.
//
//   * maximum NOALLOC_MAX_N = 2^27 phases per call (larger n: NET_ERR_SIZE, nothing launched);
//   * the array is NOALLOC_SCRATCH_BYTES = 256 B + 16 B per NOALLOC_CHUNK phases of the maximum
//     = 262400 bytes per device;
//   * ONE array per device, shared by every call: calls that overlap on the GPU (two streams, two
//     host threads, two captured graphs replayed concurrently) race on it.  Serialise them.
//   * no cudaMalloc, cudaFree or allocating library routine: one cudaMemsetAsync of the 256-byte
//     header (the ticket of the last-block-done protocol must start at zero; the partials are all
//     rewritten before they are read) and one kernel, both on the caller's stream.
//
// Host code cannot use the array's name as a device address: the name is a host-side stand-in.  The
// device address comes from cudaGetSymbolAddress, once per device, with that device current.
#include <mutex>

#include "oscnet_internal.cuh"

namespace {

constexpr int64_t NOALLOC_MAX_N = 1LL << 27;
constexpr int NOALLOC_THREADS = 256;
constexpr int NOALLOC_PER_THREAD = 32;
constexpr int64_t NOALLOC_CHUNK = (int64_t)NOALLOC_THREADS * NOALLOC_PER_THREAD;   // phases per CTA
constexpr int64_t NOALLOC_MAX_BLOCKS = NOALLOC_MAX_N / NOALLOC_CHUNK;              // 16384
constexpr size_t NOALLOC_HEADER = 256;                                             // ticket, padded
constexpr size_t NOALLOC_SCRATCH_BYTES = NOALLOC_HEADER + (size_t)NOALLOC_MAX_BLOCKS * 2 * sizeof(double);
constexpr int NOALLOC_MAX_DEVICES = 64;

static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_SCRATCH_BYTES];

std::mutex g_mu;
unsigned char* g_addr[NOALLOC_MAX_DEVICES];   // device address of g_noalloc_scratch on device d (nullptr: not asked yet)

__device__ __forceinline__ double noalloc_block_sum(double v, double* sh) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) sh[w] = v;
    __syncthreads();
    double r = 0;
    if (threadIdx.x == 0)
        for (int q = 0; q < NOALLOC_THREADS / 32; ++q) r += sh[q];
    __syncthreads();
    return r;   // valid in thread 0
}

// CTA b sums (cos, sin) of phases [b*CHUNK, (b+1)*CHUNK) in a fixed order and stores the pair; the
// CTA that takes the last ticket sums the pairs in index order and writes {R, Psi}.  The result does
// not depend on which CTA is last.
template <class T>
__global__ void __launch_bounds__(NOALLOC_THREADS)
order_noalloc_kernel(const T* __restrict__ theta, int64_t n, unsigned char* scratch, double* __restrict__ out2) {
    __shared__ double sh[NOALLOC_THREADS / 32];
    __shared__ bool is_last;
    unsigned* ticket = reinterpret_cast<unsigned*>(scratch);
    double* partial = reinterpret_cast<double*>(scratch + NOALLOC_HEADER);
    const int64_t base = (int64_t)blockIdx.x * NOALLOC_CHUNK;
    double a = 0, b = 0;
#pragma unroll 4
    for (int k = 0; k < NOALLOC_PER_THREAD; ++k) {
        const int64_t i = base + threadIdx.x + (int64_t)k * NOALLOC_THREADS;
        if (i < n) {
            double s, c;
            sincos((double)theta[i], &s, &c);
            a += c;
            b += s;
        }
    }
    const double ra = noalloc_block_sum(a, sh);
    const double rb = noalloc_block_sum(b, sh);
    if (threadIdx.x == 0) {
        partial[2 * blockIdx.x] = ra;
        partial[2 * blockIdx.x + 1] = rb;
        __threadfence();
        is_last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    a = 0; b = 0;
    for (unsigned q = threadIdx.x; q < gridDim.x; q += NOALLOC_THREADS) {
        a += __ldcg(partial + 2 * q);
        b += __ldcg(partial + 2 * q + 1);
    }
    const double ta = noalloc_block_sum(a, sh);
    const double tb = noalloc_block_sum(b, sh);
    if (threadIdx.x == 0) {
        const double c = ta / (double)n, s = tb / (double)n;
        out2[0] = sqrt(c * c + s * s);
        out2[1] = atan2(s, c);
        *ticket = 0;
    }
}

// Device address of the scratch array on the CURRENT device (asked once per device).
int32_t scratch_address(unsigned char** out) {
    int dev = -1;
    OSC_CUDA(nullptr, cudaGetDevice(&dev));
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES)
        return oscnet::set_err(nullptr, NET_ERR_UNSUPPORTED, "net_order_parameter_noalloc: device ordinal %d >= %d", dev, NOALLOC_MAX_DEVICES);
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_addr[dev]) {
        void* p = nullptr;
        OSC_CUDA(nullptr, cudaGetSymbolAddress(&p, g_noalloc_scratch));
        if (!p) return oscnet::set_err(nullptr, NET_ERR_CUDA, "net_order_parameter_noalloc: cudaGetSymbolAddress gave NULL on device %d", dev);
        g_addr[dev] = static_cast<unsigned char*>(p);
    }
    *out = g_addr[dev];
    return NET_OK;
}

}  // namespace

#pragma GCC visibility push(default)
extern "C" {

int32_t net_order_parameter_noalloc(const void* d_theta, int64_t n, int32_t dtype, double* d_out2, void* stream) {
    using oscnet::set_err;
    if (!d_theta || !d_out2) return set_err(nullptr, NET_ERR_INVALID, "net_order_parameter_noalloc: NULL pointer");
    if (dtype != NET_F32 && dtype != NET_F64) return set_err(nullptr, NET_ERR_INVALID, "net_order_parameter_noalloc: unknown dtype %d", dtype);
    if (n < 1) return set_err(nullptr, NET_ERR_INVALID, "net_order_parameter_noalloc: n = %lld < 1", (long long)n);
    if (n > NOALLOC_MAX_N)
        return set_err(nullptr, NET_ERR_SIZE, "net_order_parameter_noalloc: n = %lld exceeds the maximum %lld of the static scratch array (%zu bytes per device)",
                       (long long)n, (long long)NOALLOC_MAX_N, NOALLOC_SCRATCH_BYTES);
    unsigned char* scratch = nullptr;
    int32_t rc = scratch_address(&scratch);
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    OSC_CUDA(nullptr, cudaMemsetAsync(scratch, 0, NOALLOC_HEADER, st));   // the ticket starts at zero
    const unsigned grid = (unsigned)((n + NOALLOC_CHUNK - 1) / NOALLOC_CHUNK);
    if (dtype == NET_F32)
        order_noalloc_kernel<float><<<grid, NOALLOC_THREADS, 0, st>>>(static_cast<const float*>(d_theta), n, scratch, d_out2);
    else
        order_noalloc_kernel<double><<<grid, NOALLOC_THREADS, 0, st>>>(static_cast<const double*>(d_theta), n, scratch, d_out2);
    OSC_CUDA(nullptr, cudaGetLastError());
    return NET_OK;
}

}  // extern "C"
#pragma GCC visibility pop
