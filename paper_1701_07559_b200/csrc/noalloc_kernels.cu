// noalloc_kernels.cu -- ||x||^2 of a flat device array through an entry point that allocates NOTHING (include/mdwf.h:
// mdwf_blas_norm2_noalloc).  For callers that cannot call cudaMalloc: code under CUDA graph capture, tight serving loops,
// harnesses that forbid it.  Same arithmetic and the same fixed reduction order as mdwf_blas_norm2 (blas_kernels.cu: per-thread
// strided fp64 sums, xor-shuffle tree per warp, tree per block, one partial per block, fixed-order single-block final pass), so
// the two agree bit for bit; what differs is where the per-block partials live:
//
//   mdwf_blas_norm2          partials in a buffer the context obtained from cudaMalloc
//   mdwf_blas_norm2_noalloc  partials in the file-scope device array below: NOALLOC_MAX_BLOCKS doubles = 32 KB, held by every GPU
//                            that loads the library until the process exits
//
// In host code the array's name is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, taken once per device with that device current (noalloc_scratch()).
// Every call shares the array and the array keeps the last call's contents.  Nothing in it has to start at zero: a call with nb
// blocks overwrites partials [0, nb) and its final pass reads exactly those.  Calls that overlap on the GPU (two streams, two host
// threads without ordering between their launches) race on it: the caller serialises them.
#include <cuda_runtime.h>

#include <mutex>

#include "../../include/mdwf.h"

namespace {

constexpr int NA_THREADS = 256;
constexpr int NOALLOC_MAX_BLOCKS = 4096;                    // as RED_MAX_BLOCKS of blas_kernels.cu: same grid, same order
constexpr long long NOALLOC_MAX_N = 1LL << 30;              // reals per call: a partial then sums at most 2^18 terms per thread pass
constexpr int NOALLOC_MAX_DEVICES = 64;

static __device__ __align__(256) double g_noalloc_partial[NOALLOC_MAX_BLOCKS];

thread_local const char *tl_err = "";

__device__ __forceinline__ double na_warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

template <class T>
__global__ void __launch_bounds__(NA_THREADS) noalloc_norm2_kernel(const T *x, long long n, double *partial)
{
    double sum = 0.0;
    for (long long i = (long long)blockIdx.x * NA_THREADS + threadIdx.x; i < n; i += (long long)gridDim.x * NA_THREADS) {
        const double a = (double)x[i];
        sum += a * a;
    }
    __shared__ double wsum[NA_THREADS / 32];
    sum = na_warp_sum(sum);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) wsum[w] = sum;
    __syncthreads();
    if (w == 0) {
        double t = (lane < NA_THREADS / 32) ? wsum[lane] : 0.0;
        t = na_warp_sum(t);
        if (lane == 0) partial[blockIdx.x] = t;
    }
}

__global__ void __launch_bounds__(NA_THREADS) noalloc_final_sum_kernel(const double *partial, int n, double *result)
{
    double v = 0.0;
    for (int i = threadIdx.x; i < n; i += NA_THREADS) v += partial[i];
    __shared__ double wsum[NA_THREADS / 32];
    v = na_warp_sum(v);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) wsum[w] = v;
    __syncthreads();
    if (w == 0) {
        double t = (lane < NA_THREADS / 32) ? wsum[lane] : 0.0;
        t = na_warp_sum(t);
        if (lane == 0) *result = t;
    }
}

// device address of the scratch array on the CURRENT device; taken once per device
int noalloc_scratch(double **out)
{
    static std::mutex mu;
    static double *ptr[NOALLOC_MAX_DEVICES] = {};
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { tl_err = "mdwf_blas_norm2_noalloc: no CUDA device (cudaGetDevice failed)"; return MDWF_ECUDA; }
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) { tl_err = "mdwf_blas_norm2_noalloc: device ordinal beyond 63"; return MDWF_EARG; }
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        double *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void **)&p, g_noalloc_partial);
        if (e != cudaSuccess || !p) {
            tl_err = "mdwf_blas_norm2_noalloc: cudaGetSymbolAddress of the scratch array failed";
            return MDWF_ECUDA;
        }
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return MDWF_OK;
}

}   // namespace

extern "C" int mdwf_noalloc_setup(void)
{
    double *p = nullptr;
    return noalloc_scratch(&p);
}

extern "C" long long mdwf_noalloc_max_n(void) { return NOALLOC_MAX_N; }

extern "C" const char *mdwf_noalloc_last_error(void) { return tl_err; }

extern "C" int mdwf_blas_norm2_noalloc(const void *x_dev, long long n, int real_bytes, double *out_dev, void *stream)
{
    if (n < 0) { tl_err = "mdwf_blas_norm2_noalloc: n < 0"; return MDWF_EARG; }
    if (n > NOALLOC_MAX_N) { tl_err = "mdwf_blas_norm2_noalloc: n exceeds the maximum of 2^30 reals per call (mdwf_noalloc_max_n)"; return MDWF_EARG; }
    if (real_bytes != 8 && real_bytes != 4) { tl_err = "mdwf_blas_norm2_noalloc: real_bytes must be 8 or 4"; return MDWF_EARG; }
    if (!out_dev || (!x_dev && n > 0)) { tl_err = "mdwf_blas_norm2_noalloc: null pointer"; return MDWF_EARG; }
    double *partial = nullptr;
    const int rc = noalloc_scratch(&partial);
    if (rc != MDWF_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    long long b = ((n / 4 + 1) + NA_THREADS - 1) / NA_THREADS;          // the grid of mdwf_blas_norm2 (red_blocks(n / 4 + 1))
    if (b > NOALLOC_MAX_BLOCKS) b = NOALLOC_MAX_BLOCKS;
    if (b < 1) b = 1;
    const int nb = (int)b;
    if (real_bytes == 8) noalloc_norm2_kernel<double><<<nb, NA_THREADS, 0, st>>>((const double *)x_dev, n, partial);
    else noalloc_norm2_kernel<float><<<nb, NA_THREADS, 0, st>>>((const float *)x_dev, n, partial);
    noalloc_final_sum_kernel<<<1, NA_THREADS, 0, st>>>(partial, nb, out_dev);
    if (cudaGetLastError() != cudaSuccess) { tl_err = "mdwf_blas_norm2_noalloc: kernel launch failed"; return MDWF_ECUDA; }
    tl_err = "";
    return MDWF_OK;
}
