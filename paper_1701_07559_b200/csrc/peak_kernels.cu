// peak_kernels.cu -- live measurement of the fp32 FMA rates the ALU roofline of DESIGN.md section 6 uses:
// a 3-register FFMA stream and the packed FFMA2 (fma.rn.f32x2) stream, 16 independent chains per thread.
#include "mdwf_internal.h"

template <int PACKED>
__global__ void __launch_bounds__(256) fma_peak_kernel(float *out, float a, float b, int iters)
{
    float2 x[8];
#pragma unroll
    for (int i = 0; i < 8; i++) { x[i].x = threadIdx.x * 0.001f + i; x[i].y = threadIdx.x * 0.002f + i; }
    const float2 A = make_float2(a, a * 1.0001f), B = make_float2(b, b * 0.999f);
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 8; i++) {
            if (PACKED) x[i] = __ffma2_rn(x[i], A, B);
            else { x[i].x = fmaf(x[i].x, A.x, B.x); x[i].y = fmaf(x[i].y, A.y, B.y); }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; i++) s += x[i].x + x[i].y;
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// tfma[0] = FFMA, tfma[1] = FFMA2, in 1e12 fused multiply-adds per second (x2 for flop/s)
int mdwf_measure_fma_rates(double *tfma, cudaStream_t st)
{
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return (int)e;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int blocks = sms * 8, iters = 20000;
    float *out = nullptr;
    e = cudaMalloc((void **)&out, sizeof(float) * blocks * 256);
    if (e != cudaSuccess) return (int)e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    for (int mode = 0; mode < 2; mode++) {
        float best = 1e30f;
        for (int rep = 0; rep < 3; rep++) {
            cudaEventRecord(e0, st);
            if (mode == 0) fma_peak_kernel<0><<<blocks, 256, 0, st>>>(out, 1.0001f, 0.0001f, iters);
            else fma_peak_kernel<1><<<blocks, 256, 0, st>>>(out, 1.0001f, 0.0001f, iters);
            cudaEventRecord(e1, st);
            cudaEventSynchronize(e1);
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (ms < best) best = ms;
        }
        tfma[mode] = (double)blocks * 256 * 16.0 * iters / (best * 1e-3) / 1e12;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    return (int)cudaGetLastError();
}
