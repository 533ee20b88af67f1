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

// ---- L2 -> SM delivery rate (the binding resource of the hop kernels is claimed to be this path: measure it) -------------
// A buffer that fits the L2 (default 64 MB of the 126 MB) is read many times by all SMs, (a) with 16-byte LDG that
// bypass L1 (ld.global.cg) into registers, (b) with bulk-asynchronous copies (cp.async.bulk, the TMA engine) into a
// shared-memory ring that nothing consumes, (c) the same LDG kernel over a buffer far larger than L2 (DRAM stream).
__global__ void __launch_bounds__(512) l2_ldg_kernel(const uint4 *buf, long n16, int passes, unsigned *sink)
{
    unsigned acc = 0;
    const long stride = (long)gridDim.x * blockDim.x;
    for (int p = 0; p < passes; p++) {
        long i = (long)blockIdx.x * blockDim.x + threadIdx.x + (long)p * 977 * 32;   // shift the start: no two passes alike per SM
        for (long k = 0; k + 3 * stride < n16; k += 4 * stride) {
            uint4 v[4];
#pragma unroll
            for (int u = 0; u < 4; u++) {
                long j = i + k + u * stride;
                if (j >= n16) j -= n16;
                asm volatile("ld.global.cg.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v[u].x), "=r"(v[u].y), "=r"(v[u].z), "=r"(v[u].w) : "l"(buf + j));
            }
#pragma unroll
            for (int u = 0; u < 4; u++) acc ^= v[u].x ^ v[u].y ^ v[u].z ^ v[u].w;
        }
    }
    if (acc == 0x12345678u) sink[0] = acc;
}
template <int SLAB, int STAGES>
__global__ void __launch_bounds__(32) l2_bulk_kernel(const unsigned char *buf, long nslabs, int passes)
{
    extern __shared__ __align__(128) unsigned char ring[];
    __shared__ unsigned long long bar[STAGES];
    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; s++) {
            unsigned a = (unsigned)__cvta_generic_to_shared(&bar[s]);
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(a) : "memory");
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        const long per = nslabs / gridDim.x;
        const long total = per * passes;
        long issued = 0, done = 0;
        while (done < total) {
            while (issued < total && issued - done < STAGES) {
                const int s = (int)(issued % STAGES);
                const long slab = (long)blockIdx.x * per + ((issued + (issued / per) * 7) % per);
                unsigned b = (unsigned)__cvta_generic_to_shared(&bar[s]);
                unsigned d = (unsigned)__cvta_generic_to_shared(ring + (size_t)s * SLAB);
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%1], %0;" ::"r"((unsigned)SLAB), "r"(b) : "memory");
                asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(d),
                             "l"(buf + slab * SLAB), "r"((unsigned)SLAB), "r"(b)
                             : "memory");
                issued++;
            }
            const int s = (int)(done % STAGES);
            const unsigned phase = (unsigned)((done / STAGES) & 1);
            unsigned b = (unsigned)__cvta_generic_to_shared(&bar[s]), ok = 0;
            while (!ok)
                asm volatile("{\n\t.reg .pred P1;\n\tmbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2;\n\tselp.u32 %0, 1, 0, P1;\n\t}"
                             : "=r"(ok) : "r"(b), "r"(phase) : "memory");
            done++;
        }
    }
}
// out[0] LDG.cg from L2, out[1] bulk copies from L2 (2 CTAs/SM x 6 stages x 16 KB), out[2] LDG.cg DRAM stream, out[3] bulk
// copies DRAM stream; GB/s, best of 3
int mdwf_measure_l2_rates(double *out, cudaStream_t st)
{
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return (int)e;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const size_t small = (size_t)64 << 20, big = (size_t)4 << 30;
    unsigned char *buf = nullptr;
    unsigned *sink = nullptr;
    e = cudaMalloc((void **)&buf, big);
    if (e != cudaSuccess) return (int)e;
    cudaMalloc((void **)&sink, 16);
    cudaMemsetAsync(buf, 1, big, st);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    constexpr int SLAB = 16384, STAGES = 6;
    cudaFuncSetAttribute(l2_bulk_kernel<SLAB, STAGES>, cudaFuncAttributeMaxDynamicSharedMemorySize, SLAB * STAGES);
    for (int mode = 0; mode < 4; mode++) {
        const size_t bytes = (mode < 2) ? small : big;
        const int passes = (mode < 2) ? 40 : 1;
        float best = 1e30f;
        double moved = 0;
        for (int rep = 0; rep < 4; rep++) {          // rep 0 warms the L2
            cudaEventRecord(e0, st);
            if ((mode & 1) == 0) {
                const long n16 = (long)(bytes / 16);
                l2_ldg_kernel<<<sms * 4, 512, 0, st>>>(reinterpret_cast<const uint4 *>(buf), n16, passes, sink);
                const long stride = (long)sms * 4 * 512;
                long iters = 0;
                for (long k = 0; k + 3 * stride < n16; k += 4 * stride) iters++;
                moved = (double)iters * 4 * stride * 16 * passes;
            } else {
                const long nslabs = (long)(bytes / SLAB);
                const int grid = sms * 2;
                l2_bulk_kernel<SLAB, STAGES><<<grid, 32, SLAB * STAGES, st>>>(buf, nslabs, passes);
                moved = (double)(nslabs / grid) * grid * SLAB * passes;
            }
            cudaEventRecord(e1, st);
            cudaEventSynchronize(e1);
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms < best) best = ms;
        }
        out[mode] = moved / (best * 1e-3) / 1e9;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(buf);
    cudaFree(sink);
    return (int)cudaGetLastError();
}
