// sdense_mma.cu -- S3 as a dense contraction on the tensor cores: out = M in along s, M = the dense real L5 x L5 matrix
// A^{-1} (one per chirality), in fp64 with the double-precision MMA (mma.sync.m8n8k4.f64, SASS DMMA), which is exact to
// fp64 rounding like the FMA form it replaces.  This is the standalone kernel of source preparation and solution
// reconstruction (S10: x_e = A^{-1}(b_e - D_eo x_o), twice per solve); inside the CG the contraction is the blocked
// recurrence of hop3_kernels.cuh and needs no dense product.
//
// GEMM view per 32-site group g and chunk j (fp64 layout: chunk = one complex, NV = 12; j < 6 upper spins -> M+,
// j >= 6 lower spins -> M-):   D[s][col] = sum_s' M[s][s'] B[s'][col],  col = 2 lane' + {re, im}, 64 columns.
// One warp per group; M padded to 16 x 16 (2 m-blocks x up to 4 k-blocks of the 8 x 4 A fragment, held in registers
// for both chiralities), 8 n-blocks of 8 columns per chunk.  Fragment layouts of m8n8k4 (PTX ISA): A[row = lane/4]
// [k = lane%4]; B[k = lane%4][n = lane/4]; C[row = lane/4][n = 2 (lane%4) + {0,1}] -- the two C values of a thread
// are the (re, im) of one site, i.e. one double2 store.
#include "mdwf_device.cuh"
#include "mdwf_internal.h"

__device__ __forceinline__ void dmma_m8n8k4(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

template <int KB>   // KB = ceil(L5 / 4) k-blocks, L5 <= 16
__global__ void __launch_bounds__(128) sdense_mma_kernel(int L5, long Vh, const double2 *__restrict__ in, double2 *__restrict__ out,
                                                         const double *__restrict__ M)
{
    const int lane = threadIdx.x & 31;
    const long g = (long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);      // one warp per 32-site group
    if (g * 32 >= Vh) return;
    const int r4 = lane >> 2, c4 = lane & 3;
    // A fragments of both chiralities: a[ch][mb][kb] = M_ch[8 mb + lane/4][4 kb + lane%4] (zero padding)
    double a[2][2][KB];
#pragma unroll
    for (int ch = 0; ch < 2; ch++)
#pragma unroll
        for (int mb = 0; mb < 2; mb++)
#pragma unroll
            for (int kb = 0; kb < KB; kb++) {
                const int row = 8 * mb + r4, k = 4 * kb + c4;
                a[ch][mb][kb] = (row < L5 && k < L5) ? M[(size_t)ch * L5 * L5 + row * L5 + k] : 0.0;
            }
    const double2 *gin = in + (size_t)g * L5 * 12 * 32;
    double2 *gout = out + (size_t)g * L5 * 12 * 32;
    for (int j = 0; j < 12; j++) {
        const int ch = j < 6 ? 0 : 1;
#pragma unroll 2
        for (int nb = 0; nb < 8; nb++) {
            // B fragment: s' = 4 kb + lane%4, column 8 nb + lane/4 -> site lane' = 4 nb + lane/8, component (lane/4)&1
            double b[KB];
#pragma unroll
            for (int kb = 0; kb < KB; kb++) {
                const int sp = 4 * kb + c4;
                double v = 0.0;
                if (sp < L5) {
                    const double2 q = gin[((size_t)sp * 12 + j) * 32 + 4 * nb + (lane >> 3)];
                    v = (r4 & 1) ? q.y : q.x;
                }
                b[kb] = v;
            }
#pragma unroll
            for (int mb = 0; mb < 2; mb++) {
                double d0 = 0.0, d1 = 0.0;
#pragma unroll
                for (int kb = 0; kb < KB; kb++) dmma_m8n8k4(d0, d1, a[ch][mb][kb], b[kb]);
                const int row = 8 * mb + r4;
                const long site = g * 32 + 4 * nb + c4;
                if (row < L5 && site < Vh) gout[((size_t)row * 12 + j) * 32 + 4 * nb + c4] = make_double2(d0, d1);
            }
        }
    }
}

// out = M in for fp64 parity vectors, M = double[2][L5][L5] on the device.  Returns -1 if L5 > 16 (caller uses the FMA kernel).
int mdwf_launch_sdense_mma(int L5, int Vh, const SpinorBuf &in, const SpinorBuf &out, const void *dense, cudaStream_t st)
{
    if (L5 > 16) return -1;
    const int groups = (Vh + 31) / 32, wpb = 4;
    const unsigned nb = (unsigned)((groups + wpb - 1) / wpb);
    const double2 *i2 = (const double2 *)in.v;
    double2 *o2 = (double2 *)out.v;
    const double *M = (const double *)dense;
    switch ((L5 + 3) / 4) {
    case 1: sdense_mma_kernel<1><<<nb, 32 * wpb, 0, st>>>(L5, Vh, i2, o2, M); break;
    case 2: sdense_mma_kernel<2><<<nb, 32 * wpb, 0, st>>>(L5, Vh, i2, o2, M); break;
    case 3: sdense_mma_kernel<3><<<nb, 32 * wpb, 0, st>>>(L5, Vh, i2, o2, M); break;
    default: sdense_mma_kernel<4><<<nb, 32 * wpb, 0, st>>>(L5, Vh, i2, o2, M); break;
    }
    return (int)cudaGetLastError();
}
