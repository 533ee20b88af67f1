// s5_kernels.cu -- site-local fifth-dimension operator A^{-1} / A^{-dagger} for fp32 arithmetic (fp32 and 16-bit storage) as a
// first-order recurrence with a rank-one wall term (S3 of the hot path standing alone):
//     A = alpha (1 + kappa T) per chirality  =>  z_e = x_e - kappa z_{e-1},  W = z_{L5-1},  y_e = z_e / alpha + gw (-kappa)^{e+1} W,
//     gw = -m_f / (alpha (1 + m_f (-kappa)^{L5})),
// e = s for the "direct" half (upper spins of A^{-1}, lower spins of A^{-dagger}) and e = L5-1-s for the "mirrored" half.
// Used by the symmetric preconditioning (NEXT-1): Mpc_sym^dagger needs A^{-dagger} on the input of its first hop.
// One thread per 4D site; a half spinor of all L5 slices is held in registers (L5 x 6 complex numbers), so the vector is read
// once and written once for fp32 storage.  16-bit storage needs the largest component of all 24 reals of a (site, s) before it
// can quantise: a first pass finds it, the second recomputes and stores (the reloads hit L1 / L2).
#include "mdwf_device.cuh"
#include "mdwf_internal.h"

namespace {

typedef float2 c2;

template <class P> __device__ __forceinline__ void ld3(const void *base, const float *norm, int L5, int s, long cb, int half, c2 *v);
template <> __device__ __forceinline__ void ld3<PS>(const void *base, const float *, int L5, int s, long cb, int half, c2 *v)
{
    const float4 *p = reinterpret_cast<const float4 *>(base) + sp_off(L5, PS::NV, cb, s) + 32 * 3 * half;
#pragma unroll
    for (int j = 0; j < 3; j++) {
        const float4 q = __ldg(p + 32 * j);
        v[2 * j] = make_float2(q.x, q.y);
        v[2 * j + 1] = make_float2(q.z, q.w);
    }
}
template <> __device__ __forceinline__ void ld3<PH>(const void *base, const float *norm, int L5, int s, long cb, int half, c2 *v)
{
    const short4 *p = reinterpret_cast<const short4 *>(base) + sp_off(L5, PH::NV, cb, s) + 32 * 3 * half;
    const float sc = __ldg(norm + sp_noff(L5, cb, s)) * (1.0f / MDWF_FIXED_MAX);
#pragma unroll
    for (int j = 0; j < 3; j++) {
        const short4 q = __ldg(p + 32 * j);
        v[2 * j] = make_float2(sc * fixed_to_float((unsigned short)q.x), sc * fixed_to_float((unsigned short)q.y));
        v[2 * j + 1] = make_float2(sc * fixed_to_float((unsigned short)q.z), sc * fixed_to_float((unsigned short)q.w));
    }
}

// y = A^{-1} x (dag = 0) or A^{-dagger} x (dag = 1) on one half (0: upper spins, 1: lower spins) of one site, in place in v[s][6]
template <class P, int L5, int half, int DAG>
__device__ __forceinline__ void half_column(const void *in, const float *in_norm, long cb, float nk, float inv_alpha, float gw, c2 (*v)[6])
{
    constexpr bool mirrored = (half == 1) != (DAG != 0);
#pragma unroll
    for (int s = 0; s < L5; s++) ld3<P>(in, in_norm, L5, s, cb, half, v[s]);
#pragma unroll
    for (int e = 1; e < L5; e++) {
        const int s = mirrored ? L5 - 1 - e : e, sp = mirrored ? s + 1 : s - 1;
#pragma unroll
        for (int q = 0; q < 6; q++) { v[s][q].x = fmaf(nk, v[sp][q].x, v[s][q].x); v[s][q].y = fmaf(nk, v[sp][q].y, v[s][q].y); }
    }
    c2 W[6];
#pragma unroll
    for (int q = 0; q < 6; q++) W[q] = v[mirrored ? 0 : L5 - 1][q];
    float pw = nk;                                       // (-kappa)^{e+1}
#pragma unroll
    for (int e = 0; e < L5; e++) {
        const int s = mirrored ? L5 - 1 - e : e;
        const float w = gw * pw;
#pragma unroll
        for (int q = 0; q < 6; q++) { v[s][q].x = fmaf(inv_alpha, v[s][q].x, w * W[q].x); v[s][q].y = fmaf(inv_alpha, v[s][q].y, w * W[q].y); }
        pw *= nk;
    }
}

template <class P, int L5, int DAG>
__global__ void __launch_bounds__(128) srec_kernel(const void *in, const float *in_norm, void *out, float *out_norm, long Vh, float nk,
                                                   float inv_alpha, float gw)
{
    const long cb = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= Vh) return;
    c2 v[L5][6];
    if (!P::HALF) {
#define MDWF_S5_HALF(half)                                                                                             \
        {                                                                                                                  \
            half_column<P, L5, half, DAG>(in, in_norm, cb, nk, inv_alpha, gw, v);                                          \
            _Pragma("unroll") for (int s = 0; s < L5; s++) {                                                               \
                float4 *p = reinterpret_cast<float4 *>(out) + sp_off(L5, PS::NV, cb, s) + 32 * 3 * half;                   \
                _Pragma("unroll") for (int j = 0; j < 3; j++)                                                              \
                    p[32 * j] = make_float4(v[s][2 * j].x, v[s][2 * j].y, v[s][2 * j + 1].x, v[s][2 * j + 1].y);           \
            }                                                                                                              \
        }
        MDWF_S5_HALF(0)
        MDWF_S5_HALF(1)
#undef MDWF_S5_HALF
    } else {
        float m[L5];
#pragma unroll
        for (int s = 0; s < L5; s++) m[s] = 0.f;
#define MDWF_S5_MAX(half)                                                                                              \
        {                                                                                                                  \
            half_column<P, L5, half, DAG>(in, in_norm, cb, nk, inv_alpha, gw, v);                                          \
            _Pragma("unroll") for (int s = 0; s < L5; s++)                                                                 \
                _Pragma("unroll") for (int q = 0; q < 6; q++) m[s] = fmaxf(m[s], fmaxf(fabsf(v[s][q].x), fabsf(v[s][q].y))); \
        }
        MDWF_S5_MAX(0)
        MDWF_S5_MAX(1)
#undef MDWF_S5_MAX
#define MDWF_S5_STORE(half)                                                                                            \
        {                                                                                                                  \
            half_column<P, L5, half, DAG>(in, in_norm, cb, nk, inv_alpha, gw, v);                                          \
            _Pragma("unroll") for (int s = 0; s < L5; s++) {                                                               \
                const float isc = m[s] > 0.f ? MDWF_FIXED_MAX / m[s] : 0.f;                                                \
                short4 *p = reinterpret_cast<short4 *>(out) + sp_off(L5, PH::NV, cb, s) + 32 * 3 * half;                   \
                _Pragma("unroll") for (int j = 0; j < 3; j++)                                                              \
                    p[32 * j] = make_short4(float_to_fixed(v[s][2 * j].x, isc), float_to_fixed(v[s][2 * j].y, isc),        \
                                            float_to_fixed(v[s][2 * j + 1].x, isc), float_to_fixed(v[s][2 * j + 1].y, isc)); \
                if (half == 1) out_norm[sp_noff(L5, cb, s)] = m[s];                                                        \
            }                                                                                                              \
        }
        MDWF_S5_STORE(0)
        MDWF_S5_STORE(1)
#undef MDWF_S5_STORE
    }
}

template <class P>
int launch(int L5, long Vh, const SpinorBuf &in, const SpinorBuf &out, int dag, float nk, float ia, float gw, cudaStream_t st)
{
    const unsigned nb = (unsigned)((Vh + 127) / 128);
#define MDWF_S5_GO(L) do { if (dag) srec_kernel<P, L, 1><<<nb, 128, 0, st>>>(in.v, in.norm, out.v, out.norm, Vh, nk, ia, gw); \
                           else srec_kernel<P, L, 0><<<nb, 128, 0, st>>>(in.v, in.norm, out.v, out.norm, Vh, nk, ia, gw); } while (0)
    if (L5 == 12) MDWF_S5_GO(12);
    else if (L5 == 8) MDWF_S5_GO(8);
    else if (L5 == 16) MDWF_S5_GO(16);
    else return -1;
#undef MDWF_S5_GO
    return (int)cudaGetLastError();
}

}   // namespace

// out = A^{-1} in (dag = 0) or A^{-dagger} in (dag = 1); in != out.  Returns -1 when not covered (fp64, other L5): the caller
// falls back to the dense-table kernel.
int mdwf_launch_srec(Prec p, int L5, int Vh, const SpinorBuf &in, const SpinorBuf &out, int dag, double alpha, double beta, double mf,
                     cudaStream_t st)
{
    if (p == PREC_D || in.v == out.v) return -1;
    const double nk = -beta / alpha;
    double pL = 1.0;
    for (int i = 0; i < L5; i++) pL *= nk;
    const double gw = -mf / (alpha * (1.0 + mf * pL));
    return p == PREC_S ? launch<PS>(L5, Vh, in, out, dag, (float)nk, (float)(1.0 / alpha), (float)gw, st)
                       : launch<PH>(L5, Vh, in, out, dag, (float)nk, (float)(1.0 / alpha), (float)gw, st);
}
