// blas_kernels.cu -- deterministic BLAS-1 (S7) on device-layout parity vectors and on flat arrays.
//
// Determinism: every thread accumulates a fixed set of elements in fp64, a warp is reduced with a fixed
// xor-shuffle tree, a block with a fixed tree over its warps, each block writes ONE partial to
// partial[blockIdx.x] and a single-block second kernel adds the partials in a fixed strided order.
// The grid is a pure function of the problem size, so results are bit-reproducible run to run.
// No floating-point atomics anywhere.
#include "mdwf_device.cuh"
#include "mdwf_internal.h"

#define RED_THREADS 256
#define RED_MAX_BLOCKS 4096

int mdwf_reduce_max_blocks() { return RED_MAX_BLOCKS; }

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ void block_partial(double v, double *partial)
{
    __shared__ double wsum[RED_THREADS / 32];
    v = warp_sum(v);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) wsum[w] = v;
    __syncthreads();
    if (w == 0) {
        double t = (lane < RED_THREADS / 32) ? wsum[lane] : 0.0;
        t = warp_sum(t);
        if (lane == 0) partial[blockIdx.y * gridDim.x + blockIdx.x] = t;
    }
}

__global__ void final_sum_kernel(const double *partial, int n, double *result)
{
    double v = 0.0;
    for (int i = threadIdx.x; i < n; i += RED_THREADS) v += partial[i];
    __shared__ double wsum[RED_THREADS / 32];
    v = warp_sum(v);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) wsum[w] = v;
    __syncthreads();
    if (w == 0) {
        double t = (lane < RED_THREADS / 32) ? wsum[lane] : 0.0;
        t = warp_sum(t);
        if (lane == 0) *result = t;
    }
}

int mdwf_launch_final_sum(const double *partial, int n, double *result_dev, cudaStream_t st)
{
    final_sum_kernel<<<1, RED_THREADS, 0, st>>>(partial, n, result_dev);
    return (int)cudaGetLastError();
}

static int red_blocks(long long work)
{
    long long b = (work + RED_THREADS - 1) / RED_THREADS;
    if (b > RED_MAX_BLOCKS) b = RED_MAX_BLOCKS;
    if (b < 1) b = 1;
    return (int)b;
}

// grid of the parity-vector kernels: (nbx, L5) with nbx * L5 <= RED_MAX_BLOCKS partials
static dim3 site_grid(int L5, int Vh)
{
    int nbx = (Vh + RED_THREADS - 1) / RED_THREADS;
    const int cap = RED_MAX_BLOCKS / L5;
    if (nbx > cap) nbx = cap;
    if (nbx < 1) nbx = 1;
    return dim3((unsigned)nbx, (unsigned)L5);
}

// ---- parity vectors: out = a x + b y  (+ ||out||^2) -------------------------------------------
// arithmetic type of a BLAS kernel: fp64 as soon as one operand is stored in fp64, else fp32 (the result is
// rounded to fp32 or 16 bits anyway); reductions always accumulate across sites in fp64
template <class A, class B, class C> struct CompT { using T = float; };
template <class B, class C> struct CompT<PD, B, C> { using T = double; };
template <class C> struct CompT<PS, PD, C> { using T = double; };
template <class C> struct CompT<PH, PD, C> { using T = double; };
template <> struct CompT<PS, PS, PD> { using T = double; };
template <> struct CompT<PS, PH, PD> { using T = double; };
template <> struct CompT<PH, PS, PD> { using T = double; };
template <> struct CompT<PH, PH, PD> { using T = double; };

// CG scalars kept on the device: while a coefficient pointer is set, the (a, b) of mdwf_launch_axpby / xpupdate / xpupdate_b
// are multiplied by coef[0], coef[1] read in the kernel, so that alpha = gamma / ||q||^2 and beta = gamma' / gamma never
// travel to the host ("unless kept on device")
static thread_local const double *tl_coef = nullptr;
void mdwf_blas_set_coef(const double *coef_dev) { tl_coef = coef_dev; }
// S: [1] gamma, [2] ||q||^2, [3] ||r||^2, [4] gamma', [5..6] (alpha, 1) for r -= alpha q, [7..9] (alpha, beta, previous alpha) for the x / p update
__global__ void cg_scalars_kernel(double *S, int mode)
{
    if (mode == 0) { const double al = S[1] / S[2]; S[5] = al; S[6] = 1.0; S[9] = S[7]; S[7] = al; }   // S[9]: alpha of the iteration before
    else { S[8] = S[4] / S[1]; S[1] = S[4]; }
}
int mdwf_launch_cg_scalars(double *S, int mode, cudaStream_t st)
{
    cg_scalars_kernel<<<1, 1, 0, st>>>(S, mode);
    return (int)cudaGetLastError();
}

template <class PO, class PX, class PY, bool HASY, bool NORM>
__global__ void __launch_bounds__(RED_THREADS)
axpby_kernel(void *out, float *out_norm, double a, const void *x, const float *xn, double b, const void *y,
             const float *yn, int L5, long Vh, double *partial, const double *coef)
{
    using RO = typename PO::R;
    if (coef) { a *= coef[0]; b *= coef[1]; }        // CG scalars kept on the device (mdwf_blas_set_coef)
    // grid = (blocks over the sites of one s-slice, L5): no integer division in the loop
    const int s = blockIdx.y;
    double sum = 0.0;
    for (long cb = (long)blockIdx.x * RED_THREADS + threadIdx.x; cb < Vh; cb += (long)gridDim.x * RED_THREADS) {
        typename PX::R vx[24];
        load_spinor<PX>(x, xn, L5, s, cb, vx);
        using T = typename CompT<PO, PX, PY>::T;
        const T ta = (T)a, tb = (T)b;
        RO r[24];
        if (HASY) {
            typename PY::R vy[24];
            load_spinor<PY>(y, yn, L5, s, cb, vy);
#pragma unroll
            for (int k = 0; k < 24; k++) r[k] = (RO)(ta * (T)vx[k] + tb * (T)vy[k]);
        } else {
#pragma unroll
            for (int k = 0; k < 24; k++) r[k] = (RO)(ta * (T)vx[k]);
        }
        store_spinor<PO>(out, out_norm, L5, s, cb, r);
        if (NORM) {
            T part = 0;
#pragma unroll
            for (int k = 0; k < 24; k++) part += (T)r[k] * (T)r[k];
            sum += (double)part;
        }
    }
    if (NORM) block_partial(sum, partial);
}

template <class PX, class PY, int KIND>
__global__ void __launch_bounds__(RED_THREADS)
reduce_kernel(const void *x, const float *xn, const void *y, const float *yn, int L5, long Vh, double *partial)
{
    // grid = (blocks over the sites of one s-slice, L5): no integer division in the loop
    const int s = blockIdx.y;
    double sum = 0.0;
    for (long cb = (long)blockIdx.x * RED_THREADS + threadIdx.x; cb < Vh; cb += (long)gridDim.x * RED_THREADS) {
        typename PX::R vx[24];
        load_spinor<PX>(x, xn, L5, s, cb, vx);
        using T = typename CompT<PX, PY, PY>::T;
        T part = 0;
        if (KIND == 0) {
#pragma unroll
            for (int k = 0; k < 24; k++) part += (T)vx[k] * (T)vx[k];
        } else {
            typename PY::R vy[24];
            load_spinor<PY>(y, yn, L5, s, cb, vy);
#pragma unroll
            for (int k = 0; k < 24; k++) part += (T)vx[k] * (T)vy[k];
        }
        sum += (double)part;
    }
    block_partial(sum, partial);
}

template <class PO, class PX, class PY>
static int axpby_xy(const SpinorBuf &out, double a, const SpinorBuf &x, double b, const SpinorBuf &y, int L5, int Vh,
                    double *partial, double *result, cudaStream_t st)
{
    const dim3 nb = site_grid(L5, Vh);
    const bool hasy = (y.v != nullptr);
    const bool norm = (partial != nullptr);
#define AX(HY, NM) axpby_kernel<PO, PX, PY, HY, NM><<<nb, RED_THREADS, 0, st>>>(out.v, out.norm, a, x.v, x.norm, b, y.v, y.norm, L5, Vh, partial, tl_coef)
    if (hasy && norm) AX(true, true);
    else if (hasy) AX(true, false);
    else if (norm) AX(false, true);
    else AX(false, false);
#undef AX
    if (norm) final_sum_kernel<<<1, RED_THREADS, 0, st>>>(partial, (int)(nb.x * nb.y), result);
    return (int)cudaGetLastError();
}

template <class PO, class PX>
static int axpby_y(Prec py, const SpinorBuf &out, double a, const SpinorBuf &x, double b, const SpinorBuf &y, int L5,
                   int Vh, double *partial, double *result, cudaStream_t st)
{
    switch (py) {
    case PREC_D: return axpby_xy<PO, PX, PD>(out, a, x, b, y, L5, Vh, partial, result, st);
    case PREC_S: return axpby_xy<PO, PX, PS>(out, a, x, b, y, L5, Vh, partial, result, st);
    default: return axpby_xy<PO, PX, PH>(out, a, x, b, y, L5, Vh, partial, result, st);
    }
}
template <class PO>
static int axpby_x(Prec px, Prec py, const SpinorBuf &out, double a, const SpinorBuf &x, double b, const SpinorBuf &y,
                   int L5, int Vh, double *partial, double *result, cudaStream_t st)
{
    switch (px) {
    case PREC_D: return axpby_y<PO, PD>(py, out, a, x, b, y, L5, Vh, partial, result, st);
    case PREC_S: return axpby_y<PO, PS>(py, out, a, x, b, y, L5, Vh, partial, result, st);
    default: return axpby_y<PO, PH>(py, out, a, x, b, y, L5, Vh, partial, result, st);
    }
}

int mdwf_launch_axpby(Prec po, const SpinorBuf &out, double a, Prec px, const SpinorBuf &x, double b, Prec py,
                      const SpinorBuf &y, int L5, int Vh, double *partial, double *result_dev, cudaStream_t st)
{
    switch (po) {
    case PREC_D: return axpby_x<PD>(px, py, out, a, x, b, y, L5, Vh, partial, result_dev, st);
    case PREC_S: return axpby_x<PS>(px, py, out, a, x, b, y, L5, Vh, partial, result_dev, st);
    default: return axpby_x<PH>(px, py, out, a, x, b, y, L5, Vh, partial, result_dev, st);
    }
}

template <class PX, class PY>
static int reduce_xy(int kind, const SpinorBuf &x, const SpinorBuf &y, int L5, int Vh, double *partial,
                     double *result, cudaStream_t st)
{
    const dim3 nb = site_grid(L5, Vh);
    if (kind == 0)
        reduce_kernel<PX, PY, 0><<<nb, RED_THREADS, 0, st>>>(x.v, x.norm, y.v, y.norm, L5, Vh, partial);
    else
        reduce_kernel<PX, PY, 1><<<nb, RED_THREADS, 0, st>>>(x.v, x.norm, y.v, y.norm, L5, Vh, partial);
    final_sum_kernel<<<1, RED_THREADS, 0, st>>>(partial, (int)(nb.x * nb.y), result);
    return (int)cudaGetLastError();
}
template <class PX>
static int reduce_y(int kind, Prec py, const SpinorBuf &x, const SpinorBuf &y, int L5, int Vh, double *partial,
                    double *result, cudaStream_t st)
{
    switch (py) {
    case PREC_D: return reduce_xy<PX, PD>(kind, x, y, L5, Vh, partial, result, st);
    case PREC_S: return reduce_xy<PX, PS>(kind, x, y, L5, Vh, partial, result, st);
    default: return reduce_xy<PX, PH>(kind, x, y, L5, Vh, partial, result, st);
    }
}
int mdwf_launch_reduce(int kind, Prec px, const SpinorBuf &x, Prec py, const SpinorBuf &y, int L5, int Vh,
                       double *partial, double *result_dev, cudaStream_t st)
{
    switch (px) {
    case PREC_D: return reduce_y<PD>(kind, py, x, y, L5, Vh, partial, result_dev, st);
    case PREC_S: return reduce_y<PS>(kind, py, x, y, L5, Vh, partial, result_dev, st);
    default: return reduce_y<PH>(kind, py, x, y, L5, Vh, partial, result_dev, st);
    }
}

// ---- fused CG update: x += a p ; p = g + b p  (one read of p instead of two) --------------------------
template <class PX, class PP>
__global__ void __launch_bounds__(RED_THREADS)
xpupdate_kernel(void *x, float *xn, double a, void *p, float *pn, double b, const void *g, const float *gn, int L5, long Vh,
                const double *coef)
{
    if (coef) { a *= coef[0]; b *= coef[1]; }
    const int s = blockIdx.y;
    for (long cb = (long)blockIdx.x * RED_THREADS + threadIdx.x; cb < Vh; cb += (long)gridDim.x * RED_THREADS) {
        typename PP::R vp[24], vg[24];
        typename PX::R vx[24];
        load_spinor<PP>(p, pn, L5, s, cb, vp);
        load_spinor<PP>(g, gn, L5, s, cb, vg);
        load_spinor<PX>(x, xn, L5, s, cb, vx);
        using T = typename CompT<PX, PP, PP>::T;
        const T ta = (T)a, tb = (T)b;
#pragma unroll
        for (int k = 0; k < 24; k++) {
            vx[k] = (typename PX::R)((T)vx[k] + ta * (T)vp[k]);
            vp[k] = (typename PP::R)((T)vg[k] + tb * (T)vp[k]);
        }
        store_spinor<PX>(x, xn, L5, s, cb, vx);
        store_spinor<PP>(p, pn, L5, s, cb, vp);
    }
}
// The same update with the new p written to a SECOND buffer and B p_new = (b5 + c5 Lambda) p_new written beside it,
// so that K1 of the next Mpc reads B p without the B-on-load stencil (for 16-bit storage the stencil and the
// conversion of its halo slices cost more than this extra 16-bit stream).  p_new of the slices s-1 (upper spins)
// and s+1 (lower spins) is recomputed from p_old and g; p_old is never overwritten, so there is no race.
template <class PX, class PP>
__global__ void __launch_bounds__(128)
xpupdate_b_kernel(void *x, float *xn, double a, const void *p, const float *pn, double b, const void *g, const float *gn,
                  void *pnew, float *pnewn, void *bp, float *bpn, float b5, float c5, float mf, int L5, long Vh, const double *coef,
                  int xmode)
{
    // xmode 1: x += a p.  The x update may run every other iteration (x is the widest vector of the update): xmode 0 leaves x
    // alone, xmode 2 adds both pending terms, x += a_prev p_prev + a p, where p_prev is what the pnew buffer still holds (the
    // double buffer of p) and is read slice by slice before the new p overwrites it.
    double a_prev = 0.0;
    if (coef) { a *= coef[0]; b *= coef[1]; a_prev = coef[2]; }
    // one thread walks the L5 slices of one 4D site, so every slice of p and g is loaded once: the new p of slice
    // s+1 is formed one step ahead, its lower spins feed B at s and its upper spins feed B at s+2
    using T = typename CompT<PX, PP, PP>::T;
    using RP = typename PP::R;
    const long cb = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= Vh) return;
    const T ta = (T)a, tb = (T)b, tap = (T)a_prev;
    RP cur[24], nxt[24], prev_up[12], first_low[12], vp[24], vg[24];
    auto new_p = [&](int s, RP *out, bool update_x) {
        load_spinor<PP>(p, pn, L5, s, cb, vp);
        load_spinor<PP>(g, gn, L5, s, cb, vg);
        if (update_x && xmode != 0) {
            typename PX::R vx[24];
            load_spinor<PX>(x, xn, L5, s, cb, vx);
            if (xmode == 2) {
                RP vo[24];
                load_spinor<PP>(pnew, pnewn, L5, s, cb, vo);
#pragma unroll
                for (int k = 0; k < 24; k++) vx[k] = (typename PX::R)((T)vx[k] + tap * (T)vo[k] + ta * (T)vp[k]);
            } else {
#pragma unroll
                for (int k = 0; k < 24; k++) vx[k] = (typename PX::R)((T)vx[k] + ta * (T)vp[k]);
            }
            store_spinor<PX>(x, xn, L5, s, cb, vx);
        }
#pragma unroll
        for (int k = 0; k < 24; k++) out[k] = (RP)((T)vg[k] + tb * (T)vp[k]);
    };
    {   // upper spins of the new p at slice L5-1 (wall neighbour of slice 0)
        RP hp[12], hg[12];
        load_half<PP>(p, pn, L5, L5 - 1, cb, 0, hp);
        load_half<PP>(g, gn, L5, L5 - 1, cb, 0, hg);
#pragma unroll
        for (int k = 0; k < 12; k++) prev_up[k] = (RP)((T)hg[k] + tb * (T)hp[k]);
    }
    new_p(0, cur, true);
#pragma unroll
    for (int k = 0; k < 12; k++) first_low[k] = cur[12 + k];
    for (int s = 0; s < L5; s++) {
        if (s + 1 < L5) new_p(s + 1, nxt, true);
        const float cu = (s == 0) ? -mf * c5 : c5, cl = (s == L5 - 1) ? -mf * c5 : c5;
        RP vb[24];
#pragma unroll
        for (int k = 0; k < 12; k++) {
            vb[k] = (RP)(b5 * (float)cur[k] + cu * (float)prev_up[k]);
            vb[12 + k] = (RP)(b5 * (float)cur[12 + k] + cl * (float)((s + 1 < L5) ? nxt[12 + k] : first_low[k]));
        }
        store_spinor<PP>(pnew, pnewn, L5, s, cb, cur);
        store_spinor<PP>(bp, bpn, L5, s, cb, vb);
#pragma unroll
        for (int k = 0; k < 12; k++) prev_up[k] = cur[k];
#pragma unroll
        for (int k = 0; k < 24; k++) cur[k] = nxt[k];
    }
}
int mdwf_launch_xpupdate_b(Prec px, const SpinorBuf &x, double a, const SpinorBuf &p, double b, const SpinorBuf &g,
                           const SpinorBuf &pnew, const SpinorBuf &bp, double b5, double c5, double mf, int L5, int Vh,
                           cudaStream_t st, int xmode)
{
    const int nb = (Vh + 127) / 128;
#define XB(PX) xpupdate_b_kernel<PX, PH><<<nb, 128, 0, st>>>(x.v, x.norm, a, p.v, p.norm, b, g.v, g.norm, pnew.v, \
                                                                     pnew.norm, bp.v, bp.norm, (float)b5, (float)c5, (float)mf, L5, Vh, tl_coef, xmode)
    if (px == PREC_S) XB(PS);
    else if (px == PREC_H) XB(PH);
    else return (int)cudaErrorInvalidValue;
#undef XB
    return (int)cudaGetLastError();
}

template <class PX>
static int xpupdate_p(Prec pp, const SpinorBuf &x, double a, const SpinorBuf &p, double b, const SpinorBuf &g, int L5, int Vh,
                      cudaStream_t st)
{
    const dim3 nb = site_grid(L5, Vh);
#define XP(PP) xpupdate_kernel<PX, PP><<<nb, RED_THREADS, 0, st>>>(x.v, x.norm, a, p.v, p.norm, b, g.v, g.norm, L5, Vh, tl_coef)
    switch (pp) {
    case PREC_D: XP(PD); break;
    case PREC_S: XP(PS); break;
    default: XP(PH); break;
    }
#undef XP
    return (int)cudaGetLastError();
}
int mdwf_launch_xpupdate(Prec px, const SpinorBuf &x, double a, Prec pp, const SpinorBuf &p, double b, const SpinorBuf &g,
                         int L5, int Vh, cudaStream_t st)
{
    switch (px) {
    case PREC_D: return xpupdate_p<PD>(pp, x, a, p, b, g, L5, Vh, st);
    case PREC_S: return xpupdate_p<PS>(pp, x, a, p, b, g, L5, Vh, st);
    default: return xpupdate_p<PH>(pp, x, a, p, b, g, L5, Vh, st);
    }
}

// ---- flat arrays (mdwf_blas_* entry points) -----------------------------------------------------
template <class T, int KIND>
__global__ void __launch_bounds__(RED_THREADS) flat_reduce_kernel(const T *x, const T *y, long long n, double *partial)
{
    double sum = 0.0;
    for (long long i = (long long)blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += (long long)gridDim.x * RED_THREADS) {
        const double a = (double)x[i];
        sum += (KIND == 0) ? a * a : a * (double)y[i];
    }
    block_partial(sum, partial);
}
template <class T>
__global__ void flat_axpy_kernel(double a, const T *x, T *y, long long n)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        y[i] = (T)((double)y[i] + a * (double)x[i]);
}

int mdwf_launch_flat_reduce(int kind, const void *x, const void *y, long long n, int real_bytes, double *partial,
                            double *result_dev, cudaStream_t st)
{
    const int nb = red_blocks(n / 4 + 1);
    if (real_bytes == 8) {
        if (kind == 0) flat_reduce_kernel<double, 0><<<nb, RED_THREADS, 0, st>>>((const double *)x, (const double *)y, n, partial);
        else flat_reduce_kernel<double, 1><<<nb, RED_THREADS, 0, st>>>((const double *)x, (const double *)y, n, partial);
    } else {
        if (kind == 0) flat_reduce_kernel<float, 0><<<nb, RED_THREADS, 0, st>>>((const float *)x, (const float *)y, n, partial);
        else flat_reduce_kernel<float, 1><<<nb, RED_THREADS, 0, st>>>((const float *)x, (const float *)y, n, partial);
    }
    final_sum_kernel<<<1, RED_THREADS, 0, st>>>(partial, nb, result_dev);
    return (int)cudaGetLastError();
}
int mdwf_launch_flat_axpy(double a, const void *x, void *y, long long n, int real_bytes, cudaStream_t st)
{
    const int nb = red_blocks(n / 4 + 1);
    if (real_bytes == 8) flat_axpy_kernel<double><<<nb, 256, 0, st>>>(a, (const double *)x, (double *)y, n);
    else flat_axpy_kernel<float><<<nb, 256, 0, st>>>(a, (const float *)x, (float *)y, n);
    return (int)cudaGetLastError();
}
