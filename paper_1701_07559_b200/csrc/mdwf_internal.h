// mdwf_internal.h -- host-side declarations shared by the translation units of libmdwf_b200.so.
// Device layouts:
//   sites of one parity are grouped in 32s: g = cb >> 5, lane = cb & 31 (arrays padded to whole groups).
//   parity spinor, precision P:  chunk[((g*L5 + s)*NV + j)*32 + lane], chunk = double2 (fp64, NV=12, one
//                                complex), float4 (fp32, NV=6, two complex) or short4 (16-bit fixed point,
//                                NV=6) with one float scale norm[(g*L5 + s)*32 + lane] per 5D site.
//   gauge, per parity p of the site x: link[((g*8 + d)*NK + k)*32 + lane], one complex per chunk (double2 / float2 /
//                                short2), NK = 9 (18 reals) or 6 (12 reals); d = mu: U_mu(x), d = 4 + mu: U_mu(x-mu)^dagger.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

// slices per thread of the v3 kernels (hop3_kernels.cuh) for L5 = 12, and resident warps per SM asked of ptxas
#ifndef MDWF_H3_S12
#define MDWF_H3_S12 3
#endif
#ifndef MDWF_H3_WARPS
#define MDWF_H3_WARPS 8
#endif
#ifndef MDWF_H3_WARPS_H
#define MDWF_H3_WARPS_H 12
#endif
static inline int mdwf_h3_slices(int L5) { return L5 == 12 ? MDWF_H3_S12 : 2; }

enum Prec { PREC_D = 0, PREC_S = 1, PREC_H = 2 };

struct SpinorBuf {       // one single-parity 5D vector in a device layout
    void *v = nullptr;
    float *norm = nullptr;   // 16-bit format only
};

// n / d for 0 <= n < 2^31 as  __umulhi(n, m) >> s  (m = 0: d == 1)
struct FastDiv {
    unsigned m, s, d;
};
static inline FastDiv mdwf_fastdiv(unsigned d)
{
    FastDiv f;
    f.d = d;
    if (d <= 1) { f.m = 0; f.s = 0; return f; }
    unsigned sh = 0;
    while ((1ull << sh) < d) sh++;                       // 2^(sh-1) < d <= 2^sh
    f.m = (unsigned)((1ull << (31 + sh)) / d + 1);
    f.s = sh - 1;
    return f;
}

struct HopArgs {
    int L[4];
    FastDiv dLxh, dLy, dLz, dnb, dchunk;   // Lx/2, Ly, Lz, sweep_nb, sweep_nb * Lt
    int L5;
    int Vh;
    int parity_out;          // parity of the sites this launch writes
    int sweep_nb;            // block sweep order: blocks per (z-chunk, t) slab; 0 = plain lexicographic order
    int sweep_chunk;         // sites per (z-chunk, t) slab = ZC * Ly * Lx/2
    const void *in;          // hop input: vector on the opposite parity
    const float *in_norm;
    const void *own;         // own-site input (same parity as the output) or nullptr
    const float *own_norm;
    void *out;
    float *out_norm;
    const void *gauge;       // link tiles of the sites of parity_out: 8 directions per site (4 forward, 4 backward pulled back)
    int recon;               // 18 or 12
    double coef_hop;         // multiplies the hop sum
    double pre_d, pre_o;     // PRE = 1: input is (pre_d + pre_o Lambda) psi        (B on load)
    double own_d, own_o;     // OWN = 2/3: adds (own_d + own_o Lambda[^dagger]) psi_own
    double post_d, post_o;   // POST = 2: applies (post_d + post_o Lambda^dagger) to coef_hop * hop
    double mf;
    double *partial;         // v3 kernels: if non-null, ||out||^2 partial sums, one per block (fused norm, S7)
    const void *dense;       // POST = 1: device pointer to R[2][L5][L5] (P+ block, then P- block)
    // POST = 1 in the v3 kernels (hop3_kernels.cuh): coef_hop * B A^{-1} as a blocked recurrence
    int kver;                // host side: kernel family requested (2: hop_kernels.cuh, 3: hop3_kernels.cuh, 5: hop5 tile sweep where it pays, 6: hop5 wherever covered)
    int r_ok;                // 1 when the recurrence form is usable (|kappa| < 1)
    float r_nk;              // -kappa = -beta/alpha
    float r_cpow;            // (-kappa)^S, S = slices per thread
    float r_bz, r_cz;        // coef_hop b5/alpha, coef_hop c5/alpha
    float r_qC[4];           // coef_hop (b5 p_j + c5 p_{j-1})/alpha, p_j = (-kappa)^{j+1}, p_{-1} = 1
    float r_qW[32];          // coef_hop * wall term of slice s (effective index): -g m_f (b5 (-kappa)^{s+1} + c5 (-kappa)^s)
    // batched kernels (hop3b_kernels.cuh, NEXT-2): in / own / out hold nrhs vectors, right-hand side r at site indices [r batch_sites, ...)
    int nrhs;
    int batch_sites;         // Vh rounded up to a multiple of 32
    // v5 tile-sweep kernels (hop5_kernels.cuh): tile geometry, filled by the launcher
    int t5_NY, t5_nzq, t5_NT, t5_ntiles;   // 32-site groups along y, z-pairs per chunk, t-pairs, tiles
    int t5_l2mb;                           // L2 budget (MB) of a z-chunk's working set; 0 = default 48
    FastDiv t5_dNY, t5_dnzq, t5_dNT;
};

// hop family launcher.  dag: 0 H, 1 H^dagger.  pre: 0 none, 1 B on load.  post: 0 none, 1 dense
// s-matrix, 2 bidiagonal Lambda^dagger form.  own: 0 none, 1 + psi_own, 2 + (d + o Lambda) psi_own,
// 3 + (d + o Lambda^dagger) psi_own.  Returns cudaError_t as int.
int mdwf_launch_hop(Prec p, int dag, int pre, int post, int own, const HopArgs &a, cudaStream_t st);
// the same on a batch of a.nrhs right-hand sides (fp32 arithmetic only; Mpc / Mpc^dagger kernels); -1 = not covered
int mdwf_launch_hop_batch(Prec p, int dag, int pre, int post, int own, const HopArgs &a, cudaStream_t st);

// site-local dense s-matrix: out = M in (M = R[2][L5][L5] on device, in the precision's compute type)
int mdwf_launch_sdense(Prec p, int L5, int Vh, const SpinorBuf &in, const SpinorBuf &out, const void *dense,
                       cudaStream_t st);

// A^{-1} / A^{-dagger} as a recurrence for fp32 arithmetic (s5_kernels.cu); -1 when not covered (fp64, L5 outside {8,12,16}, in == out)
int mdwf_launch_srec(Prec p, int L5, int Vh, const SpinorBuf &in, const SpinorBuf &out, int dag, double alpha, double beta, double mf,
                     cudaStream_t st);

// BLAS-1 on parity vectors: out = a x + b y (y may be null when b == 0); if partial != nullptr also the
// deterministic reduction ||out||^2 -> *result_dev (double).  Mixed precisions allowed.
int mdwf_launch_axpby(Prec po, const SpinorBuf &out, double a, Prec px, const SpinorBuf &x, double b, Prec py,
                      const SpinorBuf &y, int L5, int Vh, double *partial, double *result_dev, cudaStream_t st);
// reductions on parity vectors: kind 0: ||x||^2, 1: Re<x,y>
int mdwf_launch_reduce(int kind, Prec px, const SpinorBuf &x, Prec py, const SpinorBuf &y, int L5, int Vh,
                       double *partial, double *result_dev, cudaStream_t st);
// fused CG update x += a p ; p = g + b p (x in precision px, p and g in precision pp)
int mdwf_launch_xpupdate(Prec px, const SpinorBuf &x, double a, Prec pp, const SpinorBuf &p, double b, const SpinorBuf &g,
                         int L5, int Vh, cudaStream_t st);
// 16-bit Krylov vectors: x += a p ; pnew = g + b p ; bp = (b5 + c5 Lambda) pnew   (p is not overwritten)
int mdwf_launch_xpupdate_b(Prec px, const SpinorBuf &x, double a, const SpinorBuf &p, double b, const SpinorBuf &g,
                           const SpinorBuf &pnew, const SpinorBuf &bp, double b5, double c5, double mf, int L5, int Vh,
                           cudaStream_t st, int xmode = 1);   // xmode 0: x untouched, 1: x += a p, 2: x += coef[2] pnew_old + a p
// device-resident CG scalars (blas_kernels.cu)
void mdwf_blas_set_coef(const double *coef_dev);
int mdwf_launch_cg_scalars(double *S, int mode, cudaStream_t st);
int mdwf_reduce_max_blocks();
// fixed-order sum of n partials into *result_dev (second pass of every reduction)
int mdwf_launch_final_sum(const double *partial, int n, double *result_dev, cudaStream_t st);

// flat-array BLAS-1 (mdwf_blas_* entry points)
int mdwf_launch_flat_reduce(int kind, const void *x, const void *y, long long n, int real_bytes, double *partial,
                            double *result_dev, cudaStream_t st);
int mdwf_launch_flat_axpy(double a, const void *x, void *y, long long n, int real_bytes, cudaStream_t st);

// layout conversion.  canonical parity spinor [s][cb][12 complex] <-> device layout
int mdwf_launch_parity_in(Prec p, const void *canon, int real_bytes, const SpinorBuf &dst, int L5, int Vh,
                          cudaStream_t st);
int mdwf_launch_parity_out(Prec p, const SpinorBuf &src, void *canon, int real_bytes, int L5, int Vh,
                           cudaStream_t st);
// canonical full 5D spinor [s][t][z][y][x][12 complex] <-> one parity in the device layout
int mdwf_launch_full_in(Prec p, const void *canon, int real_bytes, const SpinorBuf &dst, const int *L, int L5,
                        int parity, cudaStream_t st);
int mdwf_launch_full_out(Prec p, const SpinorBuf &src, void *canon, int real_bytes, const int *L, int L5,
                         int parity, cudaStream_t st);
// canonical gauge U[t][z][y][x][mu][3][3] -> device layout of one parity
int mdwf_launch_gauge_in(Prec p, const void *canon, int real_bytes, void *dst, const int *L, int parity, int recon,
                         cudaStream_t st);

// the 16-bit format as stored, in canonical order: words[(s*Vh + cb)*24 + k] (uint16, offset binary), scales[s*Vh + cb]
int mdwf_launch_half_export(const SpinorBuf &src, void *words, void *scales, int L5, int Vh, cudaStream_t st);
int mdwf_launch_half_import(const void *words, const void *scales, const SpinorBuf &dst, int L5, int Vh, cudaStream_t st);

// 4D <-> 5D maps on canonical buffers (NEXT-3): wall source injection, wall / midpoint projection
int mdwf_launch_wall_inject(const void *eta, void *b, int real_bytes, long V4, int L5, cudaStream_t st);
int mdwf_launch_wall_project(const void *psi, void *q, int real_bytes, long V4, int sm, int sp, cudaStream_t st);

// gradient flow of the gauge field (flow_kernels.cu, NEXT-4): one RK3 step in place; plaquette sum as per-block partials
int mdwf_launch_flow_step(void *U, void *Z, const int *L, double eps, double c0, double c1, cudaStream_t st);
int mdwf_launch_plaquette(const void *U, const int *L, double *partial, cudaStream_t st);
int mdwf_flow_plaquette_blocks(long V4);

// deterministic pseudo-random fill in [-1,1] (timing inputs only)
int mdwf_launch_fill(Prec p, const SpinorBuf &dst, int L5, int Vh, unsigned seed, cudaStream_t st);

size_t mdwf_spinor_bytes(Prec p, int L5, int Vh);   // bytes of the chunk array
size_t mdwf_gauge_bytes(Prec p, int Vh, int recon); // bytes of one parity's link array

// fp32 FMA rates of this device (peak_kernels.cu): tfma[0] FFMA, tfma[1] packed FFMA2, in 1e12 FMA/s
int mdwf_measure_fma_rates(double *tfma, cudaStream_t st);
