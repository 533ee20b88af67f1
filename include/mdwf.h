/*
 * mdwf.h -- C ABI of the B200-native Moebius domain-wall fermion (MDWF) solver library.
 *
 * The library computes the hot path of arXiv:1701.07559 (PAPER.md = the paper's text):
 * the valence MDWF inversion, i.e. the 4D even-odd ("asymmetric", Sec. VII)
 * Schur-preconditioned 5D Moebius operator built from the Moebius kernel of Eq. (2)
 * (parameters M5, L5, b5, c5 of Table II), applied inside
 * a mixed-precision ("double-half") conjugate-gradient solve on the normal
 * equations.  It plays the role of the Chroma<->QUDA solver interface of PAPER.md:350.
 *
 * Operator (the paper cites [113-115] for it and does not print it):
 *   D    = A - (1/2) H B,  A = alpha + beta Lambda,  B = b5 + c5 Lambda,
 *          alpha = b5 (4 - M5) + 1, beta = c5 (4 - M5) - 1,
 *          H = 4D Wilson hopping term (periodic x,y,z; antiperiodic t, applied in-kernel),
 *          (Lambda psi)_s = P- psi_{s+1} + P+ psi_{s-1} with the -m_f wall factor at the wrap.
 *   Mpc  = A - (1/4) H_oe B A^{-1} H_eo B  on odd sites (odd = (x+y+z+t) & 1 == 1).
 *
 * Conventions
 *   - All pointers named *_dev are DEVICE pointers, *_host are HOST pointers.  The caller owns
 *     every buffer it passes; the library copies what it needs and never keeps caller pointers.
 *   - real_bytes is 8 (double) or 4 (float): the type of the caller's buffer.  Complex numbers
 *     are interleaved (re, im).  Arrays are C-ordered:
 *       gauge          U[t][z][y][x][mu][row][col], mu in {x,y,z,t}; U_mu(x) is the link from x to
 *                      x+mu; plain SU(3), no boundary sign folded in.        (4 V4 x 18 reals)
 *       5D spinor      psi[s][t][z][y][x][spin][colour]                      (L5 V4 x 24 reals)
 *       parity spinor  psi[s][cb][spin][colour], cb = lex(x,y,z,t)/2 over the ODD sites,
 *                      lex = x + Lx (y + Ly (z + Lz t)).                     (L5 V4/2 x 24 reals)
 *     gamma matrices: DeGrand-Rossi basis, gamma5 = diag(+1,+1,-1,-1).
 *   - All work is enqueued on the context's stream (option "stream", default: the legacy default
 *     stream).  Functions that return scalars synchronise that stream before returning.
 *   - Every function returns MDWF_OK (0) or a negative error code; mdwf_last_error() gives text.
 *     There is no CPU fallback: without a CUDA device every compute call returns MDWF_ECUDA.
 */
#ifndef MDWF_H
#define MDWF_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mdwf_ctx mdwf_ctx; /* opaque, owned by the library */

enum {
    MDWF_OK = 0,
    MDWF_EARG = -1,     /* bad argument: odd extent, L5 < 2 or > 32, null pointer, bad real_bytes/op/option */
    MDWF_ENOGAUGE = -2, /* gauge field not loaded */
    MDWF_ECUDA = -3,    /* CUDA error (text in mdwf_last_error) */
    MDWF_ENOCONV = -4,  /* solver did not reach tol within maxiter; sol holds the best iterate */
    MDWF_ENOMEM = -5    /* device allocation failed */
};

enum { /* op codes of mdwf_apply */
    MDWF_OP_MPC = 0,       /* Mpc        : parity spinor -> parity spinor (S5 of the hot path)   */
    MDWF_OP_MPCDAG = 1,    /* Mpc^dagger : parity spinor -> parity spinor (S6)                   */
    MDWF_OP_MDAGM = 2,     /* Mpc^dagger Mpc                                                   */
    MDWF_OP_D = 3,         /* D          : full 5D spinor -> full 5D spinor                     */
    MDWF_OP_DDAG = 4,      /* D^dagger                                                          */
    MDWF_OP_MPC_SYM = 5,   /* symmetric preconditioning:              */
                           /*   Mpc_sym = 1 - (1/4) A^{-1} H_oe B A^{-1} H_eo B, parity spinor -> parity spinor */
    MDWF_OP_MPCDAG_SYM = 6 /* Mpc_sym^dagger = 1 - (1/4) B^+ H'_oe A^{-+} B^+ H'_eo A^{-+}                      */
};

/* Create a context for an Lx x Ly x Lz x Lt x L5 lattice (all 4D extents even, 2 <= L5 <= 32) and the
 * Moebius parameters of Eq. (2) / Table II.  Precomputes alpha, beta and the fifth-dimension tables. */
int mdwf_create(mdwf_ctx **out, int Lx, int Ly, int Lz, int Lt, int L5,
                double M5, double b5, double c5, double m_f);
int mdwf_destroy(mdwf_ctx *ctx);

/* Options (key, value as strings):
 *   "ladder"          "d" | "ds" | "dh" | "dsh"   precision ladder of mdwf_solve: fp64 only; fp64 reliable
 *                     updates + fp32 sloppy; fp64 + 16-bit sloppy; fp64 reliable residual + fp32 solution
 *                     accumulator + 16-bit operator and Krylov vectors ("double/single/half").  Default "d".
 *   "apply_precision" "auto" | "fp64" | "fp32" | "half"   arithmetic/storage used inside mdwf_apply;
 *                     "auto" = that of the caller's buffer (real_bytes).  Default "auto".
 *   "reconstruct"     "18" | "12"   SU(3) link storage; 12 keeps rows 0,1 and rebuilds row 2 =
 *                     conj(row0 x row1) in-kernel.  Takes effect at the next mdwf_load_gauge.  Default "18".
 *   "reliable_delta"  reliable-update threshold delta (default "0.1").
 *   "stream"          cudaStream_t as a decimal integer (default "0").
 *   "kernels"         "auto" (default: v5 where it applies and the lattice has at least 8 tiles per SM, else v3) | "v5" | "v3" |
 *                     "v2": kernel family for fp32 arithmetic.  v5: the tile-sweep kernels of hop5_kernels.cuh (TMA ring,
 *                     tensor-memory links and slice history) for K2, K1^dagger, K2^dagger and K1 from a precomputed B psi in fp32
 *                     storage when Lx/2 in {2,4,8,16}, Ly a multiple of 32/(Lx/2), L5 in {8,12}; everything else as v3.
 *                     v3: hop3_kernels.cuh (link tile by TMA, spinors through registers; L5 in {8,12,16});
 *                     v2: hop_kernels.cuh (always used for fp64 and other L5).
 *   "tile_l2_mb"      v5: L2 budget in MB for the working set of a z-chunk of tiles (default 48).
 *   "bp_stream"       "1" (default) | "0": 16-bit Krylov vectors only -- the fused CG update also writes B p, which K1 of
 *                     the next Mpc reads instead of applying B on load.
 *   "sweep_mb"        v2, v3: L2 budget in MB of one block-sweep slab (default 16; negative: lexicographic sweep).
 *   "release_workspace"  (any value) free the library's pooled work vectors now; they are reallocated on demand.
 *   "max_update_interval"  force a reliable update at least every n iterations (default "0": only the delta rule).
 *   "time_hops"       "1": mdwf_solve records CUDA events around the four hop kernels of every CG iteration (K1, K2, K1^dagger,
 *                     K2^dagger in the sloppy precision of the ladder); their average duration inside the solve is then in
 *                     mdwf_get_stat "hop_ms_k1" | "hop_ms_k2" | "hop_ms_k1dag" | "hop_ms_k2dag" (counts: "hop_n_..."). Default "0".
 *   "matpc"           "asym" (default; the operator Chroma uses) | "sym": Schur system mdwf_solve iterates on.
 *                     sym: Mpc_sym x_o = A^{-1} b'_o with Mpc_sym = 1 - (1/4) A^{-1} H_oe B A^{-1} H_eo B ("significant reduction of
 *                     the condition number"); same source preparation, reconstruction and returned residual.
 */
int mdwf_set_option(mdwf_ctx *ctx, const char *key, const char *value);

/* Copy the gauge field into the library's even-odd device layouts (fp64, fp32 and 16-bit copies). */
int mdwf_load_gauge(mdwf_ctx *ctx, const void *U_dev, int real_bytes);
int mdwf_load_gauge_host(mdwf_ctx *ctx, const void *U_host, int real_bytes);

/* out = op(in).  ops 0-2, 5, 6: parity spinors (odd sites); ops 3-4: full 5D spinors.  in_dev != out_dev. */
int mdwf_apply(mdwf_ctx *ctx, int op, const void *in_dev, void *out_dev, int real_bytes);

/* The same operators on a BATCH of right-hand sides (a propagator is 12 spin-colour columns
 * per source).  in_dev / out_dev hold nrhs parity vectors of mdwf_apply's layout back to back; op is MDWF_OP_MPC or
 * MDWF_OP_MPCDAG; the arithmetic is fp32 on fp32 or 16-bit storage ("apply_precision" "fp32" (default here) | "half").  One kernel
 * launch handles the whole batch: a thread block stages the link tile of its 32 sites once (and completes 12-real links once)
 * for all nrhs vectors.  Results are bit-identical to nrhs calls of mdwf_apply in the same precision with "kernels" "v3".
 * Errors: MDWF_EARG for other ops, nrhs outside 1..64, fp64, L5 outside {8, 12, 16} or |beta/alpha| >= 0.98. */
int mdwf_apply_batch(mdwf_ctx *ctx, int op, int nrhs, const void *in_dev, void *out_dev, int real_bytes);

/* Solve D x = src on the full 5D lattice (fp64 buffers): Schur preparation b' = b_o - D_oe A^{-1} b_e,
 * CG on Mpc^dagger Mpc (CGLS recurrences) with the configured precision ladder and reliable updates,
 * reconstruction x_e = A^{-1}(b_e - D_eo x_o).  tol is the target for ||src - D x|| / ||src||.
 * iters_out = CG iterations (one Mpc + one Mpc^dagger each); true_res_out = ||src - D x||_2 / ||src||_2
 * recomputed in fp64 with the unpreconditioned operator.  Returns MDWF_ENOCONV if maxiter was hit. */
int mdwf_solve(mdwf_ctx *ctx, const void *src_dev, void *sol_dev, double tol, int maxiter,
               int *iters_out, double *true_res_out);
/* Same with HOST buffers (fp64): host->device copy of src and device->host copy of sol included. */
int mdwf_solve_host(mdwf_ctx *ctx, const void *src_host, void *sol_host, double tol, int maxiter,
                    int *iters_out, double *true_res_out);

/* Deterministic BLAS-1 (S7) on flat device arrays of n reals (real_bytes 8 or 4); fp64 accumulation,
 * fixed reduction order (per-thread strided sums, warp shuffles, block tree, fixed-order final pass). */
int mdwf_blas_norm2(mdwf_ctx *ctx, const void *x_dev, long long n, int real_bytes, double *out);
int mdwf_blas_redot(mdwf_ctx *ctx, const void *x_dev, const void *y_dev, long long n, int real_bytes, double *out);
int mdwf_blas_axpy(mdwf_ctx *ctx, double a, const void *x_dev, void *y_dev, long long n, int real_bytes);

/* ||x||^2 (S7, as mdwf_blas_norm2: same arithmetic, same fixed reduction order, bit-identical result) through an entry point
 * that ALLOCATES NOTHING, for callers that cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses
 * that forbid it.  No context, no cudaMalloc / cudaFree / allocating library routine, no synchronisation, no host read-back:
 * two kernels are queued on `stream` (a cudaStream_t, NULL = the default stream) and the result is written to out_dev.
 *   x_dev    device pointer, n reals of real_bytes (8 or 4) bytes each; caller-owned, read only
 *   out_dev  device pointer to ONE double; caller-owned, written when the queued kernels have run
 * The per-block partial sums go to a scratch array that lives in the library image (a file-scope __device__ array of 4096 doubles
 * = 32 KB; every GPU that loads the library holds it until the process exits).  Limits and sharing:
 *   - n <= mdwf_noalloc_max_n() = 2^30 reals per call; beyond it the call returns MDWF_EARG and touches nothing;
 *   - every call on a device shares that one array, which keeps the last call's contents (nothing in it needs clearing: a call
 *     overwrites exactly the partials it reads back).  Calls that overlap on the GPU (different streams, or host threads whose
 *     launches are not ordered) RACE on it and give wrong results: the caller serialises them.
 * mdwf_noalloc_setup() takes the array's device address for the current device (cudaGetSymbolAddress; first use also loads the
 * module): call it once per device outside any graph capture; mdwf_blas_norm2_noalloc does it itself on first use otherwise.
 * Errors: MDWF_EARG (n < 0, n beyond the maximum, real_bytes, null pointer), MDWF_ECUDA; text in mdwf_noalloc_last_error()
 * (per host thread). */
int mdwf_blas_norm2_noalloc(const void *x_dev, long long n, int real_bytes, double *out_dev, void *stream);
int mdwf_noalloc_setup(void);
long long mdwf_noalloc_max_n(void);
const char *mdwf_noalloc_last_error(void);

/* 4D <-> 5D maps either side of the solve (Eq. (5), defines the quark field on the
 * walls and the midpoint field of the residual-mass ratio).  4D fields are eta[t][z][y][x][spin][colour] (V4 x 24 reals).
 * mdwf_wall_source: src(x,s) = delta_{s,0} P+ eta(x) + delta_{s,L5-1} P- eta(x) (lift = 0), or D_- applied to it (lift = 1;
 * D_- = c5 D_W - 1 slice by slice, the source of the physical 4D propagator; needs the gauge field).
 * mdwf_wall_project: q(x) = P- psi(x,0) + P+ psi(x,L5-1) (midpoint = 0) or Q(x) = P- psi(x,L5/2) + P+ psi(x,L5/2-1) (midpoint = 1). */
int mdwf_wall_source(mdwf_ctx *ctx, const void *eta_dev, void *src_dev, int real_bytes, int lift);
int mdwf_wall_project(mdwf_ctx *ctx, const void *psi_dev, void *q_dev, int real_bytes, int midpoint);

/* Gradient-flow smearing of the gauge field (Sec. III: "an infinitesimal stout-smearing
 * procedure", t_gf = 1.0; App. D: "the Symanzik action ... step size eps = 0.03").  U_dev: canonical gauge field in
 * fp64, flowed IN PLACE by nsteps steps of Luescher's third-order Runge-Kutta of size eps (flow time nsteps * eps) under
 * dV/dt = -g0^2 {dS/dV} V; action 0 = Wilson flow (plaquette), 1 = tree-level Symanzik (c0 = 5/3, c1 = -1/12); periodic
 * boundaries.  The flowed field is what mdwf_load_gauge should then be given.  plaq_out (may be null) receives the mean
 * plaquette <Re tr P>/3 of the flowed field; mdwf_plaquette returns it for any field (deterministic reduction). */
int mdwf_gradient_flow(mdwf_ctx *ctx, void *U_dev, double eps, int nsteps, int action, double *plaq_out);
int mdwf_plaquette(mdwf_ctx *ctx, const void *U_dev, double *out);

/* The 16-bit storage format of the sloppy precision as it is stored (the paper
 * says only "double-half"): one fp32 scale m = max |component| per (site, s) and 24 unsigned 16-bit words
 * u = round_to_nearest_even(v * (32767 / m)) + 32768, decoded as (u - 32768) * (m * (1 / 32767)) in fp32.
 * encode: parity spinor psi[s][cb][spin][colour] (real_bytes 8 or 4) -> words_dev uint16[s][cb][24], scales_dev
 * float[s][cb]; via_fp64 = 0 quantises the buffer with the layout kernel (the path of mdwf_apply), 1 converts it to the
 * fp64 device layout first and quantises with the BLAS-1 copy (the path of mdwf_solve).  decode is the inverse map.
 * Integer work: tests compare the words and scales bit for bit with a restatement of the formula. */
int mdwf_half_encode(mdwf_ctx *ctx, const void *in_dev, int real_bytes, int via_fp64, void *words_dev, void *scales_dev);
int mdwf_half_decode(mdwf_ctx *ctx, const void *words_dev, const void *scales_dev, void *out_dev, int real_bytes);

/* Per-context counters.  Keys: "launches" (kernels launched so far), "iterations", "reliable_updates",
 * "solve_seconds" (device time of the last solve, CUDA events), "true_residual", "op_applications"
 * (Mpc + Mpc^dagger applications in the last solve, all precisions), "sloppy_applications", and with option "time_hops" the
 * "hop_ms_*" / "hop_n_*" keys described there. */
int mdwf_get_stat(const mdwf_ctx *ctx, const char *key, double *value);

const char *mdwf_last_error(const mdwf_ctx *ctx);
/* The fixed flop count per odd 5D site per Mpc application: 2880 + 48 L5. */
int mdwf_flops_per_site(const mdwf_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* MDWF_H */
