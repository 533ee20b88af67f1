// mdwf_api.cu -- the C ABI of include/mdwf.h: context, options, gauge load, operator application,
// mixed-precision CG with reliable updates (S8-S10).  Host logic only; every arithmetic step runs in
// the kernels of hop_kernels.cuh / blas_kernels.cu / layout_kernels.cu.
#include "../../include/mdwf.h"
#include "../../include/mdwf_bench.h"
#include "mdwf_internal.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <string>
#include <vector>

int mdwf_launch_hop_D(int, int, int, int, const HopArgs &, cudaStream_t);
int mdwf_launch_hop_S(int, int, int, int, const HopArgs &, cudaStream_t);
int mdwf_launch_hop_H(int, int, int, int, const HopArgs &, cudaStream_t);
int mdwf_launch_hop3_S(int, int, int, int, const HopArgs &, cudaStream_t);
int mdwf_launch_hop3_H(int, int, int, int, const HopArgs &, cudaStream_t);
int mdwf_launch_hop5_S(int, int, int, int, const HopArgs &, cudaStream_t);
int mdwf_launch_hop6_H(int, int, int, int, const HopArgs &, cudaStream_t);
int mdwf_launch_sdense_mma(int, int, const SpinorBuf &, const SpinorBuf &, const void *, cudaStream_t);
int mdwf_launch_sdense_D(int, int, const SpinorBuf &, const SpinorBuf &, const void *, cudaStream_t);
int mdwf_launch_sdense_S(int, int, const SpinorBuf &, const SpinorBuf &, const void *, cudaStream_t);
int mdwf_launch_sdense_H(int, int, const SpinorBuf &, const SpinorBuf &, const void *, cudaStream_t);

int mdwf_launch_hop(Prec p, int dag, int pre, int post, int own, const HopArgs &a, cudaStream_t st)
{
    if (a.kver >= 5 && p == PREC_S) {        // v5 tile sweep; -1 = not covered, fall back to v3
        const int rc = mdwf_launch_hop5_S(dag, pre, post, own, a, st);
        if (rc != -1) return rc;
    }
    if (a.kver >= 5 && p == PREC_H) {        // tile sweep for 16-bit storage (two sweep sets); -1 = not covered
        const int rc = mdwf_launch_hop6_H(dag, pre, post, own, a, st);
        if (rc != -1) return rc;
    }
    if (a.kver >= 3 && p != PREC_D) {        // v3 family (fp32 arithmetic); -1 = not covered, fall back to v2
        const int rc = (p == PREC_S) ? mdwf_launch_hop3_S(dag, pre, post, own, a, st)
                                     : mdwf_launch_hop3_H(dag, pre, post, own, a, st);
        if (rc != -1) return rc;
    }
    switch (p) {
    case PREC_D: return mdwf_launch_hop_D(dag, pre, post, own, a, st);
    case PREC_S: return mdwf_launch_hop_S(dag, pre, post, own, a, st);
    default: return mdwf_launch_hop_H(dag, pre, post, own, a, st);
    }
}
int mdwf_launch_hop3_batch_S(int, int, int, int, const HopArgs &, cudaStream_t);
int mdwf_launch_hop3_batch_H(int, int, int, int, const HopArgs &, cudaStream_t);
int mdwf_launch_hop_batch(Prec p, int dag, int pre, int post, int own, const HopArgs &a, cudaStream_t st)
{
    if (p == PREC_S) return mdwf_launch_hop3_batch_S(dag, pre, post, own, a, st);
    if (p == PREC_H) return mdwf_launch_hop3_batch_H(dag, pre, post, own, a, st);
    return -1;                               // fp64: no batched kernel (hop_kernels.cuh keeps no link tile)
}
int mdwf_launch_sdense(Prec p, int L5, int Vh, const SpinorBuf &in, const SpinorBuf &out, const void *dense,
                       cudaStream_t st)
{
    switch (p) {
    case PREC_D: {   // fp64: tensor-core (DMMA) contraction for L5 <= 16, FMA kernel beyond
        const int rc = mdwf_launch_sdense_mma(L5, Vh, in, out, dense, st);
        return rc != -1 ? rc : mdwf_launch_sdense_D(L5, Vh, in, out, dense, st);
    }
    case PREC_S: return mdwf_launch_sdense_S(L5, Vh, in, out, dense, st);
    default: return mdwf_launch_sdense_H(L5, Vh, in, out, dense, st);
    }
}

enum { DENSE_BAINV = 0, DENSE_BAINV_DAG = 1, DENSE_AINV = 2, DENSE_AINV_DAG = 3, DENSE_KINDS = 4 };

struct mdwf_ctx {
    int L[4];
    int L5;
    int Vh;
    double M5, b5, c5, mf, alpha, beta;
    cudaStream_t st = 0;
    int recon_opt = 18, recon = 18;
    int ladder = 0;          // 0 d, 1 ds, 2 dh, 3 dsh
    int apply_prec = -1;     // -1 auto
    double delta = 0.1;
    int max_update_interval = 0;
    int use_bp = 1;          // 16-bit Krylov vectors: let the CG update write B p for K1 (option "bp_stream")
    int matpc_sym = 0;       // 0: asymmetric Schur operator (what Chroma uses), 1: symmetric (NEXT-1)
    int kver = 5;            // kernel family for fp32 arithmetic: 5 = hop5_kernels.cuh tile sweep where it applies, else as 3;
                             // 3 = hop3_kernels.cuh (link tile by TMA, spinors through registers),
                             // 4 = the same with the t+- neighbour groups staged by TMA too, 2 = hop_kernels.cuh
    int tile_l2_mb = 0;      // v5: L2 budget (MB) of the working set of a z-chunk of tiles; 0 = default 48
    int sweep_mb = 0;        // L2 budget (MB) of one sweep slab; 0 = default 16, < 0 = lexicographic sweep
    int sweep_rhs = 1;       // right-hand sides a block walks through per slab site (batched kernels): the slab holds that many vectors
    bool gauge_loaded = false;
    void *gauge[3][2] = {{nullptr, nullptr}, {nullptr, nullptr}, {nullptr, nullptr}};
    void *dense[2][DENSE_KINDS] = {{nullptr, nullptr, nullptr, nullptr}, {nullptr, nullptr, nullptr, nullptr}};   // [0] double, [1] float
    std::map<std::string, SpinorBuf> pool;
    std::map<std::string, void *> raw;
    double *partial = nullptr, *result_dev = nullptr, *result_host = nullptr;
    int defer_slot = -1;             // >= 0: reductions leave their result in result_dev[defer_slot] and are NOT read back
    double *hop_partial = nullptr;   // one ||out||^2 partial per block of a hop launch (fused norms)
    // stats
    double launches = 0, iterations = 0, reliable_updates = 0, solve_seconds = 0, true_residual = 0;
    double op_applications = 0, sloppy_applications = 0;
    // option "time_hops": CUDA events around the four hop kernels of a CG iteration (sloppy precision) inside mdwf_solve, so that
    // a kernel's average launch duration IN the timed solve can be reported beside the one measured alone (bench.py roofline)
    int time_hops = 0;
    int hop_time_prec = -1;          // >= 0 while a solve is running: the precision whose hop launches are timed
    std::vector<cudaEvent_t> hop_ev; // pairs (before, after)
    std::vector<int> hop_ev_tag;     // one tag per pair: 0 K1, 1 K2, 2 K1^dagger, 3 K2^dagger
    double hop_ms[4] = {0, 0, 0, 0}, hop_n[4] = {0, 0, 0, 0};
    // mdwf_solve_host: the device->host copy of the solution starts on a second stream as soon as the solution is written and
    // runs under the fp64 true-residual computation that ends the solve
    void *d2h_dst = nullptr;
    size_t d2h_bytes = 0;
    bool d2h_issued = false;
    cudaStream_t copy_st = nullptr;
    cudaEvent_t sol_ready = nullptr;
    std::string err;
};

#define CUDA_OK(ctx, call)                                                                          \
    do {                                                                                            \
        cudaError_t e_ = (cudaError_t)(call);                                                       \
        if (e_ != cudaSuccess) {                                                                    \
            (ctx)->err = std::string(#call) + ": " + cudaGetErrorString(e_);                        \
            return (e_ == cudaErrorMemoryAllocation) ? MDWF_ENOMEM : MDWF_ECUDA;                    \
        }                                                                                           \
    } while (0)
#define TRY(call)                \
    do {                         \
        int rc_ = (call);        \
        if (rc_ != MDWF_OK) return rc_; \
    } while (0)

// ---- fifth-dimension tables (host, fp64; independent numeric inverse, not a closed form) ---------
static void invert(std::vector<double> &a, int n)   // Gauss-Jordan with partial pivoting, in place
{
    std::vector<double> inv(n * n, 0.0);
    for (int i = 0; i < n; i++) inv[i * n + i] = 1.0;
    for (int c = 0; c < n; c++) {
        int piv = c;
        for (int r = c + 1; r < n; r++)
            if (std::fabs(a[r * n + c]) > std::fabs(a[piv * n + c])) piv = r;
        for (int k = 0; k < n; k++) { std::swap(a[c * n + k], a[piv * n + k]); std::swap(inv[c * n + k], inv[piv * n + k]); }
        const double d = 1.0 / a[c * n + c];
        for (int k = 0; k < n; k++) { a[c * n + k] *= d; inv[c * n + k] *= d; }
        for (int r = 0; r < n; r++)
            if (r != c) {
                const double f = a[r * n + c];
                if (f != 0.0)
                    for (int k = 0; k < n; k++) { a[r * n + k] -= f * a[c * n + k]; inv[r * n + k] -= f * inv[c * n + k]; }
            }
    }
    a = inv;
}

static void build_tables(const mdwf_ctx *c, std::vector<double> out[DENSE_KINDS])
{
    const int n = c->L5;
    // shift matrix T: (T v)_s = v_{s-1}, wall factor -m_f at the wrap.  P+ block of Lambda is T, P- block T^T.
    std::vector<double> T(n * n, 0.0);
    for (int s = 1; s < n; s++) T[s * n + s - 1] = 1.0;
    T[0 * n + n - 1] += -c->mf;
    std::vector<double> Ap(n * n), Am(n * n), Bp(n * n), Bm(n * n);
    for (int i = 0; i < n; i++)
        for (int j = 0; j < n; j++) {
            const double id = (i == j) ? 1.0 : 0.0;
            Ap[i * n + j] = c->alpha * id + c->beta * T[i * n + j];
            Am[i * n + j] = c->alpha * id + c->beta * T[j * n + i];
            Bp[i * n + j] = c->b5 * id + c->c5 * T[i * n + j];
            Bm[i * n + j] = c->b5 * id + c->c5 * T[j * n + i];
        }
    std::vector<double> Aip = Ap, Aim = Am;
    invert(Aip, n);
    invert(Aim, n);
    for (int k = 0; k < DENSE_KINDS; k++) out[k].assign(2 * n * n, 0.0);
    for (int i = 0; i < n; i++)
        for (int j = 0; j < n; j++) {
            double sp = 0, sm = 0;
            for (int k = 0; k < n; k++) { sp += Bp[i * n + k] * Aip[k * n + j]; sm += Bm[i * n + k] * Aim[k * n + j]; }
            out[DENSE_BAINV][i * n + j] = sp;
            out[DENSE_BAINV][n * n + i * n + j] = sm;
            out[DENSE_BAINV_DAG][j * n + i] = sp;            // (B A^{-1})^T per chirality = A^{-+} B^+
            out[DENSE_BAINV_DAG][n * n + j * n + i] = sm;
            out[DENSE_AINV][i * n + j] = Aip[i * n + j];
            out[DENSE_AINV][n * n + i * n + j] = Aim[i * n + j];
            out[DENSE_AINV_DAG][j * n + i] = Aip[i * n + j];           // A^{-+} per chirality = transpose
            out[DENSE_AINV_DAG][n * n + j * n + i] = Aim[i * n + j];
        }
}

// ---- memory helpers ----------------------------------------------------------------------------
static int get_spinor(mdwf_ctx *c, const std::string &name, Prec p, SpinorBuf *out)
{
    const std::string key = name + (p == PREC_D ? ".d" : p == PREC_S ? ".s" : ".h");
    auto it = c->pool.find(key);
    if (it != c->pool.end()) { *out = it->second; return MDWF_OK; }
    SpinorBuf b;
    CUDA_OK(c, cudaMalloc(&b.v, mdwf_spinor_bytes(p, c->L5, c->Vh)));
    if (p == PREC_H) CUDA_OK(c, cudaMalloc((void **)&b.norm, sizeof(float) * (size_t)c->L5 * ((c->Vh + 31) / 32 * 32)));
    c->pool[key] = b;
    *out = b;
    return MDWF_OK;
}
static int get_raw(mdwf_ctx *c, const std::string &name, size_t bytes, void **out)
{
    auto it = c->raw.find(name);
    if (it != c->raw.end()) { *out = it->second; return MDWF_OK; }
    void *p = nullptr;
    CUDA_OK(c, cudaMalloc(&p, bytes));
    c->raw[name] = p;
    *out = p;
    return MDWF_OK;
}
static void free_pool(mdwf_ctx *c)
{
    for (auto &kv : c->pool) { cudaFree(kv.second.v); if (kv.second.norm) cudaFree(kv.second.norm); }
    c->pool.clear();
    for (auto &kv : c->raw) cudaFree(kv.second);
    c->raw.clear();
}

static int ensure_scalars(mdwf_ctx *c)
{
    if (c->partial) return MDWF_OK;
    CUDA_OK(c, cudaMalloc((void **)&c->partial, sizeof(double) * mdwf_reduce_max_blocks()));
    CUDA_OK(c, cudaMalloc((void **)&c->result_dev, sizeof(double) * 16));
    CUDA_OK(c, cudaMalloc((void **)&c->hop_partial, sizeof(double) * (size_t)((c->Vh + 31) / 32)));
    CUDA_OK(c, cudaMallocHost((void **)&c->result_host, sizeof(double) * 4));
    return MDWF_OK;
}
static int fetch_scalar(mdwf_ctx *c, double *out)
{
    CUDA_OK(c, cudaMemcpyAsync(c->result_host, c->result_dev, sizeof(double), cudaMemcpyDeviceToHost, c->st));
    CUDA_OK(c, cudaStreamSynchronize(c->st));
    *out = c->result_host[0];
    return MDWF_OK;
}

// ---- BLAS-1 wrappers (count launches) ------------------------------------------------------------
static int v_axpby(mdwf_ctx *c, Prec po, const SpinorBuf &out, double a, Prec px, const SpinorBuf &x, double b, Prec py,
                   const SpinorBuf *y, double *norm2_out)
{
    SpinorBuf none;
    TRY(ensure_scalars(c));
    const bool defer = c->defer_slot >= 0;
    CUDA_OK(c, mdwf_launch_axpby(po, out, a, px, x, b, py, y ? *y : none, c->L5, c->Vh, norm2_out ? c->partial : nullptr,
                                 c->result_dev + (defer ? c->defer_slot : 0), c->st));
    c->launches += norm2_out ? 2 : 1;
    if (norm2_out && !defer) TRY(fetch_scalar(c, norm2_out));
    return MDWF_OK;
}
static int v_norm2(mdwf_ctx *c, Prec p, const SpinorBuf &x, double *out)
{
    TRY(ensure_scalars(c));
    const bool defer = c->defer_slot >= 0;
    CUDA_OK(c, mdwf_launch_reduce(0, p, x, p, x, c->L5, c->Vh, c->partial, c->result_dev + (defer ? c->defer_slot : 0), c->st));
    c->launches += 2;
    return defer ? MDWF_OK : fetch_scalar(c, out);
}
static int v_zero(mdwf_ctx *c, Prec p, const SpinorBuf &x)
{
    CUDA_OK(c, cudaMemsetAsync(x.v, 0, mdwf_spinor_bytes(p, c->L5, c->Vh), c->st));
    if (p == PREC_H) CUDA_OK(c, cudaMemsetAsync(x.norm, 0, sizeof(float) * (size_t)c->L5 * ((c->Vh + 31) / 32 * 32), c->st));
    return MDWF_OK;
}

// ---- operator building blocks ---------------------------------------------------------------------
static const void *dense_ptr(const mdwf_ctx *c, Prec p, int kind) { return c->dense[p == PREC_D ? 0 : 1][kind]; }

static HopArgs base_args(const mdwf_ctx *c, Prec p, int parity_out, const SpinorBuf &in, const SpinorBuf *own,
                         const SpinorBuf &out)
{
    HopArgs a;
    memset(&a, 0, sizeof(a));
    for (int d = 0; d < 4; d++) a.L[d] = c->L[d];
    a.L5 = c->L5;
    a.Vh = c->Vh;
    a.parity_out = parity_out;
    // z-chunked sweep: ZC = largest divisor of Lz whose slab (3 spinor streams of ZC planes) stays under the budget
    {
        const long plane = (long)(c->L[0] / 2) * c->L[1];
        const long rb = (p == PREC_D) ? 8 : (p == PREC_S ? 4 : 2);
        // (batched kernels: the slab holds sweep_rhs vectors per stream and gets half of the 126 MB L2)
        const long budget = c->sweep_mb > 0 ? (long)c->sweep_mb << 20 : ((c->sweep_rhs > 1 ? 64L : 16L) << 20);
        int zc = 0;
        for (int d = 1; d <= c->L[2]; d++)
            if (c->L[2] % d == 0 && (d * plane) % 32 == 0 && d * plane * 3 * c->L5 * 24 * rb * c->sweep_rhs <= budget) zc = d;
        if (c->sweep_mb < 0 || zc == c->L[2] || zc < 2) zc = 0;
        a.sweep_nb = zc ? (int)(zc * plane / 32) : 0;
        a.sweep_chunk = (int)(zc * plane);
    }
    a.in = in.v; a.in_norm = in.norm;
    a.own = own ? own->v : nullptr; a.own_norm = own ? own->norm : nullptr;
    a.out = out.v; a.out_norm = out.norm;
    a.gauge = c->gauge[p][parity_out];
    a.dLxh = mdwf_fastdiv((unsigned)(c->L[0] / 2)); a.dLy = mdwf_fastdiv((unsigned)c->L[1]); a.dLz = mdwf_fastdiv((unsigned)c->L[2]);
    a.dnb = mdwf_fastdiv((unsigned)a.sweep_nb); a.dchunk = mdwf_fastdiv((unsigned)(a.sweep_nb * c->L[3]));
    a.recon = c->recon;
    a.mf = c->mf;
    return a;
}
// constants of the recurrence form of coef_hop * B A^{-1} (hop3_kernels.cuh)
static void fill_recurrence(const mdwf_ctx *c, HopArgs &a, double b5, double c5)
{
    const double ka = c->beta / c->alpha, nk = -ka, coef = a.coef_hop;
    const int S = mdwf_h3_slices(c->L5);
    a.r_ok = (std::fabs(ka) < 0.98) ? 1 : 0;
    a.r_nk = (float)nk;
    a.r_cpow = (float)std::pow(nk, S);
    a.r_bz = (float)(coef * b5 / c->alpha);
    a.r_cz = (float)(coef * c5 / c->alpha);
    for (int j = 0; j < 4; j++)
        a.r_qC[j] = (float)(coef * (b5 * std::pow(nk, j + 1) + c5 * std::pow(nk, j)) / c->alpha);
    const double g = 1.0 / (c->alpha * (1.0 + c->mf * std::pow(nk, c->L5)));
    for (int s = 0; s < 32; s++)
        a.r_qW[s] = (s < c->L5) ? (float)(coef * (-g * c->mf) * (b5 * std::pow(nk, s + 1) + c5 * std::pow(nk, s))) : 0.f;
}
static int run_hop(mdwf_ctx *c, Prec p, int dag, int pre, int post, int own, HopArgs a, bool ainv_only = false)
{
    a.kver = c->kver;
    a.t5_l2mb = c->tile_l2_mb;
    if (post == 1 && p != PREC_D && a.kver >= 3) fill_recurrence(c, a, ainv_only ? 1.0 : c->b5, ainv_only ? 0.0 : c->c5);   // coef (B A^{-1}) or coef A^{-1}
    int tag = -1;
    if (c->time_hops && (int)p == c->hop_time_prec) {
        if (!dag && post == 1 && own == 0) tag = 0;
        else if (!dag && post == 0 && own == 2) tag = 1;
        else if (dag && post == 1 && own == 0) tag = 2;
        else if (dag && post == 2 && own == 3) tag = 3;
    }
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (tag >= 0) {
        const size_t k = c->hop_ev_tag.size();
        if (c->hop_ev.size() < 2 * (k + 1)) {
            CUDA_OK(c, cudaEventCreate(&e0));
            c->hop_ev.push_back(e0);
            CUDA_OK(c, cudaEventCreate(&e1));
            c->hop_ev.push_back(e1);
        }
        e0 = c->hop_ev[2 * k]; e1 = c->hop_ev[2 * k + 1];
        c->hop_ev_tag.push_back(tag);
        CUDA_OK(c, cudaEventRecord(e0, c->st));
    }
    CUDA_OK(c, mdwf_launch_hop(p, dag, pre, post, own, a, c->st));
    if (tag >= 0) CUDA_OK(c, cudaEventRecord(e1, c->st));
    c->launches += 1;
    return MDWF_OK;
}

// Mpc in_o = A in_o - (1/4) H_oe [B A^{-1}] H_eo [B in_o];  tmp holds the even-site intermediate.
static int op_Mpc_k1(mdwf_ctx *c, Prec p, const SpinorBuf &in, const SpinorBuf &tmp)
{
    HopArgs k1 = base_args(c, p, 0, in, nullptr, tmp);        // K1: t_e = (B A^{-1}) H_eo (B in_o)
    k1.coef_hop = c->b5; k1.pre_d = c->b5; k1.pre_o = c->c5; k1.dense = dense_ptr(c, p, DENSE_BAINV);   // b5 of B-on-load folded in
    return run_hop(c, p, 0, 1, 1, 0, k1);
}
// K1 of Mpc from a precomputed B in_o (written by the fused CG update for 16-bit vectors): t_e = (B A^{-1}) H_eo (B in)_o
static int op_Mpc_k1_from_B(mdwf_ctx *c, Prec p, const SpinorBuf &Bin, const SpinorBuf &tmp)
{
    HopArgs k1 = base_args(c, p, 0, Bin, nullptr, tmp);
    k1.coef_hop = 1.0; k1.dense = dense_ptr(c, p, DENSE_BAINV);
    return run_hop(c, p, 0, 0, 1, 0, k1);
}
// the v3 kernels can emit ||out||^2 partials from their epilogue (fused norm)
static bool fused_norm_available(const mdwf_ctx *c, Prec p)
{
    return p != PREC_D && c->kver >= 3 && (c->L5 == 8 || c->L5 == 12 || c->L5 == 16);
}
// K1 reading a precomputed B p exists only in the recurrence (v3) family: |kappa| < 0.98, see fill_recurrence
static bool bp_stream_available(const mdwf_ctx *c, Prec p)
{
    return fused_norm_available(c, p) && std::fabs(c->beta / c->alpha) < 0.98;
}
static int finish_norm(mdwf_ctx *c, Prec p, const SpinorBuf &out, bool fused, double *norm2_out)
{
    if (!norm2_out) return MDWF_OK;
    if (!fused) return v_norm2(c, p, out, norm2_out);
    const bool defer = c->defer_slot >= 0;
    CUDA_OK(c, mdwf_launch_final_sum(c->hop_partial, (c->Vh + 31) / 32, c->result_dev + (defer ? c->defer_slot : 0), c->st));
    c->launches += 1;
    return defer ? MDWF_OK : fetch_scalar(c, norm2_out);
}
static int op_Mpc_k2(mdwf_ctx *c, Prec p, const SpinorBuf &in, const SpinorBuf &tmp, const SpinorBuf &out,
                     double *norm2_out = nullptr)
{
    HopArgs k2 = base_args(c, p, 1, tmp, &in, out);           // K2: out_o = A in_o - (1/4) H_oe t_e
    k2.coef_hop = -0.25; k2.own_d = c->alpha; k2.own_o = c->beta;
    const bool fused = norm2_out && fused_norm_available(c, p);
    if (fused) { TRY(ensure_scalars(c)); k2.partial = c->hop_partial; }
    TRY(run_hop(c, p, 0, 0, 0, 2, k2));
    return finish_norm(c, p, out, fused, norm2_out);
}
static int op_Mpc(mdwf_ctx *c, Prec p, const SpinorBuf &in, const SpinorBuf &tmp, const SpinorBuf &out,
                  double *norm2_out = nullptr)
{
    TRY(op_Mpc_k1(c, p, in, tmp));
    TRY(op_Mpc_k2(c, p, in, tmp, out, norm2_out));
    c->op_applications += 1;
    if (p != PREC_D) c->sloppy_applications += 1;
    return MDWF_OK;
}
// Mpc^+ in_o = A^+ in_o - (1/4) B^+ H'_oe [A^{-+} B^+] H'_eo in_o
static int op_Mpcdag_k1(mdwf_ctx *c, Prec p, const SpinorBuf &in, const SpinorBuf &tmp)
{
    HopArgs k1 = base_args(c, p, 0, in, nullptr, tmp);        // K1+: u_e = (A^{-+} B^+) H'_eo in_o
    k1.coef_hop = 1.0; k1.dense = dense_ptr(c, p, DENSE_BAINV_DAG);
    return run_hop(c, p, 1, 0, 1, 0, k1);
}
static int op_Mpcdag_k2(mdwf_ctx *c, Prec p, const SpinorBuf &in, const SpinorBuf &tmp, const SpinorBuf &out,
                        double *norm2_out = nullptr)
{
    HopArgs k2 = base_args(c, p, 1, tmp, &in, out);           // K2+: out_o = A^+ in_o - (1/4) B^+ H'_oe u_e
    k2.coef_hop = -0.25; k2.post_d = c->b5; k2.post_o = c->c5; k2.own_d = c->alpha; k2.own_o = c->beta;
    const bool fused = norm2_out && fused_norm_available(c, p);
    if (fused) { TRY(ensure_scalars(c)); k2.partial = c->hop_partial; }
    TRY(run_hop(c, p, 1, 0, 2, 3, k2));
    return finish_norm(c, p, out, fused, norm2_out);
}
static int op_Mpcdag(mdwf_ctx *c, Prec p, const SpinorBuf &in, const SpinorBuf &tmp, const SpinorBuf &out,
                     double *norm2_out = nullptr)
{
    TRY(op_Mpcdag_k1(c, p, in, tmp));
    TRY(op_Mpcdag_k2(c, p, in, tmp, out, norm2_out));
    c->op_applications += 1;
    if (p != PREC_D) c->sloppy_applications += 1;
    return MDWF_OK;
}
// ---- NEXT-1: symmetric preconditioning ----------------------------------------------
// Mpc_sym in_o = in_o - (1/4) A^{-1} H_oe [B A^{-1} H_eo B in_o]: K1 as for Mpc, K2 with A^{-1} as its POST step and OWN = 1
static int op_Ainv_dag(mdwf_ctx *c, Prec p, const SpinorBuf &in, const SpinorBuf &out);
static int op_Mpc_sym(mdwf_ctx *c, Prec p, const SpinorBuf &in, const SpinorBuf &tmp, const SpinorBuf &out, double *norm2_out = nullptr)
{
    TRY(op_Mpc_k1(c, p, in, tmp));
    HopArgs k2 = base_args(c, p, 1, tmp, &in, out);
    k2.coef_hop = -0.25; k2.dense = dense_ptr(c, p, DENSE_AINV);
    const bool fused = norm2_out && fused_norm_available(c, p) && std::fabs(c->beta / c->alpha) < 0.98;
    if (fused) { TRY(ensure_scalars(c)); k2.partial = c->hop_partial; }
    TRY(run_hop(c, p, 0, 0, 1, 1, k2, true));
    c->op_applications += 1;
    if (p != PREC_D) c->sloppy_applications += 1;
    return finish_norm(c, p, out, fused, norm2_out);
}
// Mpc_sym^+ in_o = in_o - (1/4) B^+ H'_oe [A^{-+} B^+ H'_eo (A^{-+} in_o)]: a site-local A^{-+} pass (w holds it), then K1^+ as for
// Mpc^+ and K2^+ with OWN = 1
static int op_Mpcdag_sym(mdwf_ctx *c, Prec p, const SpinorBuf &in, const SpinorBuf &w, const SpinorBuf &tmp, const SpinorBuf &out,
                         double *norm2_out = nullptr)
{
    TRY(op_Ainv_dag(c, p, in, w));
    TRY(op_Mpcdag_k1(c, p, w, tmp));
    HopArgs k2 = base_args(c, p, 1, tmp, &in, out);
    k2.coef_hop = -0.25; k2.post_d = c->b5; k2.post_o = c->c5;
    const bool fused = norm2_out && fused_norm_available(c, p);
    if (fused) { TRY(ensure_scalars(c)); k2.partial = c->hop_partial; }
    TRY(run_hop(c, p, 1, 0, 2, 1, k2));
    c->op_applications += 1;
    if (p != PREC_D) c->sloppy_applications += 1;
    return finish_norm(c, p, out, fused, norm2_out);
}
// one parity of D: out_p = A in_p - (1/2) H_{p,pbar} B in_pbar
static int op_D_parity(mdwf_ctx *c, Prec p, int parity, const SpinorBuf &in_other, const SpinorBuf &in_same,
                       const SpinorBuf &out)
{
    HopArgs a = base_args(c, p, parity, in_other, &in_same, out);
    a.coef_hop = -0.5 * c->b5; a.pre_d = c->b5; a.pre_o = c->c5; a.own_d = c->alpha; a.own_o = c->beta;
    return run_hop(c, p, 0, 1, 0, 2, a);
}
// one parity of D^+: out_p = A^+ in_p - (1/2) B^+ H'_{p,pbar} in_pbar
static int op_Ddag_parity(mdwf_ctx *c, Prec p, int parity, const SpinorBuf &in_other, const SpinorBuf &in_same,
                          const SpinorBuf &out)
{
    HopArgs a = base_args(c, p, parity, in_other, &in_same, out);
    a.coef_hop = -0.5; a.post_d = c->b5; a.post_o = c->c5; a.own_d = c->alpha; a.own_o = c->beta;
    return run_hop(c, p, 1, 0, 2, 3, a);
}
// out_p = own_p + (1/2) H_{p,pbar} B in_pbar   ( = own_p - D_{p,pbar} in_pbar ), Schur preparation / reconstruction
static int op_schur_hop(mdwf_ctx *c, Prec p, int parity, const SpinorBuf &in_other, const SpinorBuf &own,
                        const SpinorBuf &out)
{
    HopArgs a = base_args(c, p, parity, in_other, &own, out);
    a.coef_hop = 0.5 * c->b5; a.pre_d = c->b5; a.pre_o = c->c5;
    return run_hop(c, p, 0, 1, 0, 1, a);
}
static int op_Ainv(mdwf_ctx *c, Prec p, const SpinorBuf &in, const SpinorBuf &out)
{
    CUDA_OK(c, mdwf_launch_sdense(p, c->L5, c->Vh, in, out, dense_ptr(c, p, DENSE_AINV), c->st));
    c->launches += 1;
    return MDWF_OK;
}

static int op_Ainv_dag(mdwf_ctx *c, Prec p, const SpinorBuf &in, const SpinorBuf &out)
{
    if (std::fabs(c->beta / c->alpha) < 0.98) {          // recurrence form (fp32 arithmetic); else the dense table
        const int rc = mdwf_launch_srec(p, c->L5, c->Vh, in, out, 1, c->alpha, c->beta, c->mf, c->st);
        if (rc != -1) { CUDA_OK(c, rc); c->launches += 1; return MDWF_OK; }
    }
    CUDA_OK(c, mdwf_launch_sdense(p, c->L5, c->Vh, in, out, dense_ptr(c, p, DENSE_AINV_DAG), c->st));
    c->launches += 1;
    return MDWF_OK;
}

static int check_ready(mdwf_ctx *c)
{
    if (!c) return MDWF_EARG;
    if (!c->gauge_loaded) { c->err = "gauge field not loaded"; return MDWF_ENOGAUGE; }
    return MDWF_OK;
}

// =====================================================================================================
extern "C" {

int mdwf_create(mdwf_ctx **out, int Lx, int Ly, int Lz, int Lt, int L5, double M5, double b5, double c5, double m_f)
{
    if (!out) return MDWF_EARG;
    *out = nullptr;
    const int L[4] = {Lx, Ly, Lz, Lt};
    for (int d = 0; d < 4; d++)
        if (L[d] < 2 || (L[d] & 1)) return MDWF_EARG;
    if (L5 < 2 || L5 > 32) return MDWF_EARG;
    const long long V4 = (long long)Lx * Ly * Lz * Lt;
    if (V4 / 2 > 0x7fffffffLL / 32) return MDWF_EARG;     // L5 * Vh must fit comfortably in int
    mdwf_ctx *c = new mdwf_ctx();
    for (int d = 0; d < 4; d++) c->L[d] = L[d];
    c->L5 = L5;
    c->Vh = (int)(V4 / 2);
    c->M5 = M5; c->b5 = b5; c->c5 = c5; c->mf = m_f;
    c->alpha = b5 * (4.0 - M5) + 1.0;
    c->beta = c5 * (4.0 - M5) - 1.0;
    if (c->alpha == 0.0 || b5 == 0.0) { delete c; return MDWF_EARG; }   // A must be invertible; b5 is divided out on load
    *out = c;
    return MDWF_OK;
}

int mdwf_destroy(mdwf_ctx *c)
{
    if (!c) return MDWF_EARG;
    free_pool(c);
    for (int p = 0; p < 3; p++)
        for (int q = 0; q < 2; q++)
            if (c->gauge[p][q]) cudaFree(c->gauge[p][q]);
    for (int p = 0; p < 2; p++)
        for (int k = 0; k < DENSE_KINDS; k++)
            if (c->dense[p][k]) cudaFree(c->dense[p][k]);
    if (c->partial) cudaFree(c->partial);
    if (c->result_dev) cudaFree(c->result_dev);
    if (c->hop_partial) cudaFree(c->hop_partial);
    if (c->result_host) cudaFreeHost(c->result_host);
    for (cudaEvent_t e : c->hop_ev) cudaEventDestroy(e);
    if (c->sol_ready) cudaEventDestroy(c->sol_ready);
    if (c->copy_st) cudaStreamDestroy(c->copy_st);
    delete c;
    return MDWF_OK;
}

const char *mdwf_last_error(const mdwf_ctx *c) { return c ? c->err.c_str() : "null context"; }
int mdwf_flops_per_site(const mdwf_ctx *c) { return c ? 2880 + 48 * c->L5 : MDWF_EARG; }

int mdwf_set_option(mdwf_ctx *c, const char *key, const char *value)
{
    if (!c || !key || !value) return MDWF_EARG;
    const std::string k(key), v(value);
    if (k == "ladder") {
        if (v == "d") c->ladder = 0;
        else if (v == "ds") c->ladder = 1;
        else if (v == "dh") c->ladder = 2;
        else if (v == "dsh") c->ladder = 3;
        else { c->err = "ladder must be d|ds|dh|dsh"; return MDWF_EARG; }
    } else if (k == "apply_precision") {
        if (v == "auto") c->apply_prec = -1;
        else if (v == "fp64") c->apply_prec = PREC_D;
        else if (v == "fp32") c->apply_prec = PREC_S;
        else if (v == "half") c->apply_prec = PREC_H;
        else { c->err = "apply_precision must be auto|fp64|fp32|half"; return MDWF_EARG; }
    } else if (k == "reconstruct") {
        if (v == "18") c->recon_opt = 18;
        else if (v == "12") c->recon_opt = 12;
        else { c->err = "reconstruct must be 18|12"; return MDWF_EARG; }
    } else if (k == "reliable_delta") {
        const double d = atof(value);
        if (!(d > 0.0 && d < 1.0)) { c->err = "reliable_delta must be in (0,1)"; return MDWF_EARG; }
        c->delta = d;
    } else if (k == "time_hops") {
        c->time_hops = atoi(value) != 0;
    } else if (k == "max_update_interval") {
        c->max_update_interval = atoi(value);
    } else if (k == "kernels") {
        if (v == "auto") c->kver = 5; else if (v == "v5") c->kver = 6; else if (v == "v3") c->kver = 3; else if (v == "v2") c->kver = 2;
        else { c->err = "kernels must be auto|v2|v3|v5"; return MDWF_EARG; }
    } else if (k == "bp_stream") {
        c->use_bp = atoi(value);
    } else if (k == "release_workspace") {
        free_pool(c);                            // pooled work vectors are reallocated on demand
    } else if (k == "tile_l2_mb") {
        c->tile_l2_mb = atoi(value);
    } else if (k == "sweep_mb") {
        c->sweep_mb = atoi(value);
    } else if (k == "stream") {
        c->st = (cudaStream_t)(uintptr_t)strtoull(value, nullptr, 10);
    } else if (k == "matpc") {
        if (v == "asym") c->matpc_sym = 0; else if (v == "sym") c->matpc_sym = 1;
        else { c->err = "matpc must be asym|sym"; return MDWF_EARG; }
    } else {
        c->err = "unknown option " + k;
        return MDWF_EARG;
    }
    return MDWF_OK;
}

int mdwf_load_gauge(mdwf_ctx *c, const void *U_dev, int real_bytes)
{
    if (!c || !U_dev || (real_bytes != 8 && real_bytes != 4)) return MDWF_EARG;
    int ndev = 0;
    CUDA_OK(c, cudaGetDeviceCount(&ndev));
    const int recon = c->recon_opt;
    const bool had = c->gauge_loaded;
    c->gauge_loaded = false;                 // true again only after every step below has succeeded
    if (had && recon != c->recon) {
        for (int p = 0; p < 3; p++)
            for (int q = 0; q < 2; q++) { cudaFree(c->gauge[p][q]); c->gauge[p][q] = nullptr; }
    }
    for (int p = 0; p < 3; p++)
        for (int q = 0; q < 2; q++) {
            if (!c->gauge[p][q]) {
                CUDA_OK(c, cudaMalloc(&c->gauge[p][q], mdwf_gauge_bytes((Prec)p, c->Vh, recon)));
                CUDA_OK(c, cudaMemsetAsync(c->gauge[p][q], 0, mdwf_gauge_bytes((Prec)p, c->Vh, recon), c->st));   // padding lanes of a ragged last group
            }
            CUDA_OK(c, mdwf_launch_gauge_in((Prec)p, U_dev, real_bytes, c->gauge[p][q], c->L, q, recon, c->st));
            c->launches += 1;
        }
    c->recon = recon;
    // fifth-dimension tables in fp64 and fp32
    std::vector<double> tab[DENSE_KINDS];
    build_tables(c, tab);
    for (int k = 0; k < DENSE_KINDS; k++) {
        const size_t n = tab[k].size();
        std::vector<float> tf(n);
        for (size_t i = 0; i < n; i++) tf[i] = (float)tab[k][i];
        if (!c->dense[0][k]) CUDA_OK(c, cudaMalloc(&c->dense[0][k], n * sizeof(double)));
        if (!c->dense[1][k]) CUDA_OK(c, cudaMalloc(&c->dense[1][k], n * sizeof(float)));
        CUDA_OK(c, cudaMemcpy(c->dense[0][k], tab[k].data(), n * sizeof(double), cudaMemcpyHostToDevice));
        CUDA_OK(c, cudaMemcpy(c->dense[1][k], tf.data(), n * sizeof(float), cudaMemcpyHostToDevice));
    }
    CUDA_OK(c, cudaStreamSynchronize(c->st));
    c->gauge_loaded = true;
    return MDWF_OK;
}

int mdwf_load_gauge_host(mdwf_ctx *c, const void *U_host, int real_bytes)
{
    if (!c || !U_host || (real_bytes != 8 && real_bytes != 4)) return MDWF_EARG;
    const size_t bytes = (size_t)2 * c->Vh * 4 * 18 * real_bytes;
    void *tmp = nullptr;
    CUDA_OK(c, cudaMalloc(&tmp, bytes));
    cudaError_t e = cudaMemcpy(tmp, U_host, bytes, cudaMemcpyHostToDevice);
    int rc = MDWF_OK;
    if (e != cudaSuccess) { c->err = cudaGetErrorString(e); rc = MDWF_ECUDA; }
    else rc = mdwf_load_gauge(c, tmp, real_bytes);
    cudaFree(tmp);
    return rc;
}

// ---- NEXT-2: Mpc / Mpc^dagger on a batch of right-hand sides (hop3b_kernels.cuh) -----------------------------------------
// A batch is one spinor array over nrhs * Vp sites (Vp = Vh rounded up to 32): right-hand side r is the single-vector layout at
// byte offset r * mdwf_spinor_bytes.
static int get_spinor_batch(mdwf_ctx *c, const std::string &name, Prec p, int nrhs, SpinorBuf *out)
{
    const std::string key = name + ".x" + std::to_string(nrhs) + (p == PREC_D ? ".d" : p == PREC_S ? ".s" : ".h");
    auto it = c->pool.find(key);
    if (it != c->pool.end()) { *out = it->second; return MDWF_OK; }
    SpinorBuf b;
    CUDA_OK(c, cudaMalloc(&b.v, (size_t)nrhs * mdwf_spinor_bytes(p, c->L5, c->Vh)));
    if (p == PREC_H) CUDA_OK(c, cudaMalloc((void **)&b.norm, sizeof(float) * (size_t)nrhs * c->L5 * ((c->Vh + 31) / 32 * 32)));
    c->pool[key] = b;
    *out = b;
    return MDWF_OK;
}
static SpinorBuf batch_view(const mdwf_ctx *c, Prec p, const SpinorBuf &b, int r)
{
    SpinorBuf v = b;
    v.v = (char *)b.v + (size_t)r * mdwf_spinor_bytes(p, c->L5, c->Vh);
    if (b.norm) v.norm = b.norm + (size_t)r * c->L5 * ((c->Vh + 31) / 32 * 32);
    return v;
}
static int run_hop_batch(mdwf_ctx *c, Prec p, int nrhs, int dag, int pre, int post, int own, HopArgs a)
{
    a.kver = 3;
    a.nrhs = nrhs;
    a.batch_sites = (c->Vh + 31) / 32 * 32;
    if (post == 1) fill_recurrence(c, a, c->b5, c->c5);
    const int rc = mdwf_launch_hop_batch(p, dag, pre, post, own, a, c->st);
    if (rc == -1) { c->err = "batched kernels: fp32 / 16-bit storage, L5 in {8, 12, 16}, |beta/alpha| < 0.98 only"; return MDWF_EARG; }
    CUDA_OK(c, rc);
    c->launches += 1;
    return MDWF_OK;
}
struct SweepRhs {            // base_args sizes the sweep slab for nrhs vectors while one of these is alive
    mdwf_ctx *c;
    SweepRhs(mdwf_ctx *c_, int nrhs) : c(c_) { c->sweep_rhs = nrhs; }
    ~SweepRhs() { c->sweep_rhs = 1; }
};
static int op_Mpc_batch(mdwf_ctx *c, Prec p, int nrhs, const SpinorBuf &in, const SpinorBuf &tmp, const SpinorBuf &out)
{
    SweepRhs guard(c, nrhs);
    HopArgs k1 = base_args(c, p, 0, in, nullptr, tmp);        // K1: t_e = (B A^{-1}) H_eo (B in_o), every right-hand side
    k1.coef_hop = c->b5; k1.pre_d = c->b5; k1.pre_o = c->c5;
    TRY(run_hop_batch(c, p, nrhs, 0, 1, 1, 0, k1));
    HopArgs k2 = base_args(c, p, 1, tmp, &in, out);           // K2: out_o = A in_o - (1/4) H_oe t_e
    k2.coef_hop = -0.25; k2.own_d = c->alpha; k2.own_o = c->beta;
    return run_hop_batch(c, p, nrhs, 0, 0, 0, 2, k2);
}
static int op_Mpcdag_batch(mdwf_ctx *c, Prec p, int nrhs, const SpinorBuf &in, const SpinorBuf &tmp, const SpinorBuf &out)
{
    SweepRhs guard(c, nrhs);
    HopArgs k1 = base_args(c, p, 0, in, nullptr, tmp);        // K1+: u_e = (A^{-+} B^+) H'_eo in_o
    k1.coef_hop = 1.0;
    TRY(run_hop_batch(c, p, nrhs, 1, 0, 1, 0, k1));
    HopArgs k2 = base_args(c, p, 1, tmp, &in, out);           // K2+: out_o = A^+ in_o - (1/4) B^+ H'_oe u_e
    k2.coef_hop = -0.25; k2.post_d = c->b5; k2.post_o = c->c5; k2.own_d = c->alpha; k2.own_o = c->beta;
    return run_hop_batch(c, p, nrhs, 1, 0, 2, 3, k2);
}
int mdwf_apply_batch(mdwf_ctx *c, int op, int nrhs, const void *in_dev, void *out_dev, int real_bytes)
{
    TRY(check_ready(c));
    if (!in_dev || !out_dev || in_dev == out_dev || (real_bytes != 8 && real_bytes != 4) || nrhs < 1 || nrhs > 64 ||
        (op != MDWF_OP_MPC && op != MDWF_OP_MPCDAG)) {
        c->err = "mdwf_apply_batch: bad argument (op must be Mpc or Mpc^dagger, 1 <= nrhs <= 64)";
        return MDWF_EARG;
    }
    const Prec p = c->apply_prec >= 0 ? (Prec)c->apply_prec : PREC_S;
    if (p == PREC_D) { c->err = "mdwf_apply_batch: fp32 or 16-bit apply_precision only"; return MDWF_EARG; }
    SpinorBuf a, b, t;
    TRY(get_spinor_batch(c, "bt.a", p, nrhs, &a));
    TRY(get_spinor_batch(c, "bt.b", p, nrhs, &b));
    TRY(get_spinor_batch(c, "bt.t", p, nrhs, &t));
    const size_t vec = (size_t)c->Vh * c->L5 * 24 * real_bytes;              // one parity vector of the caller
    for (int r = 0; r < nrhs; r++)
        CUDA_OK(c, mdwf_launch_parity_in(p, (const char *)in_dev + r * vec, real_bytes, batch_view(c, p, a, r), c->L5, c->Vh, c->st));
    if (op == MDWF_OP_MPC) TRY(op_Mpc_batch(c, p, nrhs, a, t, b));
    else TRY(op_Mpcdag_batch(c, p, nrhs, a, t, b));
    for (int r = 0; r < nrhs; r++)
        CUDA_OK(c, mdwf_launch_parity_out(p, batch_view(c, p, b, r), (char *)out_dev + r * vec, real_bytes, c->L5, c->Vh, c->st));
    c->launches += 2 * nrhs;
    CUDA_OK(c, cudaStreamSynchronize(c->st));
    return MDWF_OK;
}

int mdwf_apply(mdwf_ctx *c, int op, const void *in_dev, void *out_dev, int real_bytes)
{
    TRY(check_ready(c));
    if (!in_dev || !out_dev || in_dev == out_dev || (real_bytes != 8 && real_bytes != 4) || op < 0 || op > MDWF_OP_MPCDAG_SYM) {
        c->err = "mdwf_apply: bad argument";
        return MDWF_EARG;
    }
    const Prec p = c->apply_prec >= 0 ? (Prec)c->apply_prec : (real_bytes == 8 ? PREC_D : PREC_S);
    SpinorBuf a, b, t, u;
    TRY(get_spinor(c, "ap.a", p, &a));
    TRY(get_spinor(c, "ap.b", p, &b));
    TRY(get_spinor(c, "ap.t", p, &t));
    if (op <= MDWF_OP_MDAGM || op == MDWF_OP_MPC_SYM || op == MDWF_OP_MPCDAG_SYM) {
        CUDA_OK(c, mdwf_launch_parity_in(p, in_dev, real_bytes, a, c->L5, c->Vh, c->st));
        if (op == MDWF_OP_MPC) TRY(op_Mpc(c, p, a, t, b));
        else if (op == MDWF_OP_MPCDAG) TRY(op_Mpcdag(c, p, a, t, b));
        else if (op == MDWF_OP_MPC_SYM) TRY(op_Mpc_sym(c, p, a, t, b));
        else if (op == MDWF_OP_MPCDAG_SYM) { TRY(get_spinor(c, "ap.u", p, &u)); TRY(op_Mpcdag_sym(c, p, a, u, t, b)); }
        else {
            TRY(get_spinor(c, "ap.u", p, &u));
            TRY(op_Mpc(c, p, a, t, u));
            TRY(op_Mpcdag(c, p, u, t, b));
        }
        CUDA_OK(c, mdwf_launch_parity_out(p, b, out_dev, real_bytes, c->L5, c->Vh, c->st));
        c->launches += 2;
    } else {
        // a = even part, b = odd part of the input; t / u = even / odd part of the output
        TRY(get_spinor(c, "ap.u", p, &u));
        CUDA_OK(c, mdwf_launch_full_in(p, in_dev, real_bytes, a, c->L, c->L5, 0, c->st));
        CUDA_OK(c, mdwf_launch_full_in(p, in_dev, real_bytes, b, c->L, c->L5, 1, c->st));
        if (op == MDWF_OP_D) {
            TRY(op_D_parity(c, p, 0, b, a, t));
            TRY(op_D_parity(c, p, 1, a, b, u));
        } else {
            TRY(op_Ddag_parity(c, p, 0, b, a, t));
            TRY(op_Ddag_parity(c, p, 1, a, b, u));
        }
        CUDA_OK(c, mdwf_launch_full_out(p, t, out_dev, real_bytes, c->L, c->L5, 0, c->st));
        CUDA_OK(c, mdwf_launch_full_out(p, u, out_dev, real_bytes, c->L, c->L5, 1, c->st));
        c->launches += 4;
    }
    CUDA_OK(c, cudaStreamSynchronize(c->st));
    return MDWF_OK;
}

// ---- S8-S10: Schur preparation, CG on the normal equations with reliable updates, reconstruction -------
static int solve_device(mdwf_ctx *c, const void *src_dev, void *sol_dev, double tol, int maxiter, int *iters_out,
                        double *true_res_out)
{
    const Prec PDd = PREC_D;
    const Prec ps = (c->ladder == 0) ? PREC_D : (c->ladder == 1 ? PREC_S : PREC_H);   // sloppy operator / Krylov vectors
    const Prec pxl = (c->ladder == 0) ? PREC_D : (c->ladder == 2 ? PREC_H : PREC_S);  // sloppy solution accumulator
    SpinorBuf be, bo, bp, xhi, rhi, te;
    TRY(get_spinor(c, "sv.be", PDd, &be));
    TRY(get_spinor(c, "sv.bo", PDd, &bo));
    TRY(get_spinor(c, "sv.bp", PDd, &bp));
    TRY(get_spinor(c, "sv.xhi", PDd, &xhi));
    TRY(get_spinor(c, "sv.rhi", PDd, &rhi));
    TRY(get_spinor(c, "sv.te", PDd, &te));
    SpinorBuf rs, g, p, q, ts, xlo;
    TRY(get_spinor(c, "sv.rs", ps, &rs));
    TRY(get_spinor(c, "sv.g", ps, &g));
    TRY(get_spinor(c, "sv.p", ps, &p));
    TRY(get_spinor(c, "sv.q", ps, &q));
    TRY(get_spinor(c, "sv.ts", ps, &ts));
    TRY(get_spinor(c, "sv.xlo", pxl, &xlo));
    // 16-bit Krylov vectors: the CG update also writes B p, and p is double-buffered
    const bool sym = c->matpc_sym != 0;                 // NEXT-1: iterate on Mpc_sym x_o = A^{-1} b'_o
    const bool use_bp = (ps == PREC_H) && bp_stream_available(c, ps) && c->use_bp && !sym;
    SpinorBuf p2, bpv, ws;
    if (use_bp) { TRY(get_spinor(c, "sv.p2", ps, &p2)); TRY(get_spinor(c, "sv.bp", ps, &bpv)); }
    if (sym) TRY(get_spinor(c, "sv.ws", ps, &ws));      // A^{-+} r of Mpc_sym^+
    // the Schur operator of the iteration and its adjoint in precision pr
    auto opM = [&](Prec pr, const SpinorBuf &in, const SpinorBuf &tmp, const SpinorBuf &out, double *n2) -> int {
        return sym ? op_Mpc_sym(c, pr, in, tmp, out, n2) : op_Mpc(c, pr, in, tmp, out, n2);
    };
    auto opMdag = [&](Prec pr, const SpinorBuf &in, const SpinorBuf &tmp, const SpinorBuf &out, double *n2) -> int {
        return sym ? op_Mpcdag_sym(c, pr, in, ws, tmp, out, n2) : op_Mpcdag(c, pr, in, tmp, out, n2);
    };

    c->iterations = 0; c->reliable_updates = 0; c->op_applications = 0; c->sloppy_applications = 0;

    // S0: canonical full 5D source -> even / odd device vectors (fp64)
    CUDA_OK(c, mdwf_launch_full_in(PDd, src_dev, 8, be, c->L, c->L5, 0, c->st));
    CUDA_OK(c, mdwf_launch_full_in(PDd, src_dev, 8, bo, c->L, c->L5, 1, c->st));
    c->launches += 2;
    double be2 = 0, bo2 = 0;
    TRY(v_norm2(c, PDd, be, &be2));
    TRY(v_norm2(c, PDd, bo, &bo2));
    const double bnorm = std::sqrt(be2 + bo2);
    if (bnorm == 0.0) {
        CUDA_OK(c, cudaMemsetAsync(sol_dev, 0, (size_t)2 * c->Vh * c->L5 * 24 * 8, c->st));
        CUDA_OK(c, cudaStreamSynchronize(c->st));
        if (iters_out) *iters_out = 0;
        if (true_res_out) *true_res_out = 0.0;
        return MDWF_OK;
    }
    // S10: b'_o = b_o - D_oe A^{-1} b_e
    TRY(op_Ainv(c, PDd, be, rhi));
    TRY(op_schur_hop(c, PDd, 1, rhi, bo, bp));
    // ||b - D x|| = ||b' - Mpc x_o|| once x_e is reconstructed, so the CG target is absolute: tol * ||b||
    double target = tol * bnorm;
    if (sym) {
        // right-hand side A^{-1} b'; the residual rho of the symmetric system gives b' - Mpc x_o = A rho, ||A rho|| <= (|alpha| + |beta|) ||rho||
        TRY(op_Ainv(c, PDd, bp, te));
        TRY(v_axpby(c, PDd, bp, 1.0, PDd, te, 0.0, PDd, nullptr, nullptr));
        target /= (std::fabs(c->alpha) + std::fabs(c->beta));
    }

    TRY(v_zero(c, PDd, xhi));
    TRY(v_zero(c, pxl, xlo));
    double r2 = 0;
    TRY(v_axpby(c, PDd, rhi, 1.0, PDd, bp, 0.0, PDd, nullptr, &r2));        // r_hi = b'
    double rn = std::sqrt(r2), rmax = rn;
    bool converged = rn <= target;
    int k = 0, since_update = 0;
    if (!converged) {
        TRY(v_axpby(c, ps, rs, 1.0, PDd, rhi, 0.0, PDd, nullptr, nullptr)); // r_s = convert(r_hi)
        TRY(opMdag(ps, rs, ts, g, nullptr));                                // g = Mpc^+ r
        double gam = 0;
        SpinorBuf pc = p, pn = p2;                                          // current / next direction vector (use_bp)
        // fused update; with use_bp it also writes B p_new and flips the double buffer of p
        // With the double buffer of p (use_bp) the x update runs every other iteration: x_lo is the widest vector of the
        // update (fp32 in the dsh ladder: 3.6 of its 7.5 GB), and the direction of the iteration before is still in the buffer
        // the new p is about to overwrite.  x_pending = 1: alpha_k p_k has not been added yet (p_k = pn after the swap).
        int x_pending = 0;
        auto cg_update = [&](double ax, double bx) -> int {
            if (use_bp) {
                const int xmode = (ax == 0.0) ? 0 : (x_pending ? 2 : 0);
                CUDA_OK(c, mdwf_launch_xpupdate_b(pxl, xlo, ax, pc, bx, g, pn, bpv, c->b5, c->c5, c->mf, c->L5, c->Vh, c->st, xmode));
                if (ax != 0.0) x_pending = !x_pending;
                std::swap(pc, pn);
            } else {
                CUDA_OK(c, mdwf_launch_xpupdate(pxl, xlo, ax, ps, pc, bx, g, c->L5, c->Vh, c->st));
            }
            c->launches += 1;
            return MDWF_OK;
        };
        auto apply_Mpc = [&](double *qq) -> int {                           // q = Mpc p, ||q||^2 from the K2 epilogue
            if (!use_bp) return opM(ps, pc, ts, q, qq);
            TRY(op_Mpc_k1_from_B(c, ps, bpv, ts));
            TRY(op_Mpc_k2(c, ps, pc, ts, q, qq));
            c->op_applications += 1;
            c->sloppy_applications += 1;
            return MDWF_OK;
        };
        // The scalars of the iteration stay on the device (result_dev: [1] gamma, [2] ||q||^2, [3] ||r||^2, [4] gamma', [5..8] the
        // coefficient pairs the BLAS kernels read): alpha and beta are formed by a one-thread kernel, and the host reads back ONE
        // number per iteration, ||r||^2, for the convergence / reliable-update decision, after it has queued the rest of the
        // iteration (Mpc^+ r and the x / p update), so the device never waits for it.
        double *S = c->result_dev, dummy = 0;
        cudaEvent_t ev;
        CUDA_OK(c, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
        struct EvGuard { cudaEvent_t e; mdwf_ctx *c; ~EvGuard() { cudaEventDestroy(e); c->defer_slot = -1; mdwf_blas_set_coef(nullptr); } } guard{ev, c};
        (void)gam;
        c->defer_slot = 1;                                                  // gamma = ||g||^2
        if (use_bp) {
            TRY(v_norm2(c, ps, g, &dummy));
            c->defer_slot = -1;
            TRY(v_zero(c, ps, pc));
            TRY(cg_update(0.0, 0.0));                                       // p = g, B p
        } else {
            TRY(v_axpby(c, ps, pc, 1.0, ps, g, 0.0, ps, nullptr, &dummy));  // p = g
            c->defer_slot = -1;
        }
        // the pending term of the deferred x update: x_lo += alpha_k p_k (alpha_k = S[5], p_k = the buffer the update just left)
        auto flush_x = [&]() -> int {
            if (!x_pending) return MDWF_OK;
            mdwf_blas_set_coef(S + 5);
            const int rc = v_axpby(c, pxl, xlo, 1.0, ps, pn, 1.0, pxl, &xlo, nullptr);
            mdwf_blas_set_coef(nullptr);
            x_pending = 0;
            return rc;
        };
        while (k < maxiter && !converged) {
            c->defer_slot = 2;
            TRY(apply_Mpc(&dummy));                                         // q = Mpc p, ||q||^2
            CUDA_OK(c, mdwf_launch_cg_scalars(S, 0, c->st));                // alpha = gamma / ||q||^2
            c->defer_slot = 3;
            mdwf_blas_set_coef(S + 5);
            TRY(v_axpby(c, ps, rs, -1.0, ps, q, 1.0, ps, &rs, &dummy));     // r -= alpha q, ||r||^2
            mdwf_blas_set_coef(nullptr);
            CUDA_OK(c, cudaMemcpyAsync(c->result_host + 1, S + 3, sizeof(double), cudaMemcpyDeviceToHost, c->st));
            CUDA_OK(c, cudaEventRecord(ev, c->st));
            c->defer_slot = 4;
            TRY(opMdag(ps, rs, ts, g, &dummy));                             // g = Mpc^+ r, gamma' = ||g||^2
            c->defer_slot = -1;
            CUDA_OK(c, mdwf_launch_cg_scalars(S, 1, c->st));                // beta = gamma' / gamma, gamma = gamma'
            mdwf_blas_set_coef(S + 7);
            TRY(cg_update(1.0, 1.0));                                       // x_lo += alpha p ; p = g + beta p
            mdwf_blas_set_coef(nullptr);
            c->launches += 2;
            CUDA_OK(c, cudaEventSynchronize(ev));
            r2 = c->result_host[1];
            k++; since_update++;
            if (!(r2 == r2) || !(r2 >= 0.0)) break;                         // breakdown (gamma or ||q||^2 vanished)
            rn = std::sqrt(r2);
            const bool update = (rn < c->delta * rmax) || (rn <= target) ||
                                (c->max_update_interval > 0 && since_update >= c->max_update_interval);
            if (update) {
                // reliable update: fold x_lo into x_hi, recompute the residual in fp64 and restart the sloppy residual from it
                TRY(flush_x());
                TRY(v_axpby(c, PDd, xhi, 1.0, pxl, xlo, 1.0, PDd, &xhi, nullptr));
                TRY(v_zero(c, pxl, xlo));
                TRY(opM(PDd, xhi, te, rhi, nullptr));
                TRY(v_axpby(c, PDd, rhi, 1.0, PDd, bp, -1.0, PDd, &rhi, &r2));   // r_hi = b' - M x_hi
                rn = std::sqrt(r2);
                c->reliable_updates += 1;
                since_update = 0;
                if (rn <= target) { converged = true; break; }
                TRY(v_axpby(c, ps, rs, 1.0, PDd, rhi, 0.0, PDd, nullptr, nullptr));
                rmax = rn;
                // the search direction p_{k+1} = g_{k+1} + beta p_k is already built (from the recursive residual, which the true
                // one replaces to within the sloppy rounding): keep it, and take gamma from the true residual
                c->defer_slot = 1;
                TRY(opMdag(ps, rs, ts, g, &dummy));                         // g = Mpc^+ r, gamma = ||g||^2
                c->defer_slot = -1;
            }
        }
        if (!converged) {   // fold what we have
            TRY(flush_x());
            TRY(v_axpby(c, PDd, xhi, 1.0, pxl, xlo, 1.0, PDd, &xhi, nullptr));
        }
    }
    c->iterations = k;
    // S10: x_e = A^{-1} (b_e - D_eo x_o)
    TRY(op_schur_hop(c, PDd, 0, xhi, be, te));
    TRY(op_Ainv(c, PDd, te, rhi));                                          // rhi now holds x_e
    CUDA_OK(c, mdwf_launch_full_out(PDd, rhi, sol_dev, 8, c->L, c->L5, 0, c->st));
    CUDA_OK(c, mdwf_launch_full_out(PDd, xhi, sol_dev, 8, c->L, c->L5, 1, c->st));
    c->launches += 2;
    if (c->d2h_dst && c->copy_st && c->sol_ready) {         // host-buffer solve: copy out while the true residual is computed
        CUDA_OK(c, cudaEventRecord(c->sol_ready, c->st));
        CUDA_OK(c, cudaStreamWaitEvent(c->copy_st, c->sol_ready, 0));
        CUDA_OK(c, cudaMemcpyAsync(c->d2h_dst, sol_dev, c->d2h_bytes, cudaMemcpyDeviceToHost, c->copy_st));
        c->d2h_issued = true;
    }
    // true residual with the unpreconditioned operator, fp64: || b - D x || / || b ||
    TRY(op_D_parity(c, PDd, 0, xhi, rhi, te));
    TRY(op_D_parity(c, PDd, 1, rhi, xhi, bp));
    double re2 = 0, ro2 = 0;
    TRY(v_axpby(c, PDd, te, 1.0, PDd, be, -1.0, PDd, &te, &re2));
    TRY(v_axpby(c, PDd, bp, 1.0, PDd, bo, -1.0, PDd, &bp, &ro2));
    const double tr = std::sqrt(re2 + ro2) / bnorm;
    c->true_residual = tr;
    if (iters_out) *iters_out = k;
    if (true_res_out) *true_res_out = tr;
    if (!(tr <= tol * 1.001)) {              // the header's contract: tol is the target for ||src - D x|| / ||src||
        c->err = converged ? "CG converged on the Schur system but the recomputed full residual exceeds tol"
                           : "CG did not converge within maxiter";
        return MDWF_ENOCONV;
    }
    return MDWF_OK;
}

int mdwf_solve(mdwf_ctx *c, const void *src_dev, void *sol_dev, double tol, int maxiter, int *iters_out,
               double *true_res_out)
{
    TRY(check_ready(c));
    if (!src_dev || !sol_dev || src_dev == sol_dev || !(tol > 0.0) || maxiter < 0) { c->err = "mdwf_solve: bad argument"; return MDWF_EARG; }
    cudaEvent_t e0, e1;
    CUDA_OK(c, cudaEventCreate(&e0));
    if (cudaEventCreate(&e1) != cudaSuccess) { cudaEventDestroy(e0); c->err = "cudaEventCreate"; return MDWF_ECUDA; }
    if (cudaEventRecord(e0, c->st) != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); c->err = "cudaEventRecord"; return MDWF_ECUDA; }
    c->hop_ev_tag.clear();
    if (c->time_hops) c->hop_time_prec = (c->ladder == 0) ? (int)PREC_D : (c->ladder == 1 ? (int)PREC_S : (int)PREC_H);
    const int rc = solve_device(c, src_dev, sol_dev, tol, maxiter, iters_out, true_res_out);
    c->hop_time_prec = -1;
    cudaEventRecord(e1, c->st);
    cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    c->solve_seconds = ms * 1e-3;
    for (int t = 0; t < 4; t++) { c->hop_ms[t] = 0; c->hop_n[t] = 0; }
    for (size_t k = 0; k < c->hop_ev_tag.size(); k++) {
        float hm = 0.f;
        if (cudaEventElapsedTime(&hm, c->hop_ev[2 * k], c->hop_ev[2 * k + 1]) == cudaSuccess) {
            c->hop_ms[c->hop_ev_tag[k]] += hm;
            c->hop_n[c->hop_ev_tag[k]] += 1;
        }
    }
    c->hop_ev_tag.clear();
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return rc;
}

int mdwf_solve_host(mdwf_ctx *c, const void *src_host, void *sol_host, double tol, int maxiter, int *iters_out,
                    double *true_res_out)
{
    TRY(check_ready(c));
    if (!src_host || !sol_host) return MDWF_EARG;
    const size_t bytes = (size_t)2 * c->Vh * c->L5 * 24 * 8;
    void *src = nullptr, *sol = nullptr;
    TRY(get_raw(c, "host.src", bytes, &src));
    TRY(get_raw(c, "host.sol", bytes, &sol));
    if (!c->copy_st) CUDA_OK(c, cudaStreamCreateWithFlags(&c->copy_st, cudaStreamNonBlocking));
    if (!c->sol_ready) CUDA_OK(c, cudaEventCreateWithFlags(&c->sol_ready, cudaEventDisableTiming));
    CUDA_OK(c, cudaMemcpyAsync(src, src_host, bytes, cudaMemcpyHostToDevice, c->st));
    c->d2h_dst = sol_host; c->d2h_bytes = bytes; c->d2h_issued = false;
    const int rc = mdwf_solve(c, src, sol, tol, maxiter, iters_out, true_res_out);
    const bool issued = c->d2h_issued;
    c->d2h_dst = nullptr; c->d2h_issued = false;
    if (issued) CUDA_OK(c, cudaStreamSynchronize(c->copy_st));        // never return with a copy into the caller's buffer in flight
    if (rc != MDWF_OK && rc != MDWF_ENOCONV) return rc;
    if (!issued) CUDA_OK(c, cudaMemcpyAsync(sol_host, sol, bytes, cudaMemcpyDeviceToHost, c->st));
    CUDA_OK(c, cudaStreamSynchronize(c->st));
    return rc;
}

// ---- NEXT-3: 4D <-> 5D maps (Eq. (5)) ------------------------------------------------------------------
int mdwf_wall_source(mdwf_ctx *c, const void *eta_dev, void *src_dev, int real_bytes, int lift)
{
    if (!c || !eta_dev || !src_dev || eta_dev == src_dev || (real_bytes != 8 && real_bytes != 4)) return MDWF_EARG;
    const long V4 = 2L * c->Vh;
    if (!lift) {
        CUDA_OK(c, mdwf_launch_wall_inject(eta_dev, src_dev, real_bytes, V4, c->L5, c->st));
        c->launches += 1;
        CUDA_OK(c, cudaStreamSynchronize(c->st));
        return MDWF_OK;
    }
    // D_- b = (c5 D_W - 1) b = beta b - (c5/2) H b, slice by slice, in fp64: per parity one hop launch with the own-site term beta b
    TRY(check_ready(c));
    void *w = nullptr;
    TRY(get_raw(c, "map.w", (size_t)c->L5 * V4 * 24 * real_bytes, &w));
    CUDA_OK(c, mdwf_launch_wall_inject(eta_dev, w, real_bytes, V4, c->L5, c->st));
    SpinorBuf e, o, te, to;
    TRY(get_spinor(c, "ap.a", PREC_D, &e));
    TRY(get_spinor(c, "ap.b", PREC_D, &o));
    TRY(get_spinor(c, "ap.t", PREC_D, &te));
    TRY(get_spinor(c, "ap.u", PREC_D, &to));
    CUDA_OK(c, mdwf_launch_full_in(PREC_D, w, real_bytes, e, c->L, c->L5, 0, c->st));
    CUDA_OK(c, mdwf_launch_full_in(PREC_D, w, real_bytes, o, c->L, c->L5, 1, c->st));
    for (int parity = 0; parity < 2; parity++) {
        HopArgs a = base_args(c, PREC_D, parity, parity ? e : o, parity ? &o : &e, parity ? to : te);
        a.coef_hop = -0.5 * c->c5; a.own_d = c->beta; a.own_o = 0.0;
        TRY(run_hop(c, PREC_D, 0, 0, 0, 2, a));
    }
    CUDA_OK(c, mdwf_launch_full_out(PREC_D, te, src_dev, real_bytes, c->L, c->L5, 0, c->st));
    CUDA_OK(c, mdwf_launch_full_out(PREC_D, to, src_dev, real_bytes, c->L, c->L5, 1, c->st));
    c->launches += 5;
    CUDA_OK(c, cudaStreamSynchronize(c->st));
    return MDWF_OK;
}
int mdwf_wall_project(mdwf_ctx *c, const void *psi_dev, void *q_dev, int real_bytes, int midpoint)
{
    if (!c || !psi_dev || !q_dev || psi_dev == q_dev || (real_bytes != 8 && real_bytes != 4)) return MDWF_EARG;
    const int sm = midpoint ? c->L5 / 2 : 0, sp = midpoint ? c->L5 / 2 - 1 : c->L5 - 1;
    CUDA_OK(c, mdwf_launch_wall_project(psi_dev, q_dev, real_bytes, 2L * c->Vh, sm, sp, c->st));
    c->launches += 1;
    CUDA_OK(c, cudaStreamSynchronize(c->st));
    return MDWF_OK;
}

// ---- NEXT-4: gradient-flow smearing of the gauge field (Sec. III; App. D) ------------------
int mdwf_plaquette(mdwf_ctx *c, const void *U_dev, double *out)
{
    if (!c || !U_dev || !out) return MDWF_EARG;
    const long V4 = 2L * c->Vh;
    const int nb = mdwf_flow_plaquette_blocks(V4);
    void *part = nullptr;
    TRY(get_raw(c, "flow.part", sizeof(double) * (size_t)nb, &part));
    TRY(ensure_scalars(c));
    CUDA_OK(c, mdwf_launch_plaquette(U_dev, c->L, (double *)part, c->st));
    CUDA_OK(c, mdwf_launch_final_sum((double *)part, nb, c->result_dev, c->st));
    c->launches += 2;
    double s = 0;
    TRY(fetch_scalar(c, &s));
    *out = s / (18.0 * (double)V4);                  // <Re tr P> / 3 over the 6 planes
    return MDWF_OK;
}
int mdwf_gradient_flow(mdwf_ctx *c, void *U_dev, double eps, int nsteps, int action, double *plaq_out)
{
    if (!c || !U_dev || !(eps > 0.0) || nsteps < 0 || action < 0 || action > 1) return MDWF_EARG;
    const long V4 = 2L * c->Vh;
    void *Z = nullptr;
    TRY(get_raw(c, "flow.z", (size_t)V4 * 4 * 18 * sizeof(double), &Z));
    const double c0 = action ? 5.0 / 3.0 : 1.0, c1 = action ? -1.0 / 12.0 : 0.0;
    for (int k = 0; k < nsteps; k++) {
        CUDA_OK(c, mdwf_launch_flow_step(U_dev, Z, c->L, eps, c0, c1, c->st));
        c->launches += 6;
    }
    if (plaq_out) return mdwf_plaquette(c, U_dev, plaq_out);
    CUDA_OK(c, cudaStreamSynchronize(c->st));
    return MDWF_OK;
}

// ---- the 16-bit storage format, as stored (bit-exact tests of the quantiser) ------------------------------------------
int mdwf_half_encode(mdwf_ctx *c, const void *in_dev, int real_bytes, int via_fp64, void *words_dev, void *scales_dev)
{
    if (!c || !in_dev || !words_dev || !scales_dev || (real_bytes != 8 && real_bytes != 4)) return MDWF_EARG;
    SpinorBuf h, d;
    TRY(get_spinor(c, "hf.h", PREC_H, &h));
    if (via_fp64) {     // the path of the solver: fp64 device vector -> 16-bit by the BLAS-1 copy
        TRY(get_spinor(c, "hf.d", PREC_D, &d));
        CUDA_OK(c, mdwf_launch_parity_in(PREC_D, in_dev, real_bytes, d, c->L5, c->Vh, c->st));
        c->launches += 1;
        TRY(v_axpby(c, PREC_H, h, 1.0, PREC_D, d, 0.0, PREC_D, nullptr, nullptr));
    } else {            // the path of mdwf_apply: canonical buffer -> 16-bit by the layout kernel
        CUDA_OK(c, mdwf_launch_parity_in(PREC_H, in_dev, real_bytes, h, c->L5, c->Vh, c->st));
        c->launches += 1;
    }
    CUDA_OK(c, mdwf_launch_half_export(h, words_dev, scales_dev, c->L5, c->Vh, c->st));
    c->launches += 1;
    CUDA_OK(c, cudaStreamSynchronize(c->st));
    return MDWF_OK;
}
int mdwf_half_decode(mdwf_ctx *c, const void *words_dev, const void *scales_dev, void *out_dev, int real_bytes)
{
    if (!c || !out_dev || !words_dev || !scales_dev || (real_bytes != 8 && real_bytes != 4)) return MDWF_EARG;
    SpinorBuf h;
    TRY(get_spinor(c, "hf.h", PREC_H, &h));
    CUDA_OK(c, mdwf_launch_half_import(words_dev, scales_dev, h, c->L5, c->Vh, c->st));
    CUDA_OK(c, mdwf_launch_parity_out(PREC_H, h, out_dev, real_bytes, c->L5, c->Vh, c->st));
    c->launches += 2;
    CUDA_OK(c, cudaStreamSynchronize(c->st));
    return MDWF_OK;
}

// ---- S7 entry points on flat arrays ---------------------------------------------------------------------
int mdwf_blas_norm2(mdwf_ctx *c, const void *x, long long n, int real_bytes, double *out)
{
    if (!c || !x || !out || n < 0 || (real_bytes != 8 && real_bytes != 4)) return MDWF_EARG;
    TRY(ensure_scalars(c));
    CUDA_OK(c, mdwf_launch_flat_reduce(0, x, x, n, real_bytes, c->partial, c->result_dev, c->st));
    c->launches += 2;
    return fetch_scalar(c, out);
}
int mdwf_blas_redot(mdwf_ctx *c, const void *x, const void *y, long long n, int real_bytes, double *out)
{
    if (!c || !x || !y || !out || n < 0 || (real_bytes != 8 && real_bytes != 4)) return MDWF_EARG;
    TRY(ensure_scalars(c));
    CUDA_OK(c, mdwf_launch_flat_reduce(1, x, y, n, real_bytes, c->partial, c->result_dev, c->st));
    c->launches += 2;
    return fetch_scalar(c, out);
}
int mdwf_blas_axpy(mdwf_ctx *c, double a, const void *x, void *y, long long n, int real_bytes)
{
    if (!c || !x || !y || n < 0 || (real_bytes != 8 && real_bytes != 4)) return MDWF_EARG;
    CUDA_OK(c, mdwf_launch_flat_axpy(a, x, y, n, real_bytes, c->st));
    c->launches += 1;
    return MDWF_OK;
}

int mdwf_get_stat(const mdwf_ctx *c, const char *key, double *value)
{
    if (!c || !key || !value) return MDWF_EARG;
    const std::string k(key);
    if (k == "launches") *value = c->launches;
    else if (k == "iterations") *value = c->iterations;
    else if (k == "reliable_updates") *value = c->reliable_updates;
    else if (k == "solve_seconds") *value = c->solve_seconds;
    else if (k == "true_residual") *value = c->true_residual;
    else if (k == "op_applications") *value = c->op_applications;
    else if (k == "sloppy_applications") *value = c->sloppy_applications;
    else if (k.rfind("hop_ms_", 0) == 0 || k.rfind("hop_n_", 0) == 0) {     // option time_hops: average ms / count of the last solve
        const bool ms = k[4] == 'm';
        const std::string t = k.substr(ms ? 7 : 6);
        const int tag = t == "k1" ? 0 : (t == "k2" ? 1 : (t == "k1dag" ? 2 : (t == "k2dag" ? 3 : -1)));
        if (tag < 0) return MDWF_EARG;
        *value = ms ? (c->hop_n[tag] > 0 ? c->hop_ms[tag] / c->hop_n[tag] : 0.0) : c->hop_n[tag];
    }
    else return MDWF_EARG;
    return MDWF_OK;
}

}   // extern "C"

// measurement entry points (include/mdwf_bench.h): not part of the solver boundary
#include "mdwf_bench_api.inc"
