// hop_kernels.cuh -- the fused Wilson-hopping + fifth-dimension kernel family (S1-S6 of the hot path).
//
// One launch computes, for every site x of one 4D parity and every s:
//     r(x,s)   = coef_hop * sum_mu [ (1 -+ gamma_mu) U_mu(x) phi(x+mu,s) + (1 +- gamma_mu) U_mu(x-mu)^+ phi(x-mu,s) ]
//     phi      = psi_in                                       (PRE = 0)
//              = (1 + (pre_o/pre_d) Lambda) psi_in            (PRE = 1: "B on load"; the factor pre_d is
//                                                              folded into coef_hop by the host)
//     r        = M r  (POST = 1, dense L5 x L5 matrix per chirality along s, e.g. B A^{-1})
//              = (post_d + post_o Lambda^+) r  (POST = 2)
//     out(x,s) = r + own term (OWN = 1: psi_own, 2: (own_d + own_o Lambda) psi_own, 3: Lambda^+ form)
//
// Thread (lane, sg): lane = site within a 32-site group (coalesced 512 B per load instruction in the
// warp-blob layout), sg = group of S consecutive fifth-dimension slices.  Each thread loads a link ONCE per
// direction (12-real reconstruction included) and reuses it from registers for its S slices; the B-on-load
// stencil in s slides over the same S slices (+ one half-spinor halo on each side).
// The s-mixing POST step goes through a shared-memory transpose: thread (lane, c) then owns complex
// component c of a site for ALL s and applies the L5 x L5 matrix from registers.
// Antiperiodic t boundary (folded into the accumulate FMA) and SU(3) reconstruction happen in-kernel.
#pragma once
#include "mdwf_device.cuh"
#include "mdwf_internal.h"

// One direction of the stencil for S slices.  FWD: neighbour x+mu with U_mu(x); else x-mu with U_mu(x-mu)^+ (link
// direction 4 + mu of the site's own tile).
template <class P, int MU, bool FWD, int DAG, int PRE, int S, bool TDIR>
MDWF_DEV void hop_dir(const HopArgs &a, int L5, int s0, long cb_own, long cb_nb, typename P::R bsign,
                      typename P::R (*acc)[24])
{
    using R = typename P::R;
    using V = typename P::V;
    constexpr int SGN = (FWD ? 1 : -1) * (DAG ? -1 : 1);   // H: (1 - gamma) forward, (1 + gamma) backward
    R U[18];
    load_link<P>(a.gauge, FWD ? MU : 4 + MU, cb_own, a.recon, U);   // backward links are stored pulled back and daggered

    const V *p0 = reinterpret_cast<const V *>(a.in) + sp_off(L5, P::NV, cb_nb, s0);   // slice s0, chunk 0
    const long n0 = sp_noff(L5, cb_nb, s0);
    constexpr long SL = 32 * P::NV;                                                    // chunks per slice

    if (PRE == 0) {
#pragma unroll
        for (int k = 0; k < S; k++) {
            R v[24], h[12], chi[12];
            load_chunks_at<P, P::NV>(p0 + k * SL, load_scale<P>(a.in_norm, n0 + 32 * k), v);
            project<MU, SGN>(v, h);
            su3_mul<false>(U, h, chi);
            recon_add<MU, SGN, TDIR>(chi, bsign, acc[k]);
        }
    } else {
        // phi_s = psi_s + f (P+ psi_{s-1} + P- psi_{s+1}),  f = pre_o/pre_d, wall factor -m_f at the wrap
        const R f = (R)(a.pre_o / a.pre_d), fw = (R)(-a.mf * a.pre_o / a.pre_d);
        const int sm = (s0 == 0) ? L5 - 1 : s0 - 1;            // slice below the window
        const int sp = (s0 + S >= L5) ? 0 : s0 + S;            // slice above the window
        R prev_up[12], cur[24], nxt[24];
        {
            const V *pm = reinterpret_cast<const V *>(a.in) + sp_off(L5, P::NV, cb_nb, sm);
            load_chunks_at<P, P::NV / 2>(pm, load_scale<P>(a.in_norm, sp_noff(L5, cb_nb, sm)), prev_up);
        }
        load_chunks_at<P, P::NV>(p0, load_scale<P>(a.in_norm, n0), cur);
#pragma unroll
        for (int k = 0; k < S; k++) {
            if (k < S - 1) {
                load_chunks_at<P, P::NV>(p0 + (k + 1) * SL, load_scale<P>(a.in_norm, n0 + 32 * (k + 1)), nxt);
            } else {
                const V *pp = reinterpret_cast<const V *>(a.in) + sp_off(L5, P::NV, cb_nb, sp) + 32 * (P::NV / 2);
                load_chunks_at<P, P::NV / 2>(pp, load_scale<P>(a.in_norm, sp_noff(L5, cb_nb, sp)), nxt + 12);
            }
            const R fu = (s0 + k == 0) ? fw : f;
            const R fl = (s0 + k == L5 - 1) ? fw : f;
            R w[24], h[12], chi[12];
#pragma unroll
            for (int q = 0; q < 12; q++) {
                w[q] = fma(fu, prev_up[q], cur[q]);
                w[12 + q] = fma(fl, nxt[12 + q], cur[12 + q]);
            }
            project<MU, SGN>(w, h);
            su3_mul<false>(U, h, chi);
            recon_add<MU, SGN, TDIR>(chi, bsign, acc[k]);
#pragma unroll
            for (int q = 0; q < 12; q++) prev_up[q] = cur[q];
            if (k < S - 1) {
#pragma unroll
                for (int q = 0; q < 24; q++) cur[q] = nxt[q];
            }
        }
    }
}

template <class P, int S> struct HopCfg {
    // registers: S*24 accumulators + 18 link + ~60 working; keep >= 2-3 blocks of 128 threads per SM
    static constexpr int MAXT = (S == 1) ? 1024 : 128;
    static constexpr int MINB = (S == 1) ? 1 : (sizeof(typename P::R) == 8 ? 1 : 3);
};

template <class P, int DAG, int PRE, int POST, int OWN, int L5T, int S>
__global__ void __launch_bounds__(HopCfg<P, S>::MAXT, HopCfg<P, S>::MINB) hop_kernel(const HopArgs a)
{
    using R = typename P::R;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    R *tile = reinterpret_cast<R *>(smem_raw);           // [L5][24][32]      (POST != 0)
    const int L5 = L5T ? L5T : a.L5;
    const int lane = threadIdx.x, sg = threadIdx.y, s0 = sg * S;
    const int NSG = L5 / S;
    // Sweep order: the grid walks z-chunk by z-chunk and, inside a chunk, t-slice by
    // t-slice, so that the t+-1 neighbours are re-read from L2 after one small slab, not after a whole t-slice.
    long cb0 = (long)blockIdx.x * 32;
    if (a.sweep_nb) {
        const int Lt = a.L[3];
        const int per_chunk = a.sweep_nb * Lt;
        const int c = blockIdx.x / per_chunk, r = blockIdx.x - c * per_chunk;
        const int t = r / a.sweep_nb, q = r - t * a.sweep_nb;
        cb0 = (long)t * ((long)a.Vh / Lt) + (long)c * a.sweep_chunk + (long)q * 32;
    }
    const long cb = cb0 + lane;
    const bool active = cb < a.Vh;
    R *dense = tile + (size_t)L5 * 24 * 32;              // [2][L5][L5]       (POST == 1)
    if (POST == 1) {
        const R *src = reinterpret_cast<const R *>(a.dense);
        for (int k = sg * 32 + lane; k < 2 * L5 * L5; k += 32 * NSG) dense[k] = src[k];
    }

    R acc[S][24];
#pragma unroll
    for (int k = 0; k < S; k++)
#pragma unroll
        for (int q = 0; q < 24; q++) acc[k][q] = 0;

    if (active) {
        const int Lxh = a.L[0] >> 1, Ly = a.L[1], Lz = a.L[2], Lt = a.L[3];
        int r = (int)cb;
        const int xh = r % Lxh; r /= Lxh;
        const int y = r % Ly;   r /= Ly;
        const int z = r % Lz;
        const int t = r / Lz;
        const int xodd = (a.parity_out + y + z + t) & 1;          // x = 2 xh + xodd
        const long sy = Lxh, sz = (long)Lxh * Ly, st = (long)Lxh * Ly * Lz;
        const long cb_xp = xodd ? (xh == Lxh - 1 ? cb - (Lxh - 1) : cb + 1) : cb;
        const long cb_xm = xodd ? cb : (xh == 0 ? cb + (Lxh - 1) : cb - 1);
        const long cb_yp = (y == Ly - 1) ? cb - (Ly - 1) * sy : cb + sy;
        const long cb_ym = (y == 0) ? cb + (Ly - 1) * sy : cb - sy;
        const long cb_zp = (z == Lz - 1) ? cb - (Lz - 1) * sz : cb + sz;
        const long cb_zm = (z == 0) ? cb + (Lz - 1) * sz : cb - sz;
        const long cb_tp = (t == Lt - 1) ? cb - (Lt - 1) * st : cb + st;
        const long cb_tm = (t == 0) ? cb + (Lt - 1) * st : cb - st;
        const R one = (R)1;
        const R btp = (t == Lt - 1) ? (R)-1 : (R)1;                // antiperiodic in t
        const R btm = (t == 0) ? (R)-1 : (R)1;
        hop_dir<P, 0, true, DAG, PRE, S, false>(a, L5, s0, cb, cb_xp, one, acc);
        hop_dir<P, 0, false, DAG, PRE, S, false>(a, L5, s0, cb, cb_xm, one, acc);
        hop_dir<P, 1, true, DAG, PRE, S, false>(a, L5, s0, cb, cb_yp, one, acc);
        hop_dir<P, 1, false, DAG, PRE, S, false>(a, L5, s0, cb, cb_ym, one, acc);
        hop_dir<P, 2, true, DAG, PRE, S, false>(a, L5, s0, cb, cb_zp, one, acc);
        hop_dir<P, 2, false, DAG, PRE, S, false>(a, L5, s0, cb, cb_zm, one, acc);
        hop_dir<P, 3, true, DAG, PRE, S, true>(a, L5, s0, cb, cb_tp, btp, acc);
        hop_dir<P, 3, false, DAG, PRE, S, true>(a, L5, s0, cb, cb_tm, btm, acc);
    }
    const R coef = (R)a.coef_hop;

    if (POST != 0) {
        // ---- transpose through shared memory: (lane, s) owns a site-slice -> (lane, c) owns a column over all s
#pragma unroll
        for (int k = 0; k < S; k++)
#pragma unroll
            for (int q = 0; q < 24; q++) tile[((s0 + k) * 24 + q) * 32 + lane] = acc[k][q];
        __syncthreads();
        constexpr int LMAX = L5T ? L5T : 32;
        for (int c = sg; c < 12; c += NSG) {
            const bool up = c < 6;
            R vr[LMAX], vi[LMAX];
#pragma unroll
            for (int q = 0; q < LMAX; q++)
                if (q < L5) {
                    vr[q] = tile[(q * 24 + 2 * c) * 32 + lane];
                    vi[q] = tile[(q * 24 + 2 * c + 1) * 32 + lane];
                }
            if (POST == 1) {
                const R *M = dense + (up ? 0 : L5 * L5);
#pragma unroll
                for (int so = 0; so < LMAX; so++)
                    if (so < L5) {
                        R sr = 0, si = 0;
#pragma unroll
                        for (int q = 0; q < LMAX; q++)
                            if (q < L5) {
                                const R m = M[so * L5 + q];
                                sr = fma(m, vr[q], sr);
                                si = fma(m, vi[q], si);
                            }
                        tile[(so * 24 + 2 * c) * 32 + lane] = sr;
                        tile[(so * 24 + 2 * c + 1) * 32 + lane] = si;
                    }
            } else {
                // (post_d + post_o Lambda^+): upper spins take s+1, lower spins s-1, -m_f at the wrap
                const R d = (R)a.post_d, o = (R)a.post_o, mw = (R)(-a.mf);
#pragma unroll
                for (int so = 0; so < LMAX; so++)
                    if (so < L5) {
                        const int qu = (so + 1 >= L5) ? 0 : so + 1;            // compile-time when L5T != 0
                        const int ql = (so - 1 < 0) ? L5 - 1 : so - 1;
                        const R fu = (so + 1 >= L5) ? o * mw : o;
                        const R fl = (so - 1 < 0) ? o * mw : o;
                        const R nr = up ? fu * vr[qu] : fl * vr[ql];
                        const R ni = up ? fu * vi[qu] : fl * vi[ql];
                        tile[(so * 24 + 2 * c) * 32 + lane] = fma(d, vr[so], nr);
                        tile[(so * 24 + 2 * c + 1) * 32 + lane] = fma(d, vi[so], ni);
                    }
            }
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < S; k++)
#pragma unroll
            for (int q = 0; q < 24; q++) acc[k][q] = tile[((s0 + k) * 24 + q) * 32 + lane];
    }

    if (!active) return;

#pragma unroll
    for (int k = 0; k < S; k++) {
        const int s = s0 + k;
        R o[24];
        if (OWN == 0) {
#pragma unroll
            for (int q = 0; q < 24; q++) o[q] = coef * acc[k][q];
        } else if (OWN == 1) {
            R w[24];
            load_spinor<P>(a.own, a.own_norm, L5, s, cb, w);
#pragma unroll
            for (int q = 0; q < 24; q++) o[q] = fma(coef, acc[k][q], w[q]);
        } else {
            // (own_d + own_o Lambda) psi: upper from s-1, lower from s+1; Lambda^+ (OWN == 3): swapped
            R w[24], u[12], l[12];
            load_spinor<P>(a.own, a.own_norm, L5, s, cb, w);
            int su = (OWN == 2) ? s - 1 : s + 1;
            int sl = (OWN == 2) ? s + 1 : s - 1;
            R fu = (R)a.own_o, fl = (R)a.own_o;
            if (su < 0) { su = L5 - 1; fu *= (R)(-a.mf); }
            if (su >= L5) { su = 0; fu *= (R)(-a.mf); }
            if (sl < 0) { sl = L5 - 1; fl *= (R)(-a.mf); }
            if (sl >= L5) { sl = 0; fl *= (R)(-a.mf); }
            load_half<P>(a.own, a.own_norm, L5, su, cb, 0, u);
            load_half<P>(a.own, a.own_norm, L5, sl, cb, 1, l);
            const R d = (R)a.own_d;
#pragma unroll
            for (int q = 0; q < 12; q++) {
                o[q] = fma(coef, acc[k][q], fma(d, w[q], fu * u[q]));
                o[12 + q] = fma(coef, acc[k][12 + q], fma(d, w[12 + q], fl * l[q]));
            }
        }
        store_spinor<P>(a.out, a.out_norm, L5, s, cb, o);
    }
}

// ---- site-local dense s-matrix (A^{-1} in source preparation / reconstruction) -----------------
// one thread per 4D site.  Not on the CG hot loop (runs twice per solve).
template <class P>
__global__ void sdense_kernel(int L5, long Vh, const void *in, const float *in_norm, void *out, float *out_norm,
                              const void *dense)
{
    using R = typename P::R;
    const long cb = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= Vh) return;
    const R *M = reinterpret_cast<const R *>(dense);
    for (int so = 0; so < L5; so++) {
        R acc[24];
#pragma unroll
        for (int k = 0; k < 24; k++) acc[k] = 0;
        for (int q = 0; q < L5; q++) {
            R v[24];
            load_spinor<P>(in, in_norm, L5, q, cb, v);
            const R mu = M[so * L5 + q], ml = M[L5 * L5 + so * L5 + q];
#pragma unroll
            for (int k = 0; k < 12; k++) {
                acc[k] = fma(mu, v[k], acc[k]);
                acc[12 + k] = fma(ml, v[12 + k], acc[12 + k]);
            }
        }
        store_spinor<P>(out, out_norm, L5, so, cb, acc);
    }
}

// ---- launchers ----------------------------------------------------------------------------------
template <class P, int DAG, int PRE, int POST, int OWN, int L5T, int S>
static int launch_hop_inst(const HopArgs &a, cudaStream_t st)
{
    using R = typename P::R;
    const int L5 = a.L5;
    dim3 block(32, L5 / S);
    dim3 grid((unsigned)((a.Vh + 31) / 32));
    size_t smem = 0;
    if (POST != 0) smem = ((size_t)L5 * 24 * 32 + (POST == 1 ? 2 * L5 * L5 : 0)) * sizeof(R);
    auto k = hop_kernel<P, DAG, PRE, POST, OWN, L5T, S>;
    static size_t smem_set = 0;                            // once per instantiation (and again only for a larger L5), not per launch
    if (smem > 48 * 1024 && smem > smem_set) {
        cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return (int)e;
        smem_set = smem;
    }
    k<<<grid, block, smem, st>>>(a);
    return (int)cudaGetLastError();
}

template <class P, int DAG, int PRE, int POST, int OWN>
static int launch_hop_l5(const HopArgs &a, cudaStream_t st)
{
    // common L5 of Table II get S slices per thread and register-resident fifth-dimension columns
    if (a.L5 == 12) return launch_hop_inst<P, DAG, PRE, POST, OWN, 12, 3>(a, st);
#ifndef MDWF_DEV_FAST
    if (a.L5 == 8) return launch_hop_inst<P, DAG, PRE, POST, OWN, 8, 2>(a, st);
    if (a.L5 == 16) return launch_hop_inst<P, DAG, PRE, POST, OWN, 16, 4>(a, st);
#endif
    return launch_hop_inst<P, DAG, PRE, POST, OWN, 0, 1>(a, st);
}

template <class P>
static int launch_hop_prec(int dag, int pre, int post, int own, const HopArgs &a, cudaStream_t st)
{
    if (!dag && pre == 1 && post == 1 && own == 0) return launch_hop_l5<P, 0, 1, 1, 0>(a, st);   // K1
    if (!dag && pre == 0 && post == 0 && own == 2) return launch_hop_l5<P, 0, 0, 0, 2>(a, st);   // K2
    if (!dag && pre == 1 && post == 0 && own == 2) return launch_hop_l5<P, 0, 1, 0, 2>(a, st);   // D
    if (!dag && pre == 1 && post == 0 && own == 1) return launch_hop_l5<P, 0, 1, 0, 1>(a, st);   // Schur prep/recon
    if (dag && pre == 0 && post == 1 && own == 0) return launch_hop_l5<P, 1, 0, 1, 0>(a, st);    // K1^+
    if (dag && pre == 0 && post == 2 && own == 3) return launch_hop_l5<P, 1, 0, 2, 3>(a, st);    // K2^+, D^+
    if (!dag && pre == 0 && post == 1 && own == 1) return launch_hop_l5<P, 0, 0, 1, 1>(a, st);   // K2 of Mpc_sym: psi + coef A^{-1} H t
    if (dag && pre == 0 && post == 2 && own == 1) return launch_hop_l5<P, 1, 0, 2, 1>(a, st);    // K2^+ of Mpc_sym^+: psi + coef B^+ H' u
    return (int)cudaErrorInvalidValue;
}

template <class P>
static int launch_sdense_prec(int L5, int Vh, const SpinorBuf &in, const SpinorBuf &out, const void *dense,
                              cudaStream_t st)
{
    const int T = 128;
    sdense_kernel<P><<<(Vh + T - 1) / T, T, 0, st>>>(L5, Vh, in.v, in.norm, out.v, out.norm, dense);
    return (int)cudaGetLastError();
}
