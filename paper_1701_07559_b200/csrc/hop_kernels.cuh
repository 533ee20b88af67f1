// hop_kernels.cuh -- the fused Wilson-hopping + fifth-dimension kernel family (S1-S6 of the hot path).
//
// One launch computes, for every site x of one 4D parity and every s:
//     r(x,s)   = coef_hop * sum_mu [ (1 -+ gamma_mu) U_mu(x) phi(x+mu,s) + (1 +- gamma_mu) U_mu(x-mu)^+ phi(x-mu,s) ]
//     phi      = psi_in                      (PRE = 0)
//              = (pre_d + pre_o Lambda) psi_in, applied while loading the neighbour (PRE = 1: "B on load")
//     r        = M r  (POST = 1, dense L5 x L5 matrix per chirality along s, e.g. B A^{-1})
//              = (post_d + post_o Lambda^+) r  (POST = 2)
//     out(x,s) = r + own term (OWN = 1: psi_own, 2: (own_d + own_o Lambda) psi_own, 3: Lambda^+ form)
// Thread (i, s) = (site in block, fifth-dimension slice): consecutive lanes are consecutive checkerboard
// sites, so every global access is a coalesced vector load/store.  The s-mixing POST step goes through a
// shared-memory transpose: thread (i, c) then owns complex component c of site i for ALL s, applies the
// L5 x L5 matrix from registers and writes the column back.
// Antiperiodic t boundary and SU(3) 12-real reconstruction happen in-kernel.
#pragma once
#include "mdwf_device.cuh"
#include "mdwf_internal.h"

// One direction of the stencil.  FWD: neighbour x+mu with U_mu(x); else x-mu with U_mu(x-mu)^dagger.
template <class P, int MU, bool FWD, int DAG, int PRE>
MDWF_DEV void hop_dir(const HopArgs &a, int s, long cb_own, long cb_nb, typename P::R bsign, typename P::R *acc)
{
    using R = typename P::R;
    constexpr int SGN = (FWD ? 1 : -1) * (DAG ? -1 : 1);   // H: (1 - gamma) forward, (1 + gamma) backward
    const long Vh = a.Vh;
    R v[24];
    load_spinor<P>(a.in, a.in_norm, s, cb_nb, Vh, v);
    if (PRE == 1) {
        // (B psi)_s = pre_d psi_s + pre_o (P+ psi_{s-1} + P- psi_{s+1}), wall factor -m_f at the wrap
        int su = s - 1, sl = s + 1;
        R fu = (R)a.pre_o, fl = (R)a.pre_o;
        if (su < 0) { su = a.L5 - 1; fu *= (R)(-a.mf); }
        if (sl >= a.L5) { sl = 0; fl *= (R)(-a.mf); }
        R u[12], l[12];
        load_half<P>(a.in, a.in_norm, su, cb_nb, Vh, 0, u);
        load_half<P>(a.in, a.in_norm, sl, cb_nb, Vh, 1, l);
        const R d = (R)a.pre_d;
#pragma unroll
        for (int k = 0; k < 12; k++) {
            v[k] = d * v[k] + fu * u[k];
            v[12 + k] = d * v[12 + k] + fl * l[k];
        }
    }
    R h[12], chi[12], U[18];
    project<MU, SGN>(v, bsign, h);
    if (FWD) {
        load_link<P>(a.gauge_same, MU, cb_own, Vh, a.recon, U);
        su3_mul<false>(U, h, chi);
    } else {
        load_link<P>(a.gauge_other, MU, cb_nb, Vh, a.recon, U);
        su3_mul<true>(U, h, chi);
    }
    recon_add<MU, SGN>(chi, acc);
}

template <class P, int DAG, int PRE, int POST, int OWN, int L5T>
__global__ void __launch_bounds__(P::MAXT) hop_kernel(const HopArgs a)
{
    using R = typename P::R;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    R *tile = reinterpret_cast<R *>(smem_raw);           // [L5][24][BX]      (POST != 0)
    const int L5 = L5T ? L5T : a.L5;
    const int BX = blockDim.x;
    const int i = threadIdx.x, s = threadIdx.y;
    const long Vh = a.Vh;
    const long cb = (long)blockIdx.x * BX + i;
    const bool active = cb < Vh;
    R *dense = tile + (size_t)L5 * 24 * BX;              // [2][L5][L5]       (POST == 1)
    if (POST == 1) {
        const R *src = reinterpret_cast<const R *>(a.dense);
        for (int k = s * BX + i; k < 2 * L5 * L5; k += BX * L5) dense[k] = src[k];
    }

    R acc[24];
#pragma unroll
    for (int k = 0; k < 24; k++) acc[k] = 0;

    if (active) {
        const int Lxh = a.L[0] >> 1, Ly = a.L[1], Lz = a.L[2], Lt = a.L[3];
        int r = (int)cb;
        const int xh = r % Lxh; r /= Lxh;
        const int y = r % Ly;   r /= Ly;
        const int z = r % Lz;
        const int t = r / Lz;
        const int xodd = (a.parity_out + y + z + t) & 1;          // x = 2 xh + xodd
        const long sy = Lxh, sz = (long)Lxh * Ly, st = (long)Lxh * Ly * Lz;
        // x direction: the neighbour has the other x-parity
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
        hop_dir<P, 0, true, DAG, PRE>(a, s, cb, cb_xp, one, acc);
        hop_dir<P, 0, false, DAG, PRE>(a, s, cb, cb_xm, one, acc);
        hop_dir<P, 1, true, DAG, PRE>(a, s, cb, cb_yp, one, acc);
        hop_dir<P, 1, false, DAG, PRE>(a, s, cb, cb_ym, one, acc);
        hop_dir<P, 2, true, DAG, PRE>(a, s, cb, cb_zp, one, acc);
        hop_dir<P, 2, false, DAG, PRE>(a, s, cb, cb_zm, one, acc);
        hop_dir<P, 3, true, DAG, PRE>(a, s, cb, cb_tp, btp, acc);
        hop_dir<P, 3, false, DAG, PRE>(a, s, cb, cb_tm, btm, acc);
        const R coef = (R)a.coef_hop;
#pragma unroll
        for (int k = 0; k < 24; k++) acc[k] *= coef;
    }

    if (POST != 0) {
        // ---- transpose through shared memory: (i, s) owns a site-slice -> (i, c) owns a column over all s
#pragma unroll
        for (int k = 0; k < 24; k++) tile[((size_t)s * 24 + k) * BX + i] = acc[k];
        __syncthreads();
        constexpr int LMAX = L5T ? L5T : 32;
        const int nthr = BX * L5;
        for (int item = s * BX + i; item < BX * 12; item += nthr) {
            const int ii = item % BX, c = item / BX;
            const bool up = c < 6;
            R vr[LMAX], vi[LMAX];
#pragma unroll
            for (int q = 0; q < LMAX; q++)
                if (q < L5) {
                    vr[q] = tile[((size_t)q * 24 + 2 * c) * BX + ii];
                    vi[q] = tile[((size_t)q * 24 + 2 * c + 1) * BX + ii];
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
                                sr += m * vr[q];
                                si += m * vi[q];
                            }
                        tile[((size_t)so * 24 + 2 * c) * BX + ii] = sr;
                        tile[((size_t)so * 24 + 2 * c + 1) * BX + ii] = si;
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
                        tile[((size_t)so * 24 + 2 * c) * BX + ii] = d * vr[so] + nr;
                        tile[((size_t)so * 24 + 2 * c + 1) * BX + ii] = d * vi[so] + ni;
                    }
            }
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < 24; k++) acc[k] = tile[((size_t)s * 24 + k) * BX + i];
    }

    if (!active) return;

    if (OWN == 1) {
        R w[24];
        load_spinor<P>(a.own, a.own_norm, s, cb, Vh, w);
#pragma unroll
        for (int k = 0; k < 24; k++) acc[k] += w[k];
    } else if (OWN >= 2) {
        // (own_d + own_o Lambda) psi: upper from s-1, lower from s+1; Lambda^+ (OWN == 3): swapped
        R w[24], u[12], l[12];
        load_spinor<P>(a.own, a.own_norm, s, cb, Vh, w);
        int su = (OWN == 2) ? s - 1 : s + 1;
        int sl = (OWN == 2) ? s + 1 : s - 1;
        R fu = (R)a.own_o, fl = (R)a.own_o;
        if (su < 0) { su = L5 - 1; fu *= (R)(-a.mf); }
        if (su >= L5) { su = 0; fu *= (R)(-a.mf); }
        if (sl < 0) { sl = L5 - 1; fl *= (R)(-a.mf); }
        if (sl >= L5) { sl = 0; fl *= (R)(-a.mf); }
        load_half<P>(a.own, a.own_norm, su, cb, Vh, 0, u);
        load_half<P>(a.own, a.own_norm, sl, cb, Vh, 1, l);
        const R d = (R)a.own_d;
#pragma unroll
        for (int k = 0; k < 12; k++) {
            acc[k] += d * w[k] + fu * u[k];
            acc[12 + k] += d * w[12 + k] + fl * l[k];
        }
    }
    store_spinor<P>(a.out, a.out_norm, s, cb, Vh, acc);
}

// ---- site-local dense s-matrix (A^{-1} in source preparation / reconstruction) -----------------
// thread (i, c): complex component c of site i for all s.  Not on the CG hot loop.
template <class P>
__global__ void sdense_kernel(int L5, long Vh, const void *in, const float *in_norm, void *out, float *out_norm,
                              const void *dense)
{
    using R = typename P::R;
    // one thread per 4D site; loops over s twice (plain, this kernel runs twice per solve)
    const long cb = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= Vh) return;
    const R *M = reinterpret_cast<const R *>(dense);
    for (int so = 0; so < L5; so++) {
        R acc[24];
#pragma unroll
        for (int k = 0; k < 24; k++) acc[k] = 0;
        for (int q = 0; q < L5; q++) {
            R v[24];
            load_spinor<P>(in, in_norm, q, cb, Vh, v);
            const R mu = M[so * L5 + q], ml = M[L5 * L5 + so * L5 + q];
#pragma unroll
            for (int k = 0; k < 12; k++) {
                acc[k] += mu * v[k];
                acc[12 + k] += ml * v[12 + k];
            }
        }
        store_spinor<P>(out, out_norm, so, cb, Vh, acc);
    }
}

// ---- launchers ----------------------------------------------------------------------------------
template <class P, int DAG, int PRE, int POST, int OWN, int L5T>
static int launch_hop_inst(const HopArgs &a, cudaStream_t st)
{
    using R = typename P::R;
    const int L5 = a.L5;
    int BX = 32;
    while (BX > 1 && BX * L5 > P::MAXT) BX >>= 1;
    dim3 block(BX, L5);
    dim3 grid((unsigned)((a.Vh + BX - 1) / BX));
    size_t smem = 0;
    if (POST != 0) smem = ((size_t)L5 * 24 * BX + (POST == 1 ? 2 * L5 * L5 : 0)) * sizeof(R);
    auto k = hop_kernel<P, DAG, PRE, POST, OWN, L5T>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return (int)e;
    }
    k<<<grid, block, smem, st>>>(a);
    return (int)cudaGetLastError();
}

template <class P, int DAG, int PRE, int POST, int OWN>
static int launch_hop_l5(const HopArgs &a, cudaStream_t st)
{
    if constexpr (POST != 0) {   // the s-mixing step keeps a whole column in registers: specialise common L5
        if (a.L5 == 8) return launch_hop_inst<P, DAG, PRE, POST, OWN, 8>(a, st);
        if (a.L5 == 12) return launch_hop_inst<P, DAG, PRE, POST, OWN, 12>(a, st);
        if (a.L5 == 16) return launch_hop_inst<P, DAG, PRE, POST, OWN, 16>(a, st);
    }
    return launch_hop_inst<P, DAG, PRE, POST, OWN, 0>(a, st);
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
