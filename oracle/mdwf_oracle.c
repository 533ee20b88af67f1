/*
 * mdwf_oracle.c -- CPU ORACLE for the Moebius domain-wall fermion (MDWF) operator.
 *
 * TEST INFRASTRUCTURE ONLY.  This file is the plain, slow, fp64 reference that the
 * CUDA path is checked against.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may load it.  It shares no
 * code, header, table or constant generator with paper_1701_07559_b200/csrc.
 *
 * What the paper fixes (PAPER.md = /root/reference/PAPER.md, arXiv:1701.07559):
 *   - Eq. (2): D^Moebius(M5) = (b5+c5) D^Wilson(M5) / (2 + (b5-c5) D^Wilson(M5)),
 *     i.e. the Wilson kernel with negative mass -M5 and the two Moebius parameters b5, c5.
 *   - Eq. (3): b5 - c5 = 1 in all of the paper's runs (not assumed here).
 *   - Sec. VII: the "asymmetric" even-odd preconditioned operator is the
 *     one solved; the solver is a mixed-precision MDWF solver.
 * The 5D operator itself is never written in the paper (it cites Brower-Neff-Orginos
 * [113-115]); the definitions D1..D9 of SURVEY.md section 8(c) are the reading used,
 * restated here, and pinned by tests/test_oracle_pins.py (plane waves, the overlap
 * identity that ties the 5D operator back to Eq. (2), hermiticity, gauge covariance,
 * dense brute force).
 *
 * Definitions:
 *   D1 fields   psi(x,s) in C^{4x3}; U_mu(x) in SU(3); 4D parity p(x) = (x+y+z+t) mod 2.
 *   D2 gamma    DeGrand-Rossi basis, gamma5 = diag(+1,+1,-1,-1); P+- = (1 +- gamma5)/2.
 *   D3 hopping  (H psi)(x,s) = sum_mu (1-gamma_mu) U_mu(x) psi(x+mu,s)
 *                                     + (1+gamma_mu) U_mu(x-mu)^dagger psi(x-mu,s),
 *               periodic in x,y,z, antiperiodic in t.
 *   D4 Wilson   D_W = (4 - M5) - H/2.
 *   D5 Lambda   (Lambda psi)_s = P- psi_{s+1} + P+ psi_{s-1},
 *               psi_{L5} = -m_f psi_0, psi_{-1} = -m_f psi_{L5-1}.
 *   D6 Moebius  D = D_W (b5 + c5 Lambda) + (1 - Lambda) = A - H B / 2,
 *               A = alpha + beta Lambda, B = b5 + c5 Lambda,
 *               alpha = b5 (4-M5) + 1, beta = c5 (4-M5) - 1.
 *               A^{-1} closed form on the P+ half:
 *               (A+^{-1})_{s,s'} = (-kappa)^{(s-s') mod L5} f / (alpha (1 + m_f (-kappa)^{L5})),
 *               f = 1 if s >= s' else -m_f, kappa = beta/alpha; A-^{-1} = (A+^{-1})^T.
 *   The compositions D7 (Mpc), D8 (Schur solve), D9 (CGLS) are written step by step in
 *   oracle/mdwf_oracle.py from the primitives below.
 *
 *   D10 flop convention used when a rate is quoted for this oracle or for the CUDA path:
 *       hop = 1320 per 5D site, B = A = 72, xpay = 48, A^{-1} = 48 L5 - 24,
 *       F_Mpc(L5) = 2880 + 48 L5 per odd 5D site per application of Mpc or Mpc^dagger.
 *
 * Data layout (canonical interchange layout, C order, complex = (re,im) doubles):
 *   gauge  U[t][z][y][x][mu][row][col], mu in {x,y,z,t}; U_mu(x) is the link x -> x+mu;
 *          no boundary sign folded in.
 *   spinor psi[s][t][z][y][x][spin][colour] on the full lattice.  Single-parity vectors
 *          are full-lattice arrays that are zero on the other parity.
 * Every primitive takes a list of 4D lexicographic site indices (x + Lx (y + Ly (z + Lz t)))
 * and writes the output on those sites only (all s); other output sites are untouched.
 * No blocking, fusion or projection tricks: gamma matrices are applied as 4x4 matrices.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

/* ---- D2: gamma matrices, DeGrand-Rossi basis (row-major 4x4) ---------------------- */
static void gamma_matrix(int mu, cplx g[16])
{
    for (int i = 0; i < 16; i++) g[i] = 0;
    switch (mu) {
    case 0: /* gamma_1 (x) */
        g[0 * 4 + 3] = I;  g[1 * 4 + 2] = I;  g[2 * 4 + 1] = -I; g[3 * 4 + 0] = -I; break;
    case 1: /* gamma_2 (y) */
        g[0 * 4 + 3] = -1; g[1 * 4 + 2] = 1;  g[2 * 4 + 1] = 1;  g[3 * 4 + 0] = -1; break;
    case 2: /* gamma_3 (z) */
        g[0 * 4 + 2] = I;  g[1 * 4 + 3] = -I; g[2 * 4 + 0] = -I; g[3 * 4 + 1] = I;  break;
    case 3: /* gamma_4 (t) */
        g[0 * 4 + 2] = 1;  g[1 * 4 + 3] = 1;  g[2 * 4 + 0] = 1;  g[3 * 4 + 1] = 1;  break;
    default: /* gamma_5 = gamma_1 gamma_2 gamma_3 gamma_4 */
        g[0] = 1; g[5] = 1; g[10] = -1; g[15] = -1; break;
    }
}

void orc_gamma(int mu, double *out_re_im /* 32 doubles */)
{
    cplx g[16];
    gamma_matrix(mu, g);
    for (int i = 0; i < 16; i++) { out_re_im[2 * i] = creal(g[i]); out_re_im[2 * i + 1] = cimag(g[i]); }
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- D3: the 4D Wilson hopping term on every s-slice ------------------------------ */
/* dagger = 0: H.  dagger = 1: H^dagger = gamma5 H gamma5 (signs of gamma_mu swapped). */
void orc_hop(const int *L, int L5, const double *U_, const double *in_, double *out_,
             const int64_t *sites, int64_t nsites, int dagger)
{
    const cplx *U = (const cplx *)U_;
    const cplx *in = (const cplx *)in_;
    cplx *out = (cplx *)out_;
    const int64_t V4 = (int64_t)L[0] * L[1] * L[2] * L[3];
    cplx gam[4][16];
    for (int mu = 0; mu < 4; mu++) gamma_matrix(mu, gam[mu]);
    const double sgn = dagger ? -1.0 : 1.0;

#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < nsites; n++) {
        const int64_t i4 = sites[n];
        int x[4];
        int64_t r = i4;
        for (int d = 0; d < 4; d++) { x[d] = (int)(r % L[d]); r /= L[d]; }
        for (int s = 0; s < L5; s++) {
            cplx acc[12];
            for (int k = 0; k < 12; k++) acc[k] = 0;
            for (int mu = 0; mu < 4; mu++) {
                int xp[4] = { x[0], x[1], x[2], x[3] }, xm[4] = { x[0], x[1], x[2], x[3] };
                xp[mu] = (x[mu] + 1) % L[mu];
                xm[mu] = (x[mu] + L[mu] - 1) % L[mu];
                /* antiperiodic boundary in t (mu == 3) */
                const double bp = (mu == 3 && x[3] == L[3] - 1) ? -1.0 : 1.0;
                const double bm = (mu == 3 && x[3] == 0) ? -1.0 : 1.0;
                const int64_t ip = xp[0] + (int64_t)L[0] * (xp[1] + (int64_t)L[1] * (xp[2] + (int64_t)L[2] * xp[3]));
                const int64_t im = xm[0] + (int64_t)L[0] * (xm[1] + (int64_t)L[1] * (xm[2] + (int64_t)L[2] * xm[3]));
                const cplx *Uf = U + (i4 * 4 + mu) * 9; /* U_mu(x)      */
                const cplx *Ub = U + (im * 4 + mu) * 9; /* U_mu(x - mu) */
                const cplx *pf = in + ((int64_t)s * V4 + ip) * 12;
                const cplx *pb = in + ((int64_t)s * V4 + im) * 12;
                cplx cf[12], cb[12];
                for (int sp = 0; sp < 4; sp++)
                    for (int a = 0; a < 3; a++) {
                        cplx f = 0, b = 0;
                        for (int c = 0; c < 3; c++) {
                            f += Uf[a * 3 + c] * pf[sp * 3 + c];       /* U psi(x+mu)         */
                            b += conj(Ub[c * 3 + a]) * pb[sp * 3 + c]; /* U^dagger psi(x-mu)  */
                        }
                        cf[sp * 3 + a] = bp * f;
                        cb[sp * 3 + a] = bm * b;
                    }
                for (int sp = 0; sp < 4; sp++)
                    for (int a = 0; a < 3; a++) {
                        cplx gf = 0, gb = 0;
                        for (int sq = 0; sq < 4; sq++) {
                            gf += gam[mu][sp * 4 + sq] * cf[sq * 3 + a];
                            gb += gam[mu][sp * 4 + sq] * cb[sq * 3 + a];
                        }
                        acc[sp * 3 + a] += (cf[sp * 3 + a] - sgn * gf) + (cb[sp * 3 + a] + sgn * gb);
                    }
            }
            cplx *o = out + ((int64_t)s * V4 + i4) * 12;
            for (int k = 0; k < 12; k++) o[k] = acc[k];
        }
    }
}

/* ---- D5: out = a psi + b Lambda psi   (dagger: Lambda -> Lambda^dagger) ------------ */
/* Lambda        : upper spin components (P+) come from s-1, lower (P-) from s+1.       */
/* Lambda^dagger : upper from s+1, lower from s-1.  The wrap carries the factor -m_f.   */
void orc_s_affine(int64_t V4, int L5, double mf, double a, double b, const double *in_, double *out_,
                  const int64_t *sites, int64_t nsites, int dagger)
{
    const cplx *in = (const cplx *)in_;
    cplx *out = (cplx *)out_;
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < nsites; n++) {
        const int64_t i4 = sites[n];
        for (int s = 0; s < L5; s++) {
            int s_up = dagger ? s + 1 : s - 1;  /* source slice of the P+ half */
            int s_lo = dagger ? s - 1 : s + 1;  /* source slice of the P- half */
            double f_up = 1.0, f_lo = 1.0;
            if (s_up < 0) { s_up = L5 - 1; f_up = -mf; }
            if (s_up >= L5) { s_up = 0; f_up = -mf; }
            if (s_lo < 0) { s_lo = L5 - 1; f_lo = -mf; }
            if (s_lo >= L5) { s_lo = 0; f_lo = -mf; }
            const cplx *p = in + ((int64_t)s * V4 + i4) * 12;
            const cplx *pu = in + ((int64_t)s_up * V4 + i4) * 12;
            const cplx *pl = in + ((int64_t)s_lo * V4 + i4) * 12;
            cplx *o = out + ((int64_t)s * V4 + i4) * 12;
            cplx tmp[12];
            for (int k = 0; k < 6; k++) tmp[k] = a * p[k] + b * f_up * pu[k];
            for (int k = 6; k < 12; k++) tmp[k] = a * p[k] + b * f_lo * pl[k];
            for (int k = 0; k < 12; k++) o[k] = tmp[k];
        }
    }
}

/* ---- D6: closed-form inverse of A = alpha + beta Lambda ---------------------------- */
/* Fills Ainv_plus[s*L5+s'] (P+ half); the P- half is its transpose.                    */
void orc_Ainv_table(int L5, double alpha, double beta, double mf, double *Ainv_plus)
{
    const double kappa = beta / alpha;
    const double denom = alpha * (1.0 + mf * pow(-kappa, L5));
    for (int s = 0; s < L5; s++)
        for (int sp = 0; sp < L5; sp++) {
            const int d = ((s - sp) % L5 + L5) % L5;
            const double f = (s >= sp) ? 1.0 : -mf;
            Ainv_plus[s * L5 + sp] = pow(-kappa, d) * f / denom;
        }
}

/* out = A^{-1} in (dagger: A^{-dagger} = transpose per chirality), site-local in 4D.   */
void orc_Ainv(int64_t V4, int L5, double alpha, double beta, double mf, const double *in_, double *out_,
              const int64_t *sites, int64_t nsites, int dagger)
{
    const cplx *in = (const cplx *)in_;
    cplx *out = (cplx *)out_;
    double *Tp = (double *)malloc(sizeof(double) * L5 * L5);
    orc_Ainv_table(L5, alpha, beta, mf, Tp);
#pragma omp parallel
    {
        cplx *tmp = (cplx *)malloc(sizeof(cplx) * 12 * L5);
#pragma omp for schedule(static)
        for (int64_t n = 0; n < nsites; n++) {
            const int64_t i4 = sites[n];
            for (int s = 0; s < L5; s++) {
                for (int k = 0; k < 12; k++) tmp[s * 12 + k] = 0;
                for (int sp = 0; sp < L5; sp++) {
                    const cplx *p = in + ((int64_t)sp * V4 + i4) * 12;
                    /* P+ half uses A+^{-1}[s][s'], P- half its transpose; dagger swaps them */
                    const double cu = dagger ? Tp[sp * L5 + s] : Tp[s * L5 + sp];
                    const double cl = dagger ? Tp[s * L5 + sp] : Tp[sp * L5 + s];
                    for (int k = 0; k < 6; k++) tmp[s * 12 + k] += cu * p[k];
                    for (int k = 6; k < 12; k++) tmp[s * 12 + k] += cl * p[k];
                }
            }
            for (int s = 0; s < L5; s++) {
                cplx *o = out + ((int64_t)s * V4 + i4) * 12;
                for (int k = 0; k < 12; k++) o[k] = tmp[s * 12 + k];
            }
        }
        free(tmp);
    }
    free(Tp);
}

/* ---- vector helpers on listed sites (all s): out = a*x + b*y, and Re<x,y> ---------- */
void orc_axpby(int64_t V4, int L5, double a, const double *x_, double b, const double *y_, double *out_,
               const int64_t *sites, int64_t nsites)
{
    const cplx *x = (const cplx *)x_, *y = (const cplx *)y_;
    cplx *out = (cplx *)out_;
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < nsites; n++)
        for (int s = 0; s < L5; s++) {
            const int64_t o = ((int64_t)s * V4 + sites[n]) * 12;
            for (int k = 0; k < 12; k++) out[o + k] = a * x[o + k] + b * y[o + k];
        }
}

double orc_redot(int64_t V4, int L5, const double *x_, const double *y_, const int64_t *sites, int64_t nsites)
{
    const cplx *x = (const cplx *)x_, *y = (const cplx *)y_;
    double sum = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : sum)
    for (int64_t n = 0; n < nsites; n++)
        for (int s = 0; s < L5; s++) {
            const int64_t o = ((int64_t)s * V4 + sites[n]) * 12;
            for (int k = 0; k < 12; k++) sum += creal(conj(x[o + k]) * y[o + k]);
        }
    return sum;
}
