// flow_kernels.cu -- gradient-flow smearing of the gauge field (Sec. III: "an
// infinitesimal stout-smearing procedure" to t_gf = 1; App. D: Symanzik flow, eps = 0.03).  fp64, canonical
// layout U[t][z][y][x][mu][3][3] (interleaved re/im), periodic in all four directions.
//
//   dV_mu(x)/dt = Z_mu(x) V_mu(x),  Z = -TA( V_mu(x) S_mu(x) ),  S = c0 (6 plaquette staples) + c1 (18 rectangle staples),
//   TA(M) = (M - M^+)/2 - tr(M - M^+)/6;  Wilson flow c0 = 1, c1 = 0;  tree-level Symanzik c0 = 5/3, c1 = -1/12.
//   Luescher's third-order Runge-Kutta in its two-register form:
//       Z <- eps Z(W);                 W <- exp(Z/4) W
//       Z <- 8/9 eps Z(W) - 17/36 Z;   W <- exp(Z) W
//       Z <- 3/4 eps Z(W) - Z;         W <- exp(Z) W
// One thread per link; the force kernel reads neighbours through L2 (the field is read-only during a stage), the update
// kernel is site-local.  Pre-processing step of the action, not on the solver's hot loop.
#include "mdwf_internal.h"

namespace {

struct M3 {
    double2 e[9];
};
__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double2 cmac(double2 a, double2 b, double2 c) { return make_double2(fma(a.x, b.x, fma(-a.y, b.y, c.x)), fma(a.x, b.y, fma(a.y, b.x, c.y))); }
__device__ __forceinline__ M3 mload(const double2 *U, long site, int mu)
{
    M3 m;
    const double2 *p = U + (site * 4 + mu) * 9;
#pragma unroll
    for (int k = 0; k < 9; k++) m.e[k] = p[k];
    return m;
}
__device__ __forceinline__ M3 mdag(const M3 &a)
{
    M3 r;
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) r.e[i * 3 + j] = make_double2(a.e[j * 3 + i].x, -a.e[j * 3 + i].y);
    return r;
}
__device__ __forceinline__ M3 mmul(const M3 &a, const M3 &b)
{
    M3 r;
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            double2 s = cmul(a.e[i * 3], b.e[j]);
            s = cmac(a.e[i * 3 + 1], b.e[3 + j], s);
            s = cmac(a.e[i * 3 + 2], b.e[6 + j], s);
            r.e[i * 3 + j] = s;
        }
    return r;
}
__device__ __forceinline__ void maxpy(M3 &acc, double w, const M3 &a)
{
#pragma unroll
    for (int k = 0; k < 9; k++) { acc.e[k].x = fma(w, a.e[k].x, acc.e[k].x); acc.e[k].y = fma(w, a.e[k].y, acc.e[k].y); }
}

struct Geo {
    int L[4];
    long V4;
};
// site index of x + i mu + j nu (periodic)
__device__ __forceinline__ long nbr(const Geo &g, const int *c, int mu, int i, int nu, int j)
{
    int d[4] = {c[0], c[1], c[2], c[3]};
    d[mu] += i;
    d[nu] += j;
#pragma unroll
    for (int k = 0; k < 4; k++) {
        if (d[k] < 0) d[k] += g.L[k];
        if (d[k] >= g.L[k]) d[k] -= g.L[k];
        if (d[k] < 0) d[k] += g.L[k];               // shifts of up to two sites on an extent of 2
        if (d[k] >= g.L[k]) d[k] -= g.L[k];
    }
    return d[0] + (long)g.L[0] * (d[1] + (long)g.L[1] * (d[2] + (long)g.L[2] * d[3]));
}
// a path of links: product of U_dir(site)^(+-1) factors, built left to right
#define LK(i, j, dir) mload(U, nbr(g, c, mu, (i), nu, (j)), (dir))

// Z_new = a * eps * Z(U) + b * Z_old at link (site, mu)
__global__ void __launch_bounds__(128) flow_force_kernel(const double2 *__restrict__ U, double2 *Z, Geo g, double eps, double c0, double c1,
                                                         double a, double b)
{
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= g.V4 * 4) return;
    const int mu = (int)(idx & 3);
    const long site = idx >> 2;
    int c[4];
    {
        long r = site;
        c[0] = (int)(r % g.L[0]); r /= g.L[0];
        c[1] = (int)(r % g.L[1]); r /= g.L[1];
        c[2] = (int)(r % g.L[2]); r /= g.L[2];
        c[3] = (int)r;
    }
    M3 S;
#pragma unroll
    for (int k = 0; k < 9; k++) S.e[k] = make_double2(0.0, 0.0);
#pragma unroll 1
    for (int nu = 0; nu < 4; nu++) {
        if (nu == mu) continue;
        // plaquette staples: above  U_nu(x+mu) U_mu(x+nu)^+ U_nu(x)^+ ; below  U_nu(x+mu-nu)^+ U_mu(x-nu)^+ U_nu(x-nu)
        {
            M3 p = mmul(LK(1, 0, nu), mdag(LK(0, 1, mu)));
            maxpy(S, c0, mmul(p, mdag(LK(0, 0, nu))));
            p = mmul(mdag(LK(1, -1, nu)), mdag(LK(0, -1, mu)));
            maxpy(S, c0, mmul(p, LK(0, -1, nu)));
        }
        if (c1 == 0.0) continue;
        {   // long side along mu, this link first, above:  U_mu(x+mu) U_nu(x+2mu) U_mu(x+mu+nu)^+ U_mu(x+nu)^+ U_nu(x)^+
            M3 p = mmul(LK(1, 0, mu), LK(2, 0, nu));
            p = mmul(p, mdag(LK(1, 1, mu)));
            p = mmul(p, mdag(LK(0, 1, mu)));
            maxpy(S, c1, mmul(p, mdag(LK(0, 0, nu))));
        }
        {   // this link second, above:  U_nu(x+mu) U_mu(x+nu)^+ U_mu(x-mu+nu)^+ U_nu(x-mu)^+ U_mu(x-mu)
            M3 p = mmul(LK(1, 0, nu), mdag(LK(0, 1, mu)));
            p = mmul(p, mdag(LK(-1, 1, mu)));
            p = mmul(p, mdag(LK(-1, 0, nu)));
            maxpy(S, c1, mmul(p, LK(-1, 0, mu)));
        }
        {   // first, below:  U_mu(x+mu) U_nu(x+2mu-nu)^+ U_mu(x+mu-nu)^+ U_mu(x-nu)^+ U_nu(x-nu)
            M3 p = mmul(LK(1, 0, mu), mdag(LK(2, -1, nu)));
            p = mmul(p, mdag(LK(1, -1, mu)));
            p = mmul(p, mdag(LK(0, -1, mu)));
            maxpy(S, c1, mmul(p, LK(0, -1, nu)));
        }
        {   // second, below:  U_nu(x+mu-nu)^+ U_mu(x-nu)^+ U_mu(x-mu-nu)^+ U_nu(x-mu-nu) U_mu(x-mu)
            M3 p = mmul(mdag(LK(1, -1, nu)), mdag(LK(0, -1, mu)));
            p = mmul(p, mdag(LK(-1, -1, mu)));
            p = mmul(p, LK(-1, -1, nu));
            maxpy(S, c1, mmul(p, LK(-1, 0, mu)));
        }
        {   // long side along nu, up by two:  U_nu(x+mu) U_nu(x+mu+nu) U_mu(x+2nu)^+ U_nu(x+nu)^+ U_nu(x)^+
            M3 p = mmul(LK(1, 0, nu), LK(1, 1, nu));
            p = mmul(p, mdag(LK(0, 2, mu)));
            p = mmul(p, mdag(LK(0, 1, nu)));
            maxpy(S, c1, mmul(p, mdag(LK(0, 0, nu))));
        }
        {   // down by two:  U_nu(x+mu-nu)^+ U_nu(x+mu-2nu)^+ U_mu(x-2nu)^+ U_nu(x-2nu) U_nu(x-nu)
            M3 p = mmul(mdag(LK(1, -1, nu)), mdag(LK(1, -2, nu)));
            p = mmul(p, mdag(LK(0, -2, mu)));
            p = mmul(p, LK(0, -2, nu));
            maxpy(S, c1, mmul(p, LK(0, -1, nu)));
        }
    }
    const M3 M = mmul(mload(U, site, mu), S);
    // Z = -TA(M)
    double2 *zp = Z + idx * 9;
    const double tri = (M.e[0].y + M.e[4].y + M.e[8].y) * (1.0 / 3.0);          // tr(M - M^+)/6 = i Im tr M / 3
    const double w = a * eps;
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            double2 t;
            t.x = 0.5 * (M.e[i * 3 + j].x - M.e[j * 3 + i].x);
            t.y = 0.5 * (M.e[i * 3 + j].y + M.e[j * 3 + i].y) - (i == j ? tri : 0.0);
            double2 old = make_double2(0.0, 0.0);
            if (b != 0.0) old = zp[i * 3 + j];
            zp[i * 3 + j] = make_double2(fma(-w, t.x, b * old.x), fma(-w, t.y, b * old.y));
        }
}
#undef LK

// U <- exp(c Z) U at every link: scaling and squaring around a 16-term Taylor polynomial (||cZ|| / 2^k <= 1/2)
__global__ void __launch_bounds__(128) flow_update_kernel(double2 *U, const double2 *__restrict__ Z, long nlinks, double cz)
{
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= nlinks) return;
    M3 X, W;
    double n2 = 0.0;
#pragma unroll
    for (int k = 0; k < 9; k++) {
        const double2 z = Z[idx * 9 + k];
        X.e[k] = make_double2(cz * z.x, cz * z.y);
        n2 += X.e[k].x * X.e[k].x + X.e[k].y * X.e[k].y;
        W.e[k] = U[idx * 9 + k];
    }
    int sq = 0;
    double nrm = sqrt(n2);
    while (nrm > 0.5 && sq < 30) { nrm *= 0.5; sq++; }
    const double sc = ldexp(1.0, -sq);
#pragma unroll
    for (int k = 0; k < 9; k++) { X.e[k].x *= sc; X.e[k].y *= sc; }
    M3 E;                                                                        // Horner: 1 + X (1 + X/2 (1 + X/3 (...)))
#pragma unroll
    for (int k = 0; k < 9; k++) E.e[k] = make_double2((k % 4 == 0) ? 1.0 : 0.0, 0.0);
#pragma unroll 1
    for (int n = 16; n >= 1; n--) {
        M3 T = mmul(X, E);
        const double inv = 1.0 / n;
#pragma unroll
        for (int k = 0; k < 9; k++) E.e[k] = make_double2(fma(inv, T.e[k].x, (k % 4 == 0) ? 1.0 : 0.0), inv * T.e[k].y);
    }
    for (int k = 0; k < sq; k++) E = mmul(E, E);
    W = mmul(E, W);
#pragma unroll
    for (int k = 0; k < 9; k++) U[idx * 9 + k] = W.e[k];
}

// per-site sum over the 6 planes of Re tr P, reduced per block in a fixed order (one partial per block)
__global__ void __launch_bounds__(128) plaquette_kernel(const double2 *__restrict__ U, Geo g, double *partial)
{
    const long site = (long)blockIdx.x * blockDim.x + threadIdx.x;
    double s = 0.0;
    if (site < g.V4) {
        int c[4];
        long r = site;
        c[0] = (int)(r % g.L[0]); r /= g.L[0];
        c[1] = (int)(r % g.L[1]); r /= g.L[1];
        c[2] = (int)(r % g.L[2]); r /= g.L[2];
        c[3] = (int)r;
        for (int mu = 0; mu < 4; mu++)
            for (int nu = mu + 1; nu < 4; nu++) {
                M3 p = mmul(mload(U, site, mu), mload(U, nbr(g, c, mu, 1, nu, 0), nu));
                p = mmul(p, mdag(mload(U, nbr(g, c, mu, 0, nu, 1), mu)));
                const M3 q = mload(U, site, nu);                                 // Re tr(p q^+) = sum_ij Re(p_ij conj(q_ij))
#pragma unroll
                for (int k = 0; k < 9; k++) s += p.e[k].x * q.e[k].x + p.e[k].y * q.e[k].y;
            }
    }
    __shared__ double ws[4];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) partial[blockIdx.x] = (ws[0] + ws[1]) + (ws[2] + ws[3]);
}

}   // namespace

int mdwf_flow_plaquette_blocks(long V4) { return (int)((V4 + 127) / 128); }

// sum over sites and planes of Re tr P -> partial[] (one per block); the caller sums them in fixed order
int mdwf_launch_plaquette(const void *U, const int *L, double *partial, cudaStream_t st)
{
    Geo g;
    for (int d = 0; d < 4; d++) g.L[d] = L[d];
    g.V4 = (long)L[0] * L[1] * L[2] * L[3];
    plaquette_kernel<<<mdwf_flow_plaquette_blocks(g.V4), 128, 0, st>>>(reinterpret_cast<const double2 *>(U), g, partial);
    return (int)cudaGetLastError();
}

// one RK3 step of the flow on U (in place), Z = workspace of the size of U
int mdwf_launch_flow_step(void *U, void *Z, const int *L, double eps, double c0, double c1, cudaStream_t st)
{
    Geo g;
    for (int d = 0; d < 4; d++) g.L[d] = L[d];
    g.V4 = (long)L[0] * L[1] * L[2] * L[3];
    const long nl = g.V4 * 4;
    const unsigned nb = (unsigned)((nl + 127) / 128);
    double2 *u = reinterpret_cast<double2 *>(U), *z = reinterpret_cast<double2 *>(Z);
    const double a[3] = {1.0, 8.0 / 9.0, 0.75}, b[3] = {0.0, -17.0 / 36.0, -1.0}, cz[3] = {0.25, 1.0, 1.0};
    for (int stage = 0; stage < 3; stage++) {
        flow_force_kernel<<<nb, 128, 0, st>>>(u, z, g, eps, c0, c1, a[stage], b[stage]);
        flow_update_kernel<<<nb, 128, 0, st>>>(u, z, nl, cz[stage]);
    }
    return (int)cudaGetLastError();
}
