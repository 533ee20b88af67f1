// layout_kernels.cu -- S0: canonical interchange layouts (include/mdwf.h) <-> even-odd device layouts.
// One thread per (s, checkerboard site).  Runs once per load / apply / solve, not on the CG hot loop.
#include "mdwf_device.cuh"
#include "mdwf_internal.h"

static size_t padded(int Vh) { return ((size_t)Vh + 31) / 32 * 32; }   // sites are stored in groups of 32
size_t mdwf_spinor_bytes(Prec p, int L5, int Vh)
{
    const size_t n = (size_t)L5 * padded(Vh) * 24;
    return p == PREC_D ? n * 8 : (p == PREC_S ? n * 4 : n * 2);
}
size_t mdwf_gauge_bytes(Prec p, int Vh, int recon)
{
    const size_t n = (size_t)8 * padded(Vh) * recon;         // 4 forward links + 4 pulled-back backward links per site
    return p == PREC_D ? n * 8 : (p == PREC_S ? n * 4 : n * 2);
}

// lexicographic 4D index of checkerboard site cb of the given parity
__device__ __forceinline__ long cb_to_lex(long cb, int parity, int Lx, int Ly, int Lz)
{
    const int Lxh = Lx >> 1;
    long r = cb;
    const int xh = (int)(r % Lxh); r /= Lxh;
    const int y = (int)(r % Ly);   r /= Ly;
    const int z = (int)(r % Lz);
    const int t = (int)(r / Lz);
    const int x = 2 * xh + ((parity + y + z + t) & 1);
    return x + (long)Lx * (y + (long)Ly * (z + (long)Lz * t));
}

// canonical site block of 24 reals at element offset `off` (in units of sites) -> device layout
template <class P, class T>
__global__ void spinor_in_kernel(const T *canon, void *dst, float *dst_norm, int L5, long Vh, int full, int parity,
                                 int Lx, int Ly, int Lz, long V4)
{
    using R = typename P::R;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long)L5 * Vh) return;
    const int s = (int)(idx / Vh);
    const long cb = idx - (long)s * Vh;
    const long site = full ? ((long)s * V4 + cb_to_lex(cb, parity, Lx, Ly, Lz)) : idx;
    const T *p = canon + site * 24;
    R v[24];
#pragma unroll
    for (int k = 0; k < 24; k++) v[k] = (R)p[k];
    store_spinor<P>(dst, dst_norm, L5, s, cb, v);
}
template <class P, class T>
__global__ void spinor_out_kernel(const void *src, const float *src_norm, T *canon, int L5, long Vh, int full,
                                  int parity, int Lx, int Ly, int Lz, long V4)
{
    using R = typename P::R;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long)L5 * Vh) return;
    const int s = (int)(idx / Vh);
    const long cb = idx - (long)s * Vh;
    const long site = full ? ((long)s * V4 + cb_to_lex(cb, parity, Lx, Ly, Lz)) : idx;
    T *p = canon + site * 24;
    R v[24];
    load_spinor<P>(src, src_norm, L5, s, cb, v);
#pragma unroll
    for (int k = 0; k < 24; k++) p[k] = (T)v[k];
}

MDWF_DEV double2 gpack(double re, double im, double2 *) { return make_double2(re, im); }
MDWF_DEV float2 gpack(double re, double im, float2 *) { return make_float2((float)re, (float)im); }
MDWF_DEV short2 gpack(double re, double im, short2 *)
{
    // offset binary, like the spinors (mdwf_device.cuh)
    // clamped: a component above 1 (a non-unitary field) saturates instead of wrapping
    const int qr = max(-32767, min(32767, __double2int_rn(re * (double)MDWF_FIXED_MAX)));
    const int qi = max(-32767, min(32767, __double2int_rn(im * (double)MDWF_FIXED_MAX)));
    return make_short2((short)(unsigned short)(qr + 32768), (short)(unsigned short)(qi + 32768));
}

// Link tile of a site x of the given parity, 8 directions d:
//   d = mu     : U_mu(x)                      (forward hop)
//   d = 4 + mu : U_mu(x - mu)^dagger          (backward hop, pulled back to x and already daggered)
// so the 8 links of a 32-site group are ONE contiguous slab [8][NK][32] (one bulk copy per block in the hop kernels).
// With recon = 12 rows 0 and 1 of the stored matrix are kept (row 2 = conj(row0 x row1) holds for U and for U^dagger).
template <class P, class T>
__global__ void gauge_in_kernel(const T *canon, void *dst, long Vh, int parity, int recon, int Lx, int Ly, int Lz, int Lt)
{
    using G = typename P::G;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 8 * Vh) return;
    const int d = (int)(idx / Vh), mu = d & 3;
    const long cb = idx - (long)d * Vh;
    long lex = cb_to_lex(cb, parity, Lx, Ly, Lz);
    if (d >= 4) {                                   // site x - mu (periodic; the antiperiodic sign lives in the kernels)
        long r = lex;
        const int x = (int)(r % Lx); r /= Lx;
        const int y = (int)(r % Ly); r /= Ly;
        const int z = (int)(r % Lz);
        const int t = (int)(r / Lz);
        const int xm = (mu == 0) ? (x + Lx - 1) % Lx : x, ym = (mu == 1) ? (y + Ly - 1) % Ly : y;
        const int zm = (mu == 2) ? (z + Lz - 1) % Lz : z, tm = (mu == 3) ? (t + Lt - 1) % Lt : t;
        lex = xm + (long)Lx * (ym + (long)Ly * (zm + (long)Lz * tm));
    }
    const T *p = canon + (lex * 4 + mu) * 18;
    const int NK = recon >> 1;
    G *q = reinterpret_cast<G *>(dst) + ((((cb >> 5) * 8 + d) * NK) << 5) + (cb & 31);
    for (int k = 0; k < NK; k++) {
        const int a = k / 3, c = k - 3 * a;
        if (d < 4) q[32 * k] = gpack((double)p[2 * k], (double)p[2 * k + 1], (G *)nullptr);
        else q[32 * k] = gpack((double)p[2 * (c * 3 + a)], -(double)p[2 * (c * 3 + a) + 1], (G *)nullptr);   // conj(U_ca)
    }
}

template <class P>
static int spinor_in(const void *canon, int real_bytes, const SpinorBuf &dst, int L5, long Vh, int full, int parity,
                     const int *L, cudaStream_t st)
{
    const long n = (long)L5 * Vh;
    const int T = 128;
    const unsigned nb = (unsigned)((n + T - 1) / T);
    const int Lx = L ? L[0] : 2, Ly = L ? L[1] : 1, Lz = L ? L[2] : 1;
    const long V4 = 2 * Vh;
    if (real_bytes == 8)
        spinor_in_kernel<P, double><<<nb, T, 0, st>>>((const double *)canon, dst.v, dst.norm, L5, Vh, full, parity, Lx, Ly, Lz, V4);
    else
        spinor_in_kernel<P, float><<<nb, T, 0, st>>>((const float *)canon, dst.v, dst.norm, L5, Vh, full, parity, Lx, Ly, Lz, V4);
    return (int)cudaGetLastError();
}
template <class P>
static int spinor_out(const SpinorBuf &src, void *canon, int real_bytes, int L5, long Vh, int full, int parity,
                      const int *L, cudaStream_t st)
{
    const long n = (long)L5 * Vh;
    const int T = 128;
    const unsigned nb = (unsigned)((n + T - 1) / T);
    const int Lx = L ? L[0] : 2, Ly = L ? L[1] : 1, Lz = L ? L[2] : 1;
    const long V4 = 2 * Vh;
    if (real_bytes == 8)
        spinor_out_kernel<P, double><<<nb, T, 0, st>>>(src.v, src.norm, (double *)canon, L5, Vh, full, parity, Lx, Ly, Lz, V4);
    else
        spinor_out_kernel<P, float><<<nb, T, 0, st>>>(src.v, src.norm, (float *)canon, L5, Vh, full, parity, Lx, Ly, Lz, V4);
    return (int)cudaGetLastError();
}

#define DISPATCH_P(p, CALL)                      \
    switch (p) {                                 \
    case PREC_D: return CALL(PD);                \
    case PREC_S: return CALL(PS);                \
    default: return CALL(PH);                    \
    }

int mdwf_launch_parity_in(Prec p, const void *canon, int real_bytes, const SpinorBuf &dst, int L5, int Vh,
                          cudaStream_t st)
{
#define C(PP) spinor_in<PP>(canon, real_bytes, dst, L5, Vh, 0, 0, nullptr, st)
    DISPATCH_P(p, C)
#undef C
}
int mdwf_launch_parity_out(Prec p, const SpinorBuf &src, void *canon, int real_bytes, int L5, int Vh,
                           cudaStream_t st)
{
#define C(PP) spinor_out<PP>(src, canon, real_bytes, L5, Vh, 0, 0, nullptr, st)
    DISPATCH_P(p, C)
#undef C
}
int mdwf_launch_full_in(Prec p, const void *canon, int real_bytes, const SpinorBuf &dst, const int *L, int L5,
                        int parity, cudaStream_t st)
{
    const long Vh = (long)L[0] * L[1] * L[2] * L[3] / 2;
#define C(PP) spinor_in<PP>(canon, real_bytes, dst, L5, Vh, 1, parity, L, st)
    DISPATCH_P(p, C)
#undef C
}
int mdwf_launch_full_out(Prec p, const SpinorBuf &src, void *canon, int real_bytes, const int *L, int L5,
                         int parity, cudaStream_t st)
{
    const long Vh = (long)L[0] * L[1] * L[2] * L[3] / 2;
#define C(PP) spinor_out<PP>(src, canon, real_bytes, L5, Vh, 1, parity, L, st)
    DISPATCH_P(p, C)
#undef C
}

template <class P>
static int gauge_in(const void *canon, int real_bytes, void *dst, const int *L, int parity, int recon, cudaStream_t st)
{
    const long Vh = (long)L[0] * L[1] * L[2] * L[3] / 2;
    const int T = 128;
    const unsigned nb = (unsigned)((8 * Vh + T - 1) / T);
    if (real_bytes == 8)
        gauge_in_kernel<P, double><<<nb, T, 0, st>>>((const double *)canon, dst, Vh, parity, recon, L[0], L[1], L[2], L[3]);
    else
        gauge_in_kernel<P, float><<<nb, T, 0, st>>>((const float *)canon, dst, Vh, parity, recon, L[0], L[1], L[2], L[3]);
    return (int)cudaGetLastError();
}
int mdwf_launch_gauge_in(Prec p, const void *canon, int real_bytes, void *dst, const int *L, int parity, int recon,
                         cudaStream_t st)
{
#define C(PP) gauge_in<PP>(canon, real_bytes, dst, L, parity, recon, st)
    DISPATCH_P(p, C)
#undef C
}

// ---- the 16-bit storage format as stored: words[(s*Vh + cb)*24 + k] (offset binary), scales[s*Vh + cb] ---------------
__global__ void half_export_kernel(const void *src, const float *src_norm, unsigned short *words, float *scales, int L5, long Vh)
{
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long)L5 * Vh) return;
    const int s = (int)(idx / Vh);
    const long cb = idx - (long)s * Vh;
    const short4 *p = reinterpret_cast<const short4 *>(src) + sp_off(L5, PH::NV, cb, s);
#pragma unroll
    for (int j = 0; j < PH::NV; j++) {
        const short4 q = p[32 * j];
        words[idx * 24 + 4 * j] = (unsigned short)q.x; words[idx * 24 + 4 * j + 1] = (unsigned short)q.y;
        words[idx * 24 + 4 * j + 2] = (unsigned short)q.z; words[idx * 24 + 4 * j + 3] = (unsigned short)q.w;
    }
    scales[idx] = src_norm[sp_noff(L5, cb, s)];
}
__global__ void half_import_kernel(const unsigned short *words, const float *scales, void *dst, float *dst_norm, int L5, long Vh)
{
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long)L5 * Vh) return;
    const int s = (int)(idx / Vh);
    const long cb = idx - (long)s * Vh;
    short4 *p = reinterpret_cast<short4 *>(dst) + sp_off(L5, PH::NV, cb, s);
#pragma unroll
    for (int j = 0; j < PH::NV; j++)
        p[32 * j] = make_short4((short)words[idx * 24 + 4 * j], (short)words[idx * 24 + 4 * j + 1], (short)words[idx * 24 + 4 * j + 2],
                                (short)words[idx * 24 + 4 * j + 3]);
    dst_norm[sp_noff(L5, cb, s)] = scales[idx];
}
int mdwf_launch_half_export(const SpinorBuf &src, void *words, void *scales, int L5, int Vh, cudaStream_t st)
{
    const long n = (long)L5 * Vh;
    half_export_kernel<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(src.v, src.norm, (unsigned short *)words, (float *)scales, L5, Vh);
    return (int)cudaGetLastError();
}
int mdwf_launch_half_import(const void *words, const void *scales, const SpinorBuf &dst, int L5, int Vh, cudaStream_t st)
{
    const long n = (long)L5 * Vh;
    half_import_kernel<<<(unsigned)((n + 127) / 128), 128, 0, st>>>((const unsigned short *)words, (const float *)scales, dst.v, dst.norm, L5, Vh);
    return (int)cudaGetLastError();
}

// ---- timing inputs: hash-filled vectors ------------------------------------------------------------
template <class P>
__global__ void fill_kernel(void *dst, float *dst_norm, int L5, long Vh, unsigned seed)
{
    using R = typename P::R;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long)L5 * Vh) return;
    const int s = (int)(idx / Vh);
    const long cb = idx - (long)s * Vh;
    R v[24];
#pragma unroll
    for (int k = 0; k < 24; k++) {
        unsigned h = (unsigned)(idx * 24 + k) * 2654435761u + seed;
        h ^= h >> 15; h *= 2246822519u; h ^= h >> 13; h *= 3266489917u; h ^= h >> 16;
        v[k] = (R)((double)h * (2.0 / 4294967295.0) - 1.0);
    }
    store_spinor<P>(dst, dst_norm, L5, s, cb, v);
}
int mdwf_launch_fill(Prec p, const SpinorBuf &dst, int L5, int Vh, unsigned seed, cudaStream_t st)
{
    const long n = (long)L5 * Vh;
    const int T = 128;
    const unsigned nb = (unsigned)((n + T - 1) / T);
    switch (p) {
    case PREC_D: fill_kernel<PD><<<nb, T, 0, st>>>(dst.v, dst.norm, L5, Vh, seed); break;
    case PREC_S: fill_kernel<PS><<<nb, T, 0, st>>>(dst.v, dst.norm, L5, Vh, seed); break;
    default: fill_kernel<PH><<<nb, T, 0, st>>>(dst.v, dst.norm, L5, Vh, seed); break;
    }
    return (int)cudaGetLastError();
}

// ---- 4D <-> 5D maps on canonical buffers (Eq. (5)) --------------------------
// wall source: b(x,s) = delta_{s,0} P+ eta(x) + delta_{s,L5-1} P- eta(x); P+ keeps spins 0,1, P- spins 2,3 (gamma5 = diag(+,+,-,-))
template <class T>
__global__ void wall_inject_kernel(const T *eta, T *b, long V4, int L5)
{
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;       // one complex number of the 4D field: (site, spin, colour)
    if (i >= V4 * 12) return;
    const int spin = (int)((i / 3) % 4);
    const int s = (spin < 2) ? 0 : L5 - 1;
    b[2 * ((long)s * V4 * 12 + i)] = eta[2 * i];
    b[2 * ((long)s * V4 * 12 + i) + 1] = eta[2 * i + 1];
}
// q(x) = P- psi(x, sm) + P+ psi(x, sp): walls (sm = 0, sp = L5-1) or midpoint (sm = L5/2, sp = L5/2 - 1)
template <class T>
__global__ void wall_project_kernel(const T *psi, T *q, long V4, int sm, int sp)
{
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= V4 * 12) return;
    const int spin = (int)((i / 3) % 4);
    const int s = (spin < 2) ? sp : sm;
    q[2 * i] = psi[2 * ((long)s * V4 * 12 + i)];
    q[2 * i + 1] = psi[2 * ((long)s * V4 * 12 + i) + 1];
}
int mdwf_launch_wall_inject(const void *eta, void *b, int real_bytes, long V4, int L5, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(b, 0, (size_t)L5 * V4 * 24 * real_bytes, st);
    if (e != cudaSuccess) return (int)e;
    const int T = 256;
    const unsigned nb = (unsigned)((V4 * 12 + T - 1) / T);
    if (real_bytes == 8) wall_inject_kernel<double><<<nb, T, 0, st>>>((const double *)eta, (double *)b, V4, L5);
    else wall_inject_kernel<float><<<nb, T, 0, st>>>((const float *)eta, (float *)b, V4, L5);
    return (int)cudaGetLastError();
}
int mdwf_launch_wall_project(const void *psi, void *q, int real_bytes, long V4, int sm, int sp, cudaStream_t st)
{
    const int T = 256;
    const unsigned nb = (unsigned)((V4 * 12 + T - 1) / T);
    if (real_bytes == 8) wall_project_kernel<double><<<nb, T, 0, st>>>((const double *)psi, (double *)q, V4, sm, sp);
    else wall_project_kernel<float><<<nb, T, 0, st>>>((const float *)psi, (float *)q, V4, sm, sp);
    return (int)cudaGetLastError();
}
