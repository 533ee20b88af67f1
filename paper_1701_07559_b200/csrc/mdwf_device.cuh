// mdwf_device.cuh -- precision traits, spinor / link loads and stores, spin projection.
// Hand-written for sm_100a.  A spinor in registers is R v[24]: v[2*(spin*3+colour)+{0:re,1:im}].
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define MDWF_DEV __device__ __forceinline__

// ---- precision traits ------------------------------------------------------------------------
struct PD {   // fp64 storage and arithmetic
    using R = double; using V = double2; using G = double2;
    static constexpr int NV = 12;      // chunks per spinor
    static constexpr int CH = 2;       // reals per chunk
    static constexpr bool HALF = false;
    static constexpr int MAXT = 256;   // max threads per block of the hop kernels
};
struct PS {   // fp32 storage and arithmetic
    using R = float; using V = float4; using G = float2;
    static constexpr int NV = 6;
    static constexpr int CH = 4;
    static constexpr bool HALF = false;
    static constexpr int MAXT = 512;
};
struct PH {   // 16-bit fixed-point storage (+ one fp32 scale per 5D site), fp32 arithmetic
    using R = float; using V = short4; using G = short2;
    static constexpr int NV = 6;
    static constexpr int CH = 4;
    static constexpr bool HALF = true;
    static constexpr int MAXT = 512;
};
#define MDWF_FIXED_MAX 32767.0f

// ---- chunk <-> reals -------------------------------------------------------------------------
MDWF_DEV void unpack(const double2 c, double *r, double) { r[0] = c.x; r[1] = c.y; }
MDWF_DEV void unpack(const float4 c, float *r, float) { r[0] = c.x; r[1] = c.y; r[2] = c.z; r[3] = c.w; }
MDWF_DEV void unpack(const short4 c, float *r, float sc)
{
    r[0] = sc * (float)c.x; r[1] = sc * (float)c.y; r[2] = sc * (float)c.z; r[3] = sc * (float)c.w;
}
MDWF_DEV double2 pack(const double *r, double, double2 *) { return make_double2(r[0], r[1]); }
MDWF_DEV float4 pack(const float *r, float, float4 *) { return make_float4(r[0], r[1], r[2], r[3]); }
MDWF_DEV short4 pack(const float *r, float isc, short4 *)
{
    return make_short4((short)__float2int_rn(r[0] * isc), (short)__float2int_rn(r[1] * isc),
                       (short)__float2int_rn(r[2] * isc), (short)__float2int_rn(r[3] * isc));
}

// Load chunks [j0, j0+nj) of the spinor at (s, cb) into out[nj*CH].  For the 16-bit format the values
// are multiplied by norm/32767.
template <class P>
MDWF_DEV void load_chunks(const void *base, const float *norm, int s, long cb, long Vh, int j0, int nj,
                          typename P::R *out)
{
    using V = typename P::V;
    using R = typename P::R;
    const V *p = reinterpret_cast<const V *>(base) + ((long)s * P::NV + j0) * Vh + cb;
    R sc = (R)1;
    if (P::HALF) sc = (R)(__ldg(norm + (long)s * Vh + cb) * (1.0f / MDWF_FIXED_MAX));
#pragma unroll
    for (int j = 0; j < P::NV; j++)
        if (j < nj) unpack(__ldg(p + (long)j * Vh), out + j * P::CH, sc);
}
template <class P>
MDWF_DEV void load_spinor(const void *base, const float *norm, int s, long cb, long Vh, typename P::R *v)
{
    load_chunks<P>(base, norm, s, cb, Vh, 0, P::NV, v);
}
// upper (spins 0,1: reals 0..11) or lower (spins 2,3: reals 12..23) half into out[12]
template <class P>
MDWF_DEV void load_half(const void *base, const float *norm, int s, long cb, long Vh, int lower,
                        typename P::R *out)
{
    load_chunks<P>(base, norm, s, cb, Vh, lower ? P::NV / 2 : 0, P::NV / 2, out);
}

template <class P>
MDWF_DEV void store_spinor(void *base, float *norm, int s, long cb, long Vh, const typename P::R *v)
{
    using V = typename P::V;
    using R = typename P::R;
    V *p = reinterpret_cast<V *>(base) + ((long)s * P::NV) * Vh + cb;
    R isc = (R)1;
    if (P::HALF) {
        float m = 0.f;
#pragma unroll
        for (int k = 0; k < 24; k++) m = fmaxf(m, fabsf((float)v[k]));
        norm[(long)s * Vh + cb] = m;
        isc = (R)(m > 0.f ? MDWF_FIXED_MAX / m : 0.f);
    }
#pragma unroll
    for (int j = 0; j < P::NV; j++) p[(long)j * Vh] = pack(v + j * P::CH, isc, (V *)nullptr);
}

// ---- SU(3) links ------------------------------------------------------------------------------
MDWF_DEV void gunpack(const double2 c, double *r) { r[0] = c.x; r[1] = c.y; }
MDWF_DEV void gunpack(const float2 c, float *r) { r[0] = c.x; r[1] = c.y; }
MDWF_DEV void gunpack(const short2 c, float *r)
{
    r[0] = (float)c.x * (1.0f / MDWF_FIXED_MAX); r[1] = (float)c.y * (1.0f / MDWF_FIXED_MAX);
}
// U[2*(row*3+col)+ri]; with RECON == 12 the third row is conj(row0 x row1).
template <class P>
MDWF_DEV void load_link(const void *gbase, int mu, long cb, long Vh, int recon, typename P::R *U)
{
    using G = typename P::G;
    using R = typename P::R;
    const int NK = recon >> 1;
    const G *p = reinterpret_cast<const G *>(gbase) + ((long)mu * NK) * Vh + cb;
#pragma unroll
    for (int k = 0; k < 6; k++) gunpack(__ldg(p + (long)k * Vh), U + 2 * k);
    if (recon == 18) {
#pragma unroll
        for (int k = 6; k < 9; k++) gunpack(__ldg(p + (long)k * Vh), U + 2 * k);
    } else {
        // row2[c] = conj(row0[a] row1[b] - row0[b] row1[a]),  (a,b) = (c+1, c+2) mod 3
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const int a = (c + 1) % 3, b = (c + 2) % 3;
            const R ar = U[2 * a], ai = U[2 * a + 1], br = U[2 * b], bi = U[2 * b + 1];
            const R cr = U[6 + 2 * a], ci = U[6 + 2 * a + 1], dr = U[6 + 2 * b], di = U[6 + 2 * b + 1];
            // row0[a]*row1[b] - row0[b]*row1[a]
            const R re = (ar * dr - ai * di) - (br * cr - bi * ci);
            const R im = (ar * di + ai * dr) - (br * ci + bi * cr);
            U[12 + 2 * c] = re;
            U[12 + 2 * c + 1] = -im;
        }
    }
}

// chi[spin2][a] = sum_c U[a][c] h[spin2][c]          (DAGGER_U = false)
//               = sum_c conj(U[c][a]) h[spin2][c]    (DAGGER_U = true)
template <bool DAGGER_U, class R>
MDWF_DEV void su3_mul(const R *U, const R *h, R *chi)
{
#pragma unroll
    for (int sp = 0; sp < 2; sp++)
#pragma unroll
        for (int a = 0; a < 3; a++) {
            R re = 0, im = 0;
#pragma unroll
            for (int c = 0; c < 3; c++) {
                const R hr = h[2 * (sp * 3 + c)], hi = h[2 * (sp * 3 + c) + 1];
                if (!DAGGER_U) {
                    const R ur = U[2 * (a * 3 + c)], ui = U[2 * (a * 3 + c) + 1];
                    re += ur * hr - ui * hi;
                    im += ur * hi + ui * hr;
                } else {
                    const R ur = U[2 * (c * 3 + a)], ui = U[2 * (c * 3 + a) + 1];
                    re += ur * hr + ui * hi;
                    im += ur * hi - ui * hr;
                }
            }
            chi[2 * (sp * 3 + a)] = re;
            chi[2 * (sp * 3 + a) + 1] = im;
        }
}

// ---- spin projection (1 - SGN gamma_mu) in the DeGrand-Rossi basis ---------------------------
// project: h[spin2 = 0,1][colour] (12 reals) from v[24], scaled by sc.
// recon_add: acc += the 4-spinor whose upper half is chi and whose lower half follows from chi.
//   mu=0: h0 = v0 - S i v3, h1 = v1 - S i v2;  r2 =  S i h1, r3 =  S i h0
//   mu=1: h0 = v0 + S v3,   h1 = v1 - S v2;    r2 = -S h1,   r3 =  S h0
//   mu=2: h0 = v0 - S i v2, h1 = v1 + S i v3;  r2 =  S i h0, r3 = -S i h1
//   mu=3: h0 = v0 - S v2,   h1 = v1 - S v3;    r2 = -S h0,   r3 = -S h1
template <int MU, int SGN, class R>
MDWF_DEV void project(const R *v, R sc, R *h)
{
    const R S = (R)SGN;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const R v0r = v[2 * c], v0i = v[2 * c + 1], v1r = v[6 + 2 * c], v1i = v[6 + 2 * c + 1];
        const R v2r = v[12 + 2 * c], v2i = v[12 + 2 * c + 1], v3r = v[18 + 2 * c], v3i = v[18 + 2 * c + 1];
        R h0r, h0i, h1r, h1i;
        if (MU == 0) {        // -S i (a + i b) = S (b - i a)
            h0r = v0r + S * v3i; h0i = v0i - S * v3r; h1r = v1r + S * v2i; h1i = v1i - S * v2r;
        } else if (MU == 1) {
            h0r = v0r + S * v3r; h0i = v0i + S * v3i; h1r = v1r - S * v2r; h1i = v1i - S * v2i;
        } else if (MU == 2) {
            h0r = v0r + S * v2i; h0i = v0i - S * v2r; h1r = v1r - S * v3i; h1i = v1i + S * v3r;
        } else {
            h0r = v0r - S * v2r; h0i = v0i - S * v2i; h1r = v1r - S * v3r; h1i = v1i - S * v3i;
        }
        h[2 * c] = sc * h0r; h[2 * c + 1] = sc * h0i; h[6 + 2 * c] = sc * h1r; h[6 + 2 * c + 1] = sc * h1i;
    }
}
template <int MU, int SGN, class R>
MDWF_DEV void recon_add(const R *chi, R *acc)
{
    const R S = (R)SGN;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const R h0r = chi[2 * c], h0i = chi[2 * c + 1], h1r = chi[6 + 2 * c], h1i = chi[6 + 2 * c + 1];
        acc[2 * c] += h0r; acc[2 * c + 1] += h0i; acc[6 + 2 * c] += h1r; acc[6 + 2 * c + 1] += h1i;
        if (MU == 0) {        // S i (a + i b) = S (-b + i a)
            acc[12 + 2 * c] -= S * h1i; acc[12 + 2 * c + 1] += S * h1r;
            acc[18 + 2 * c] -= S * h0i; acc[18 + 2 * c + 1] += S * h0r;
        } else if (MU == 1) {
            acc[12 + 2 * c] -= S * h1r; acc[12 + 2 * c + 1] -= S * h1i;
            acc[18 + 2 * c] += S * h0r; acc[18 + 2 * c + 1] += S * h0i;
        } else if (MU == 2) {
            acc[12 + 2 * c] -= S * h0i; acc[12 + 2 * c + 1] += S * h0r;
            acc[18 + 2 * c] += S * h1i; acc[18 + 2 * c + 1] -= S * h1r;
        } else {
            acc[12 + 2 * c] -= S * h0r; acc[12 + 2 * c + 1] -= S * h0i;
            acc[18 + 2 * c] -= S * h1r; acc[18 + 2 * c + 1] -= S * h1i;
        }
    }
}
