// mdwf_device.cuh -- precision traits, device data layout, spinor / link loads and stores, spin projection.
// Hand-written for sm_100a.  A spinor in registers is R v[24]: v[2*(spin*3+colour)+{0:re,1:im}].
//
// Device layout ("warp-blob" layout).  Checkerboard sites are grouped in 32s
// (g = cb >> 5, lane = cb & 31); one parity vector is
//     chunk[ ((g*L5 + s)*NV + j)*32 + lane ],  j = 0..NV-1
// so the NV chunks of one (site, s) sit at a CONSTANT stride of 32 chunks (512 B): a warp reads 512
// contiguous bytes per instruction and the chunk index becomes an immediate offset in the load.
// All L5 slices of a 32-site group are contiguous (L5*NV*512 B), which keeps the s-neighbourhood of a
// site group in a few DRAM pages.  The 16-bit format adds norm[(g*L5 + s)*32 + lane] (fp32 scale).
// Gauge links of the sites of one parity: link[ ((g*8 + d)*NK + k)*32 + lane ], one complex per chunk; d = mu is
// U_mu(x), d = 4 + mu is U_mu(x - mu)^dagger pulled back to x (the 8 links of a 32-site group are one slab).
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
};
struct PS {   // fp32 storage and arithmetic
    using R = float; using V = float4; using G = float2;
    static constexpr int NV = 6;
    static constexpr int CH = 4;
    static constexpr bool HALF = false;
};
struct PH {   // 16-bit fixed-point storage, offset binary (+ one fp32 scale per 5D site), fp32 arithmetic
    using R = float; using V = short4; using G = short2;
    static constexpr int NV = 6;
    static constexpr int CH = 4;
    static constexpr bool HALF = true;
};
#define MDWF_FIXED_MAX 32767.0f

// chunk offset of chunk 0 of (s, cb); chunk j is at +32*j.  norm offset = sp_noff.
MDWF_DEV long sp_off(int L5, int NV, long cb, int s) { return ((((cb >> 5) * L5 + s) * NV) << 5) + (cb & 31); }
MDWF_DEV long sp_noff(int L5, long cb, int s) { return (((cb >> 5) * L5 + s) << 5) + (cb & 31); }

// ---- chunk <-> reals -------------------------------------------------------------------------
MDWF_DEV void unpack(const double2 c, double *r, double) { r[0] = c.x; r[1] = c.y; }
MDWF_DEV void unpack(const float4 c, float *r, float) { r[0] = c.x; r[1] = c.y; r[2] = c.z; r[3] = c.w; }
// int16 -> fp32 on the integer and FMA pipes (the I2F conversion pipe runs at a quarter of their rate):
// the 16 bits are stored offset-binary (u = q + 32768), so 0x4B400000 | u is the float 12582912 + 32768 + q;
// subtracting 12615680 is exact.
MDWF_DEV float fixed_to_float(unsigned bits16)
{
    return __uint_as_float(0x4B400000u | bits16) - 12615680.0f;
}
MDWF_DEV void unpack(const short4 c, float *r, float sc)
{
    r[0] = sc * fixed_to_float((unsigned short)c.x); r[1] = sc * fixed_to_float((unsigned short)c.y);
    r[2] = sc * fixed_to_float((unsigned short)c.z); r[3] = sc * fixed_to_float((unsigned short)c.w);
}
MDWF_DEV double2 pack(const double *r, double, double2 *) { return make_double2(r[0], r[1]); }
MDWF_DEV float4 pack(const float *r, float, float4 *) { return make_float4(r[0], r[1], r[2], r[3]); }
// fp32 -> 16 bits: the low 16 bits of fma(v, isc, 1.5 * 2^23 + 32768) are round-to-nearest(v * isc) + 32768
MDWF_DEV short float_to_fixed(float v, float isc) { return (short)(__float_as_uint(fmaf(v, isc, 12615680.0f)) & 0xFFFFu); }
MDWF_DEV short4 pack(const float *r, float isc, short4 *)
{
    return make_short4(float_to_fixed(r[0], isc), float_to_fixed(r[1], isc), float_to_fixed(r[2], isc),
                       float_to_fixed(r[3], isc));
}

// Load NJ chunks starting at chunk pointer p (stride 32 chunks) into out[NJ*CH], scaled by sc (16-bit only).
template <class P, int NJ>
MDWF_DEV void load_chunks_at(const typename P::V *p, typename P::R sc, typename P::R *out)
{
#pragma unroll
    for (int j = 0; j < NJ; j++) unpack(__ldg(p + 32 * j), out + j * P::CH, sc);
}
template <class P>
MDWF_DEV typename P::R load_scale(const float *norm, long noff)
{
    if (P::HALF) return (typename P::R)(__ldg(norm + noff) * (1.0f / MDWF_FIXED_MAX));
    return (typename P::R)1;
}

template <class P>
MDWF_DEV void load_spinor(const void *base, const float *norm, int L5, int s, long cb, typename P::R *v)
{
    const typename P::V *p = reinterpret_cast<const typename P::V *>(base) + sp_off(L5, P::NV, cb, s);
    load_chunks_at<P, P::NV>(p, load_scale<P>(norm, sp_noff(L5, cb, s)), v);
}
// upper (spins 0,1: reals 0..11) or lower (spins 2,3: reals 12..23) half into out[12]
template <class P>
MDWF_DEV void load_half(const void *base, const float *norm, int L5, int s, long cb, int lower, typename P::R *out)
{
    const typename P::V *p = reinterpret_cast<const typename P::V *>(base) + sp_off(L5, P::NV, cb, s) +
                             (lower ? 32 * (P::NV / 2) : 0);
    load_chunks_at<P, P::NV / 2>(p, load_scale<P>(norm, sp_noff(L5, cb, s)), out);
}

template <class P>
MDWF_DEV void store_spinor(void *base, float *norm, int L5, int s, long cb, const typename P::R *v)
{
    using V = typename P::V;
    using R = typename P::R;
    V *p = reinterpret_cast<V *>(base) + sp_off(L5, P::NV, cb, s);
    R isc = (R)1;
    if (P::HALF) {
        float m = 0.f;
#pragma unroll
        for (int k = 0; k < 24; k++) m = fmaxf(m, fabsf((float)v[k]));
        norm[sp_noff(L5, cb, s)] = m;
        isc = (R)(m > 0.f ? MDWF_FIXED_MAX / m : 0.f);
    }
#pragma unroll
    for (int j = 0; j < P::NV; j++) p[32 * j] = pack(v + j * P::CH, isc, (V *)nullptr);
}

// ---- SU(3) links ------------------------------------------------------------------------------
MDWF_DEV void gunpack(const double2 c, double *r) { r[0] = c.x; r[1] = c.y; }
MDWF_DEV void gunpack(const float2 c, float *r) { r[0] = c.x; r[1] = c.y; }
MDWF_DEV void gunpack(const short2 c, float *r)
{
    r[0] = fixed_to_float((unsigned short)c.x) * (1.0f / MDWF_FIXED_MAX);
    r[1] = fixed_to_float((unsigned short)c.y) * (1.0f / MDWF_FIXED_MAX);
}
// U[2*(row*3+col)+ri] of direction d (0-3 forward, 4-7 backward, already daggered) at site cb; with recon == 12 the
// third row is conj(row0 x row1).
template <class P>
MDWF_DEV void load_link(const void *gbase, int d, long cb, int recon, typename P::R *U)
{
    using G = typename P::G;
    using R = typename P::R;
    const int NK = recon >> 1;
    const G *p = reinterpret_cast<const G *>(gbase) + ((((cb >> 5) * 8 + d) * NK) << 5) + (cb & 31);
#pragma unroll
    for (int k = 0; k < 6; k++) gunpack(__ldg(p + 32 * k), U + 2 * k);
    if (recon == 18) {
#pragma unroll
        for (int k = 6; k < 9; k++) gunpack(__ldg(p + 32 * k), U + 2 * k);
    } else {
        // row2[c] = conj(row0[a] row1[b] - row0[b] row1[a]),  (a,b) = (c+1, c+2) mod 3
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const int a = (c + 1) % 3, b = (c + 2) % 3;
            const R ar = U[2 * a], ai = U[2 * a + 1], br = U[2 * b], bi = U[2 * b + 1];
            const R cr = U[6 + 2 * a], ci = U[6 + 2 * a + 1], dr = U[6 + 2 * b], di = U[6 + 2 * b + 1];
            R re = ar * dr;
            re = fma(-ai, di, re); re = fma(-br, cr, re); re = fma(bi, ci, re);
            R im = ar * di;
            im = fma(ai, dr, im); im = fma(-br, ci, im); im = fma(-bi, cr, im);
            U[12 + 2 * c] = re;
            U[12 + 2 * c + 1] = -im;
        }
    }
}

// chi[spin2][a] = sum_c U[a][c] h[spin2][c]          (DAGGER_U = false)
//               = sum_c conj(U[c][a]) h[spin2][c]    (DAGGER_U = true)
// written as explicit FMA chains: 12 FMUL + 60 FFMA per call
template <bool DAGGER_U, class R>
MDWF_DEV void su3_mul(const R *U, const R *h, R *chi)
{
#pragma unroll
    for (int sp = 0; sp < 2; sp++)
#pragma unroll
        for (int a = 0; a < 3; a++) {
            R re, im;
#pragma unroll
            for (int c = 0; c < 3; c++) {
                const R hr = h[2 * (sp * 3 + c)], hi = h[2 * (sp * 3 + c) + 1];
                const R ur = DAGGER_U ? U[2 * (c * 3 + a)] : U[2 * (a * 3 + c)];
                const R ui = DAGGER_U ? -U[2 * (c * 3 + a) + 1] : U[2 * (a * 3 + c) + 1];
                if (c == 0) { re = ur * hr; im = ur * hi; }
                else { re = fma(ur, hr, re); im = fma(ur, hi, im); }
                re = fma(-ui, hi, re);
                im = fma(ui, hr, im);
            }
            chi[2 * (sp * 3 + a)] = re;
            chi[2 * (sp * 3 + a) + 1] = im;
        }
}

// ---- spin projection (1 - SGN gamma_mu) in the DeGrand-Rossi basis ---------------------------
// project: h[spin2 = 0,1][colour] (12 reals) from v[24].
// recon_add: acc += sc * (the 4-spinor whose upper half is chi and whose lower half follows from chi).
//   mu=0: h0 = v0 - S i v3, h1 = v1 - S i v2;  r2 =  S i h1, r3 =  S i h0
//   mu=1: h0 = v0 + S v3,   h1 = v1 - S v2;    r2 = -S h1,   r3 =  S h0
//   mu=2: h0 = v0 - S i v2, h1 = v1 + S i v3;  r2 =  S i h0, r3 = -S i h1
//   mu=3: h0 = v0 - S v2,   h1 = v1 - S v3;    r2 = -S h0,   r3 = -S h1
template <int MU, int SGN, class R>
MDWF_DEV void project(const R *v, R *h)
{
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const R v0r = v[2 * c], v0i = v[2 * c + 1], v1r = v[6 + 2 * c], v1i = v[6 + 2 * c + 1];
        const R v2r = v[12 + 2 * c], v2i = v[12 + 2 * c + 1], v3r = v[18 + 2 * c], v3i = v[18 + 2 * c + 1];
        R h0r, h0i, h1r, h1i;
        if (MU == 0) {        // -S i (a + i b) = S (b - i a)
            if (SGN > 0) { h0r = v0r + v3i; h0i = v0i - v3r; h1r = v1r + v2i; h1i = v1i - v2r; }
            else { h0r = v0r - v3i; h0i = v0i + v3r; h1r = v1r - v2i; h1i = v1i + v2r; }
        } else if (MU == 1) {
            if (SGN > 0) { h0r = v0r + v3r; h0i = v0i + v3i; h1r = v1r - v2r; h1i = v1i - v2i; }
            else { h0r = v0r - v3r; h0i = v0i - v3i; h1r = v1r + v2r; h1i = v1i + v2i; }
        } else if (MU == 2) {
            if (SGN > 0) { h0r = v0r + v2i; h0i = v0i - v2r; h1r = v1r - v3i; h1i = v1i + v3r; }
            else { h0r = v0r - v2i; h0i = v0i + v2r; h1r = v1r + v3i; h1i = v1i - v3r; }
        } else {
            if (SGN > 0) { h0r = v0r - v2r; h0i = v0i - v2i; h1r = v1r - v3r; h1i = v1i - v3i; }
            else { h0r = v0r + v2r; h0i = v0i + v2i; h1r = v1r + v3r; h1i = v1i + v3i; }
        }
        h[2 * c] = h0r; h[2 * c + 1] = h0i; h[6 + 2 * c] = h1r; h[6 + 2 * c + 1] = h1i;
    }
}
// WITHSC = false: sc is ignored (plain adds); true: acc = fma(+-sc, chi, acc)  (antiperiodic t hop)
template <int MU, int SGN, bool WITHSC, class R>
MDWF_DEV void recon_add(const R *chi, R sc, R *acc)
{
    const R p = WITHSC ? sc : (R)1;              // + sc
    const R s = (SGN > 0) ? p : -p;              // S * sc
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const R h0r = chi[2 * c], h0i = chi[2 * c + 1], h1r = chi[6 + 2 * c], h1i = chi[6 + 2 * c + 1];
#define ACC(idx, coef, val) acc[idx] = WITHSC ? fma(coef, val, acc[idx]) : ((coef) > 0 ? acc[idx] + (val) : acc[idx] - (val))
        ACC(2 * c, p, h0r); ACC(2 * c + 1, p, h0i); ACC(6 + 2 * c, p, h1r); ACC(6 + 2 * c + 1, p, h1i);
        if (MU == 0) {        // S i (a + i b) = S (-b + i a)
            ACC(12 + 2 * c, -s, h1i); ACC(12 + 2 * c + 1, s, h1r);
            ACC(18 + 2 * c, -s, h0i); ACC(18 + 2 * c + 1, s, h0r);
        } else if (MU == 1) {
            ACC(12 + 2 * c, -s, h1r); ACC(12 + 2 * c + 1, -s, h1i);
            ACC(18 + 2 * c, s, h0r); ACC(18 + 2 * c + 1, s, h0i);
        } else if (MU == 2) {
            ACC(12 + 2 * c, -s, h0i); ACC(12 + 2 * c + 1, s, h0r);
            ACC(18 + 2 * c, s, h1i); ACC(18 + 2 * c + 1, -s, h1r);
        } else {
            ACC(12 + 2 * c, -s, h0r); ACC(12 + 2 * c + 1, -s, h0i);
            ACC(18 + 2 * c, -s, h1r); ACC(18 + 2 * c + 1, -s, h1i);
        }
#undef ACC
    }
}
