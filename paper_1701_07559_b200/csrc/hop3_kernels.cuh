// hop3_kernels.cuh -- v3 of the fused Wilson-hopping + fifth-dimension kernels for fp32 ARITHMETIC
// (precisions PS = fp32 storage and PH = 16-bit storage), L5 in {8, 12, 16}.
//
// Same operator family and same thread mapping as hop_kernels.cuh (thread = one 4D site x S consecutive
// s-slices; block = 32 sites x L5/S warps), rebuilt around three B200 facts measured in profiles/:
//   1. sm_100a issues a 3-register FFMA at half rate; the packed FFMA2 (fma.rn.f32x2) carries two FMAs per
//      lane and reaches 65 TFLOP/s against 40 for FFMA.  A complex number is one float2 register pair and
//      every arithmetic step below is a packed f32x2 instruction.  FFMA2 takes a scalar register broadcast to
//      both lanes and a swapped pair as free operand forms, so SU(3) x half-spinor is chi_a = P + iQ with
//      P = sum_c ur (hr,hi), Q = sum_c ui (hr,hi): the link stays 18 scalars, reused for the S slices and both
//      spin components, and multiplication by +-i costs nothing.
//   2. The dense L5 x L5 matrix B A^{-1} (S3 of the hot path) is semiseparable: A = alpha (1 + kappa T) with T
//      the cyclic shift carrying -m_f at the wall, so A^{-1} is a first-order recurrence plus a rank-one wall
//      term.  Each thread runs the recurrence over its own S slices in registers, the warps of a block
//      exchange ONE carry per component through shared memory, and
//          t_s = (b5 z_s + c5 z_{s-1}) / alpha + qW_s W,    z_s = x_s - kappa z_{s-1},  W = z_{L5-1}
//      replaces 2 L5 FMAs per real by about 6 (DESIGN.md section 5 derives it; the fp64 path and any L5 outside
//      {8,12,16} keep the dense table of hop_kernels.cuh).
//   3. The first stall of every direction used to be the link load: the 8 links of the block's 32 sites are built
//      ONCE per block in shared memory (12-real reconstruction and the dagger of backward hops included) and
//      read back with 9 LDS.64 per direction.  No register spills: the s-window of the B-on-load stencil slides
//      slice by slice.
#pragma once
#include "mdwf_device.cuh"
#include "mdwf_internal.h"

namespace h3 {

typedef float2 c2;   // one complex number = one packed f32x2 operand
MDWF_DEV c2 fma2(c2 a, c2 b, c2 c) { return __ffma2_rn(a, b, c); }
MDWF_DEV c2 add2(c2 a, c2 b) { return __fadd2_rn(a, b); }
MDWF_DEV c2 mul2(c2 a, c2 b) { return __fmul2_rn(a, b); }
MDWF_DEV c2 dup(float a) { return make_float2(a, a); }
MDWF_DEV c2 swp(c2 a) { return make_float2(a.y, a.x); }
MDWF_DEV c2 mk(float a, float b) { return make_float2(a, b); }

// ---- spinor chunk loads into complex pairs ------------------------------------------------------
// PS: chunk j = float4 = complexes 2j, 2j+1.  PH: chunk j = short4, value = scale * int16.
// G = true: global memory (read-only path); G = false: a neighbour group staged in shared memory by the copy engine
template <bool G, class T> MDWF_DEV T ldx(const T *p) { if (G) return __ldg(p); else return *p; }
template <class P> struct Ld;
template <> struct Ld<PS> {
    // NC complexes (NC even) from chunk pointer p (stride 32 chunks)
    template <int NC, bool G = true> static MDWF_DEV void chunks(const float4 *p, float, c2 *v)
    {
#pragma unroll
        for (int j = 0; j < NC / 2; j++) {
            const float4 q = ldx<G>(p + 32 * j);
            v[2 * j] = mk(q.x, q.y);
            v[2 * j + 1] = mk(q.z, q.w);
        }
    }
};
// 16-bit fixed point -> fp32 without the conversion pipe.  The 16 bits are stored offset-binary (u = q + 32768), so
// 0x4B400000 | u is the float 12582912 + 32768 + q and value = (that - 12615680) * scale, both steps exact up to the
// one rounding of the product: one PRMT per value, one FADD2 (+ one FMUL2) per complex.
MDWF_DEV c2 cvt_raw(unsigned w)                // w = two 16-bit values (low half = first) -> the two integers as floats
{
    const c2 f = mk(__uint_as_float(__byte_perm(w, 0x4B400000u, 0x7610)), __uint_as_float(__byte_perm(w, 0x4B400000u, 0x7632)));
    return add2(f, dup(-12615680.0f));
}
MDWF_DEV c2 cvt_pair(unsigned w, c2 sc) { return mul2(cvt_raw(w), sc); }
template <> struct Ld<PH> {
    template <int NC, bool G = true> static MDWF_DEV void chunks(const short4 *p, float sc, c2 *v)
    {
        const c2 s2 = dup(sc);
#pragma unroll
        for (int j = 0; j < NC / 2; j++) {
            const uint2 q = ldx<G>(reinterpret_cast<const uint2 *>(p + 32 * j));
            v[2 * j] = cvt_pair(q.x, s2);
            v[2 * j + 1] = cvt_pair(q.y, s2);
        }
    }
    // the stored integers as floats, unscaled: the hop is linear, so the scale of the slice is applied once, in the
    // reconstruction FMAs (saves one FMUL2 per complex on every neighbour load without B-on-load)
    template <int NC, bool G = true> static MDWF_DEV void raw(const short4 *p, c2 *v)
    {
#pragma unroll
        for (int j = 0; j < NC / 2; j++) {
            const uint2 q = ldx<G>(reinterpret_cast<const uint2 *>(p + 32 * j));
            v[2 * j] = cvt_raw(q.x);
            v[2 * j + 1] = cvt_raw(q.y);
        }
    }
};

// ---- links ---------------------------------------------------------------------------------------------
// M = U (forward hop) or U^dagger (backward hop), entry (a,c) = re[a*3+c] + i im[a*3+c]: 18 scalar registers.
// FFMA2 takes a scalar register broadcast to both lanes and a swapped (LO_HI) pair as free operand forms, so
// chi_a = P + i Q with P = sum_c re (h_r,h_i), Q = sum_c im (h_r,h_i) needs no expanded copies of the link and no
// register moves: chi = fma2((-1,1), (Q_i,Q_r), P).
struct Link {
    float re[9], im[9];
};
MDWF_DEV void gget(const float2 q, float &re, float &im) { re = q.x; im = q.y; }
MDWF_DEV void gget(const short2 q, float &re, float &im)
{
    const unsigned w = ((unsigned)(unsigned short)q.y << 16) | (unsigned short)q.x;
    const c2 v = cvt_pair(w, dup(1.0f / MDWF_FIXED_MAX));
    re = v.x;
    im = v.y;
}
// The link tile of the block's 32 sites ([8 directions][NK][32] in the gauge layout, backward links already pulled back
// and daggered) is brought into shared memory by ONE bulk copy of the TMA engine (hop3_kernel).  expand_link finishes
// direction d of this lane in the link table sL (element k at sL[(d*9 + k)*32 + lane]):
//   fp32 storage : the copy lands in the table itself; with 12-real storage row 2 = conj(row0 x row1) is added in place;
//   16-bit       : the raw tile lands in sR, is converted (and completed) here.
MDWF_DEV void row2_from_rows01(float *ur, float *ui)
{
    // row2[c] = conj(row0[a] row1[b] - row0[b] row1[a]),  (a,b) = (c+1, c+2) mod 3
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const int a = (c + 1) % 3, b = (c + 2) % 3;
        float re = ur[a] * ur[3 + b];
        re = fmaf(-ui[a], ui[3 + b], re); re = fmaf(-ur[b], ur[3 + a], re); re = fmaf(ui[b], ui[3 + a], re);
        float im = ur[a] * ui[3 + b];
        im = fmaf(ui[a], ur[3 + b], im); im = fmaf(-ur[b], ui[3 + a], im); im = fmaf(-ui[b], ur[3 + a], im);
        ur[6 + c] = re;
        ui[6 + c] = -im;
    }
}
template <class P>
MDWF_DEV void expand_link(const void *sR, float2 *sL, int d, int lane, int recon)
{
    float ur[9], ui[9];
    float2 *row = sL + d * 288 + lane;
    if (!P::HALF) {
        if (recon == 18) return;
#pragma unroll
        for (int k = 0; k < 6; k++) gget(row[32 * k], ur[k], ui[k]);
        row2_from_rows01(ur, ui);
#pragma unroll
        for (int k = 6; k < 9; k++) row[32 * k] = make_float2(ur[k], ui[k]);
    } else {
        const int NK = recon >> 1;
        const short2 *raw = reinterpret_cast<const short2 *>(sR) + d * NK * 32 + lane;
#pragma unroll
        for (int k = 0; k < 6; k++) gget(raw[32 * k], ur[k], ui[k]);
        if (recon == 18) {
#pragma unroll
            for (int k = 6; k < 9; k++) gget(raw[32 * k], ur[k], ui[k]);
        } else {
            row2_from_rows01(ur, ui);
        }
#pragma unroll
        for (int k = 0; k < 9; k++) row[32 * k] = make_float2(ur[k], ui[k]);
    }
}
// p = this lane's column of the shared-memory link table of one direction
MDWF_DEV void load_link3(const float2 *p, Link &L)
{
#pragma unroll
    for (int k = 0; k < 9; k++) {
        const float2 q = p[32 * k];
        L.re[k] = q.x;
        L.im[k] = q.y;
    }
}

// chi[sp*3+a] = sum_c M[a][c] h[sp*3+c]: per output two chains of 3 packed operations and one combine
MDWF_DEV void su3_mul3(const Link &L, const c2 *h, c2 *chi)
{
    const c2 mp = mk(-1.f, 1.f);
#pragma unroll
    for (int sp = 0; sp < 2; sp++)
#pragma unroll
        for (int a = 0; a < 3; a++) {
            c2 P = mul2(dup(L.re[a * 3]), h[sp * 3]);
            c2 Q = mul2(dup(L.im[a * 3]), h[sp * 3]);
#pragma unroll
            for (int c = 1; c < 3; c++) {
                P = fma2(dup(L.re[a * 3 + c]), h[sp * 3 + c], P);
                Q = fma2(dup(L.im[a * 3 + c]), h[sp * 3 + c], Q);
            }
            chi[sp * 3 + a] = fma2(mp, mk(Q.y, Q.x), P);
        }
}

// ---- spin projection / reconstruction in the DeGrand-Rossi basis, complex-pair form ----------------
// v[spin*3+colour].  (1 - SGN gamma_mu) v has upper half h (returned) and a lower half that follows from h:
//   mu=0: h0 = v0 - S i v3, h1 = v1 - S i v2;  r2 =  S i h1, r3 =  S i h0
//   mu=1: h0 = v0 + S v3,   h1 = v1 - S v2;    r2 = -S h1,   r3 =  S h0
//   mu=2: h0 = v0 - S i v2, h1 = v1 + S i v3;  r2 =  S i h0, r3 = -S i h1
//   mu=3: h0 = v0 - S v2,   h1 = v1 - S v3;    r2 = -S h0,   r3 = -S h1
// -S i (a + i b) = S (b, -a) = swp(.) * (S, -S);   S i (a + i b) = swp(.) * (-S, S).
template <int MU, int SGN>
MDWF_DEV void project3(const c2 *v, c2 *h)
{
    const float S = (float)SGN;
    const c2 pm = mk(S, -S), mp = mk(-S, S), ss = mk(S, S), mm = mk(-S, -S);
#pragma unroll
    for (int c = 0; c < 3; c++) {
        if (MU == 0) {
            h[c] = fma2(swp(v[9 + c]), pm, v[c]);
            h[3 + c] = fma2(swp(v[6 + c]), pm, v[3 + c]);
        } else if (MU == 1) {
            h[c] = fma2(v[9 + c], ss, v[c]);
            h[3 + c] = fma2(v[6 + c], mm, v[3 + c]);
        } else if (MU == 2) {
            h[c] = fma2(swp(v[6 + c]), pm, v[c]);
            h[3 + c] = fma2(swp(v[9 + c]), mp, v[3 + c]);
        } else {
            h[c] = fma2(v[6 + c], mm, v[c]);
            h[3 + c] = fma2(v[9 + c], mm, v[3 + c]);
        }
    }
}
// ---- spin projection straight from the stored 16-bit words ------------------------------------------------------------
// 0x4B400000 | u is the float M + q (M = 12615680, q the stored integer; cvt_raw above).  The projected half spinor
// h = v_a +- v_b (or +- i v_b) is needed as the integers q_a +- q_b, so the magic constant need not be subtracted from each input
// first: a "-" lane is (M + q_a) - (M + q_b), a "+" lane is (M + q_a) + ((M + q_b) - 2M); every intermediate is an integer below
// 2^24, so all of it is exact and the result is bit-identical to converting first.  Per projected complex: one FFMA2, plus one
// FADD2 when it has a "+" lane, instead of two FADD2 and the FFMA2: 84 instead of 144 FMA-pipe instructions per 8 directions.
MDWF_DEV c2 magic_pair(unsigned w)
{
    return mk(__uint_as_float(__byte_perm(w, 0x4B400000u, 0x7610)), __uint_as_float(__byte_perm(w, 0x4B400000u, 0x7632)));
}
// (q_a.x + SX q_b[SWAP ? y : x], q_a.y + SY q_b[SWAP ? x : y]) from the magic floats of a and b
template <int SX, int SY, bool SWAP>
MDWF_DEV c2 comb(c2 fa, c2 fb)
{
    constexpr float M2 = -2.0f * 12615680.0f;
    constexpr float kx = SWAP ? (SY > 0 ? M2 : 0.f) : (SX > 0 ? M2 : 0.f), ky = SWAP ? (SX > 0 ? M2 : 0.f) : (SY > 0 ? M2 : 0.f);
    const c2 t = (SX > 0 || SY > 0) ? add2(fb, mk(kx, ky)) : fb;
    return fma2(SWAP ? swp(t) : t, mk((float)SX, (float)SY), fa);
}
// project3 on the magic floats f[spin*3+colour] of a stored spinor: h = the projected integers (same table as project3)
template <int MU, int SGN>
MDWF_DEV void project3m(const c2 *f, c2 *h)
{
    constexpr int S = SGN;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        if (MU == 0) {
            h[c] = comb<S, -S, true>(f[c], f[9 + c]);
            h[3 + c] = comb<S, -S, true>(f[3 + c], f[6 + c]);
        } else if (MU == 1) {
            h[c] = comb<S, S, false>(f[c], f[9 + c]);
            h[3 + c] = comb<-S, -S, false>(f[3 + c], f[6 + c]);
        } else if (MU == 2) {
            h[c] = comb<S, -S, true>(f[c], f[6 + c]);
            h[3 + c] = comb<-S, S, true>(f[3 + c], f[9 + c]);
        } else {
            h[c] = comb<-S, -S, false>(f[c], f[6 + c]);
            h[3 + c] = comb<-S, -S, false>(f[3 + c], f[9 + c]);
        }
    }
}
// acc += sc * [chi ; lower(chi)],  sc = +-1 (antiperiodic t hop), acc[spin*3+colour]
template <int MU, int SGN, bool WITHSC>
MDWF_DEV void recon3(const c2 *chi, float sc, c2 *acc)
{
    const float p = WITHSC ? sc : 1.0f, S = (float)SGN * p;
    const c2 pp = mk(p, p), mp = mk(-S, S), pm = mk(S, -S), ss = mk(S, S), mm = mk(-S, -S);
#pragma unroll
    for (int c = 0; c < 3; c++) {
        if (WITHSC) {
            acc[c] = fma2(chi[c], pp, acc[c]);
            acc[3 + c] = fma2(chi[3 + c], pp, acc[3 + c]);
        } else {
            acc[c] = add2(acc[c], chi[c]);
            acc[3 + c] = add2(acc[3 + c], chi[3 + c]);
        }
        if (MU == 0) {
            acc[6 + c] = fma2(swp(chi[3 + c]), mp, acc[6 + c]);
            acc[9 + c] = fma2(swp(chi[c]), mp, acc[9 + c]);
        } else if (MU == 1) {
            acc[6 + c] = fma2(chi[3 + c], mm, acc[6 + c]);
            acc[9 + c] = fma2(chi[c], ss, acc[9 + c]);
        } else if (MU == 2) {
            acc[6 + c] = fma2(swp(chi[c]), mp, acc[6 + c]);
            acc[9 + c] = fma2(swp(chi[3 + c]), pm, acc[9 + c]);
        } else {
            acc[6 + c] = fma2(chi[c], mm, acc[6 + c]);
            acc[9 + c] = fma2(chi[3 + c], mm, acc[9 + c]);
        }
    }
}

// ---- one direction of the stencil for the S slices of this thread ----------------------------------
// FWD: neighbour x+mu through U_mu(x); else neighbour x-mu through U_mu(x-mu)^dagger.
// PRE = 1 applies (1 + f Lambda) to the neighbour on load: upper spins add f * (slice s-1), lower spins
// f * (slice s+1), wall factor -m_f at the wrap.  The window slides over the S slices (one half-spinor of
// halo on each side), so only one full slice and two half slices are live at a time.
// The neighbour's slices are read through a source object: SrcMem = global memory (G = true, read-only path) or a group
// staged in shared memory (G = false), which keeps the [s][chunk][lane] layout; SrcReg = raw chunks loaded into
// registers ahead of their use (the first direction of a block, whose loads are issued before the link tile is waited
// for).  Window slice k = 0..S-1 is slice s0 + k; k = -1 / k = S are the halo slices of the B-on-load stencil.
template <class P, bool G> MDWF_DEV float ld_scale(const float *np)
{
    if (!P::HALF) return 1.0f;
    return ldx<G>(np) * (1.0f / MDWF_FIXED_MAX);
}
template <class P, int S, bool G> struct SrcMem {
    const typename P::V *gb;      // chunk 0 of slice 0 of this thread's neighbour site
    const float *nb;              // scale of slice 0 (16-bit storage)
    int s0, sm, sp;               // first slice of the window, slice below (wrapped), slice above (wrapped)
    MDWF_DEV int slice(int k) const { return k < 0 ? sm : (k >= S ? sp : s0 + k); }
    MDWF_DEV typename P::V chunk(int k, int j) const { return ldx<G>(gb + slice(k) * (32 * P::NV) + 32 * j); }
    MDWF_DEV float scale(int k) const { return ld_scale<P, G>(nb + 32 * slice(k)); }
};
template <class P, int PRE, int S> struct SrcReg {
    typename P::V q[S][6], up[3], lo[3];
    float sc[S], scu, scl;
    template <bool G> MDWF_DEV void load(const SrcMem<P, S, G> &m)
    {
#pragma unroll
        for (int k = 0; k < S; k++) {
#pragma unroll
            for (int j = 0; j < 6; j++) q[k][j] = m.chunk(k, j);
            sc[k] = m.scale(k);
        }
        if (PRE) {
#pragma unroll
            for (int j = 0; j < 3; j++) { up[j] = m.chunk(-1, j); lo[j] = m.chunk(S, 3 + j); }
            scu = m.scale(-1);
            scl = m.scale(S);
        }
    }
    MDWF_DEV typename P::V chunk(int k, int j) const { return k < 0 ? up[j] : (k >= S ? lo[j - 3] : q[k][j]); }
    MDWF_DEV float scale(int k) const { return k < 0 ? scu : (k >= S ? scl : sc[k]); }
};
// chunk -> two complex numbers; SCALED = false leaves the 16-bit integers unscaled (the scale then goes into the
// reconstruction weight: the hop is linear)
template <bool SCALED> MDWF_DEV void unp(const float4 q, float, c2 &x, c2 &y) { x = mk(q.x, q.y); y = mk(q.z, q.w); }
template <bool SCALED> MDWF_DEV void unp(const short4 q, float sc, c2 &x, c2 &y)
{
    const uint2 w = *reinterpret_cast<const uint2 *>(&q);       // the two 32-bit words as loaded: no repacking
    const unsigned w0 = w.x, w1 = w.y;
    if (SCALED) { x = cvt_pair(w0, dup(sc)); y = cvt_pair(w1, dup(sc)); }
    else { x = cvt_raw(w0); y = cvt_raw(w1); }
}
// complexes [2*J0, 2*J0 + 2*NJ) of window slice k into v[0 .. 2*NJ)
template <bool SCALED, int J0, int NJ, class SRC> MDWF_DEV void take(const SRC &src, int k, float sc, c2 *v)
{
#pragma unroll
    for (int j = 0; j < NJ; j++) unp<SCALED>(src.chunk(k, J0 + j), sc, v[2 * j], v[2 * j + 1]);
}

template <class P, int MU, bool FWD, int DAG, int PRE, int S, bool TDIR, class SRC>
MDWF_DEV void hop_dir3(const HopArgs &a, int L5, int s0, const float2 *sl, const SRC &src, float bsign, c2 (*acc)[12])
{
    constexpr int SGN = (FWD ? 1 : -1) * (DAG ? -1 : 1);
    Link U;
    load_link3(sl, U);

    if (PRE == 0) {
#pragma unroll
        for (int k = 0; k < S; k++) {
            c2 v[12], h[6], chi[6];
            if constexpr (P::HALF) {
                const float sck = src.scale(k);
#pragma unroll
                for (int j = 0; j < 6; j++) {
                    const typename P::V q = src.chunk(k, j);
                    const uint2 w = *reinterpret_cast<const uint2 *>(&q);
                    v[2 * j] = magic_pair(w.x);
                    v[2 * j + 1] = magic_pair(w.y);
                }
                project3m<MU, SGN>(v, h);
                su3_mul3(U, h, chi);
                recon3<MU, SGN, true>(chi, TDIR ? bsign * sck : sck, acc[k]);
            } else {
                take<true, 0, 6>(src, k, 1.f, v);
                project3<MU, SGN>(v, h);
                su3_mul3(U, h, chi);
                recon3<MU, SGN, TDIR>(chi, bsign, acc[k]);
            }
        }
    } else {
        const float f = (float)(a.pre_o / a.pre_d), fw = (float)(-a.mf * a.pre_o / a.pre_d);
        c2 prev_up[6], cur[12], nxt[12];
        take<true, 0, 3>(src, -1, src.scale(-1), prev_up);
        take<true, 0, 6>(src, 0, src.scale(0), cur);
#pragma unroll
        for (int k = 0; k < S; k++) {
            if (k < S - 1) take<true, 0, 6>(src, k + 1, src.scale(k + 1), nxt);
            else take<true, 3, 3>(src, S, src.scale(S), nxt + 6);
            const c2 fu = dup((s0 + k == 0) ? fw : f);
            const c2 fl = dup((s0 + k == L5 - 1) ? fw : f);
            c2 w[12], h[6], chi[6];
#pragma unroll
            for (int q = 0; q < 6; q++) {
                w[q] = fma2(fu, prev_up[q], cur[q]);
                w[6 + q] = fma2(fl, nxt[6 + q], cur[6 + q]);
            }
            project3<MU, SGN>(w, h);
            su3_mul3(U, h, chi);
            recon3<MU, SGN, TDIR>(chi, bsign, acc[k]);
#pragma unroll
            for (int q = 0; q < 6; q++) prev_up[q] = cur[q];
            if (k < S - 1) {
#pragma unroll
                for (int q = 0; q < 12; q++) cur[q] = nxt[q];
            }
        }
    }
}

// ---- spinor store from complex pairs ---------------------------------------------------------------
// returns the sum of squares of the values as stored (for the fused norm of the output vector)
// stores one (site, slice); returns its contribution to the fused norm (of the values as stored) when want_norm is set
template <class P> MDWF_DEV float store3(void *base, float *norm, int L5, int s, long cb, const c2 *o, bool want_norm = true);
template <> MDWF_DEV float store3<PS>(void *base, float *, int L5, int s, long cb, const c2 *o, bool)
{
    float4 *p = reinterpret_cast<float4 *>(base) + sp_off(L5, PS::NV, cb, s);
#pragma unroll
    for (int j = 0; j < 6; j++) p[32 * j] = make_float4(o[2 * j].x, o[2 * j].y, o[2 * j + 1].x, o[2 * j + 1].y);
    c2 n2 = mul2(o[0], o[0]);
#pragma unroll
    for (int q = 1; q < 12; q++) n2 = fma2(o[q], o[q], n2);
    return n2.x + n2.y;
}
template <> MDWF_DEV float store3<PH>(void *base, float *norm, int L5, int s, long cb, const c2 *o, bool want_norm)
{
    short4 *p = reinterpret_cast<short4 *>(base) + sp_off(L5, PH::NV, cb, s);
    float m = 0.f;
#pragma unroll
    for (int q = 0; q < 12; q++) m = fmaxf(m, fmaxf(fabsf(o[q].x), fabsf(o[q].y)));
    norm[sp_noff(L5, cb, s)] = m;
    // fp32 -> 16-bit offset binary by the magic-number add: the low 16 bits of fma(v, isc, 1.5 * 2^23 + 2^15) are round(v isc) + 2^15
    const c2 isc = dup(m > 0.f ? MDWF_FIXED_MAX / m : 0.f), magic = dup(12615680.0f);
    uint2 *pw = reinterpret_cast<uint2 *>(p);
    const c2 nmagic = dup(-12615680.0f);
    c2 n2 = mk(0.f, 0.f);
#pragma unroll
    for (int j = 0; j < 6; j++) {
        const c2 e = fma2(o[2 * j], isc, magic), f = fma2(o[2 * j + 1], isc, magic);
        pw[32 * j] = make_uint2(__byte_perm(__float_as_uint(e.x), __float_as_uint(e.y), 0x5410),
                                __byte_perm(__float_as_uint(f.x), __float_as_uint(f.y), 0x5410));
        if (want_norm) {                                          // uniform over the kernel: K1 / K1^dagger have no fused norm
            const c2 qe = add2(e, nmagic), qf = add2(f, nmagic);  // the stored integers, exactly
            n2 = fma2(qe, qe, n2);
            n2 = fma2(qf, qf, n2);
        }
    }
    const float sc = m * (1.0f / MDWF_FIXED_MAX);
    return (n2.x + n2.y) * sc * sc;
}

// ---- fifth-dimension epilogues on the S slices of a thread -----------------------------------------
// Orientation: "direct" (MIRROR = false) is the P+ pattern of A = alpha + beta Lambda (slice s couples to s-1);
// MIRROR = true is the P- pattern (s couples to s+1), i.e. the same recurrence with s -> L5-1-s.
// Effective index of a thread's slice k:  j = MIRROR ? S-1-k : k,  of its warp: g = MIRROR ? NSG-1-sg : sg.

// local recurrence z_j = x_j - kappa z_{j-1} (z_{-1} = 0) in place on components [off, off+6)
template <int S, bool MIRROR>
MDWF_DEV void rec_local(c2 (*x)[12], int off, c2 nk)
{
#pragma unroll
    for (int j = 1; j < S; j++) {
        const int k = MIRROR ? S - 1 - j : j, kp = MIRROR ? k + 1 : k - 1;
#pragma unroll
        for (int q = 0; q < 6; q++) x[k][off + q] = fma2(nk, x[kp][off + q], x[k][off + q]);
    }
}
// t_j = bz z_j + cz z_{j-1} + qC_j C + qW_s W  in place (j descending so that z_{j-1} is still the local value)
template <int S, int NSG, bool MIRROR>
MDWF_DEV void rec_finish(c2 (*x)[12], int off, int sg, const c2 *sE, int lane, const HopArgs &a)
{
    const int g = MIRROR ? NSG - 1 - sg : sg;
    const c2 cS = dup(a.r_cpow);
    c2 C[6], W[6];
#pragma unroll
    for (int q = 0; q < 6; q++) { C[q] = mk(0.f, 0.f); W[q] = mk(0.f, 0.f); }
#pragma unroll
    for (int j = 0; j < NSG; j++) {          // Horner over the carries of the warps in effective order
        const int jj = MIRROR ? NSG - 1 - j : j;
        if (j == g) {
#pragma unroll
            for (int q = 0; q < 6; q++) C[q] = W[q];
        }
#pragma unroll
        for (int q = 0; q < 6; q++) W[q] = fma2(cS, W[q], sE[(jj * 12 + off + q) * 32 + lane]);
    }
    const c2 bz = dup(a.r_bz), cz = dup(a.r_cz);
#pragma unroll
    for (int j = S - 1; j >= 0; j--) {
        const int k = MIRROR ? S - 1 - j : j, kp = MIRROR ? k + 1 : k - 1;
        const c2 qC = dup(a.r_qC[j]), qW = dup(a.r_qW[g * S + j]);
#pragma unroll
        for (int q = 0; q < 6; q++) {
            c2 t = mul2(bz, x[k][off + q]);
            if (j > 0) t = fma2(cz, x[kp][off + q], t);
            t = fma2(qC, C[q], t);
            x[k][off + q] = fma2(qW, W[q], t);
        }
    }
}

template <class P, int S> struct Hop3Cfg {
    // 8 warps per SM (two blocks of 128 threads or one of 256): up to 255 registers per thread
    // resident warps per SM asked of ptxas: 8 (255 registers) for fp32 storage, whose 16-byte loads in flight need
    // the registers; 12 (168 registers) for 16-bit storage
    static constexpr int WARPS = P::HALF ? MDWF_H3_WARPS_H : MDWF_H3_WARPS;
};

// ---- epilogue shared by the v3 and v5 kernels: fifth-dimension POST step, own-site term, store, fused norm ----
template <class P, int DAG, int POST, int OWN, int L5, int S>
MDWF_DEV void epilogue3(const HopArgs &a, c2 (*acc)[12], c2 *sE, int lane, int sg, int s0, long cb, bool active, int pidx)
{
    constexpr int NSG = L5 / S;
    using V = typename P::V;
    if (POST == 1) {
        // coef_hop * (B A^{-1}) acc per chirality (DAG: the transposed pattern) by blocked recurrence
        const c2 nk = dup(a.r_nk);
        rec_local<S, DAG != 0>(acc, 0, nk);              // upper spins: direct pattern (mirrored for the dagger)
        rec_local<S, DAG == 0>(acc, 6, nk);              // lower spins: mirrored pattern (direct for the dagger)
        constexpr int kU = DAG ? 0 : S - 1, kL = DAG ? S - 1 : 0;    // slice holding the carry-out
#pragma unroll
        for (int q = 0; q < 6; q++) {
            sE[(sg * 12 + q) * 32 + lane] = acc[kU][q];
            sE[(sg * 12 + 6 + q) * 32 + lane] = acc[kL][6 + q];
        }
        __syncthreads();
        rec_finish<S, NSG, DAG != 0>(acc, 0, sg, sE, lane, a);
        rec_finish<S, NSG, DAG == 0>(acc, 6, sg, sE, lane, a);
    } else if (POST == 2) {
        // coef_hop * (post_d + post_o Lambda^dagger) acc: upper spins take s+1, lower spins s-1, -m_f at the wrap
#pragma unroll
        for (int q = 0; q < 6; q++) {
            sE[(sg * 12 + q) * 32 + lane] = acc[0][q];               // first slice, upper: halo of warp sg-1
            sE[(sg * 12 + 6 + q) * 32 + lane] = acc[S - 1][6 + q];   // last slice, lower: halo of warp sg+1
        }
        __syncthreads();
        const int gu = (sg == NSG - 1) ? 0 : sg + 1, gl = (sg == 0) ? NSG - 1 : sg - 1;
        const float coef = (float)a.coef_hop, o = coef * (float)a.post_o, ow = -o * (float)a.mf;
        const c2 d2 = dup(coef * (float)a.post_d), o2 = dup(o);
        const c2 ou = dup(sg == NSG - 1 ? ow : o), ol = dup(sg == 0 ? ow : o);
#pragma unroll
        for (int k = 0; k < S; k++)
#pragma unroll
            for (int q = 0; q < 6; q++) {
                const c2 nb = (k < S - 1) ? acc[k + 1][q] : sE[(gu * 12 + q) * 32 + lane];
                acc[k][q] = fma2(d2, acc[k][q], mul2((k < S - 1) ? o2 : ou, nb));
            }
#pragma unroll
        for (int k = S - 1; k >= 0; k--)
#pragma unroll
            for (int q = 0; q < 6; q++) {
                const c2 nb = (k > 0) ? acc[k - 1][6 + q] : sE[(gl * 12 + 6 + q) * 32 + lane];
                acc[k][6 + q] = fma2(d2, acc[k][6 + q], mul2((k > 0) ? o2 : ol, nb));
            }
    }
    float nsum = 0.f;
    if (active) {
    const c2 coef2 = dup(POST == 0 ? (float)a.coef_hop : 1.0f);     // POST != 0: coef_hop is already folded in
#pragma unroll
    for (int k = 0; k < S; k++) {
        const int s = s0 + k;
        c2 o[12];
        if (OWN == 0) {
#pragma unroll
            for (int q = 0; q < 12; q++) o[q] = (POST == 0) ? mul2(coef2, acc[k][q]) : acc[k][q];
        } else if (OWN == 1) {
            c2 w[12];
            const V *p = reinterpret_cast<const V *>(a.own) + sp_off(L5, P::NV, cb, s);
            Ld<P>::template chunks<12>(p, load_scale<P>(a.own_norm, sp_noff(L5, cb, s)), w);
#pragma unroll
            for (int q = 0; q < 12; q++) o[q] = fma2(coef2, acc[k][q], w[q]);
        } else {
            // (own_d + own_o Lambda) psi: upper from s-1, lower from s+1; Lambda^dagger (OWN == 3): swapped.
            // 16-bit storage: the stored integers are used as they are and the scale of each slice goes into its coefficient
            c2 w[12], u[6], l[6];
            const V *p = reinterpret_cast<const V *>(a.own) + sp_off(L5, P::NV, cb, s);
            int su = (OWN == 2) ? s - 1 : s + 1;
            int sl = (OWN == 2) ? s + 1 : s - 1;
            float fu = (float)a.own_o, fl = (float)a.own_o, fd = (float)a.own_d;
            if (su < 0) { su = L5 - 1; fu *= (float)(-a.mf); }
            if (su >= L5) { su = 0; fu *= (float)(-a.mf); }
            if (sl < 0) { sl = L5 - 1; fl *= (float)(-a.mf); }
            if (sl >= L5) { sl = 0; fl *= (float)(-a.mf); }
            const V *pu = reinterpret_cast<const V *>(a.own) + sp_off(L5, P::NV, cb, su);
            const V *pl = reinterpret_cast<const V *>(a.own) + sp_off(L5, P::NV, cb, sl) + 32 * (P::NV / 2);
            if constexpr (P::HALF) {
                Ld<P>::template raw<12>(p, w);
                Ld<P>::template raw<6>(pu, u);
                Ld<P>::template raw<6>(pl, l);
                fd *= load_scale<P>(a.own_norm, sp_noff(L5, cb, s));
                fu *= load_scale<P>(a.own_norm, sp_noff(L5, cb, su));
                fl *= load_scale<P>(a.own_norm, sp_noff(L5, cb, sl));
            } else {
                Ld<P>::template chunks<12>(p, 1.f, w);
                Ld<P>::template chunks<6>(pu, 1.f, u);
                Ld<P>::template chunks<6>(pl, 1.f, l);
            }
            const c2 d2 = dup(fd), fu2 = dup(fu), fl2 = dup(fl);
#pragma unroll
            for (int q = 0; q < 6; q++) {
                o[q] = fma2(coef2, acc[k][q], fma2(d2, w[q], mul2(fu2, u[q])));
                o[6 + q] = fma2(coef2, acc[k][6 + q], fma2(d2, w[6 + q], mul2(fl2, l[q])));
            }
        }
        nsum += store3<P>(a.out, a.out_norm, L5, s, cb, o, a.partial != nullptr);
    }
    }
    if (a.partial) {
        // fused ||out||^2 (S7): fp32 per thread, then a fixed shuffle tree and a fixed order over the warps in fp64;
        // one partial per block, summed in fixed order by final_sum_kernel -> bit-reproducible
        __shared__ double wsum[NSG];
        double v = (double)nsum;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) wsum[sg] = v;
        __syncthreads();
        if (lane == 0 && sg == 0) {
            double t = 0.0;
#pragma unroll
            for (int j = 0; j < NSG; j++) t += wsum[j];
            a.partial[pidx] = t;                     // pidx = index of the 32-site group in the sweep order
        }
    }
}

// ---- bulk-asynchronous copies (TMA engine) and their barriers ------------------------------------------------
MDWF_DEV unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
MDWF_DEV void mbar_init(unsigned long long *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%1], %0;" ::"r"(count), "r"(smem_u32(bar)) : "memory");
}
MDWF_DEV void mbar_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%1], %0;" ::"r"(bytes), "r"(smem_u32(bar)) : "memory");
}
MDWF_DEV void mbar_wait(unsigned long long *bar, unsigned phase)
{
    unsigned ok = 0;
    const unsigned addr = smem_u32(bar);
    while (!ok) {
        asm volatile("{\n\t.reg .pred P1;\n\tmbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2, %3;\n\tselp.u32 %0, 1, 0, P1;\n\t}"
                     : "=r"(ok)
                     : "r"(addr), "r"(phase), "r"(0x989680u)          // suspend-time hint: sleep in hardware rather than poll
                     : "memory");
    }
}
MDWF_DEV void bulk_g2s(void *dst_smem, const void *src_gmem, unsigned bytes, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

MDWF_DEV void bulk_prefetch_l2(const void *src_gmem, unsigned bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src_gmem), "r"(bytes) : "memory");
}
MDWF_DEV unsigned fdiv(unsigned n, const FastDiv &f) { return f.m ? (__umulhi(n, f.m) >> f.s) : n; }

template <class P, int DAG, int PRE, int POST, int OWN, int L5, int S>
__global__ void __launch_bounds__(32 * (L5 / S), Hop3Cfg<P, S>::WARPS / (L5 / S) > 0 ? Hop3Cfg<P, S>::WARPS / (L5 / S) : 1) hop3_kernel(const HopArgs a)
{
    constexpr int NSG = L5 / S, NV = P::NV;
    using V = typename P::V;
    constexpr unsigned BUF_BYTES = L5 * NV * 32 * sizeof(V);          // all slices of one 32-site group
    constexpr unsigned NRM_BYTES = P::HALF ? L5 * 32 * sizeof(float) : 0;
    constexpr unsigned SE_BYTES = (POST != 0) ? NSG * 12 * 32 * sizeof(c2) : 0;
    using G = typename P::G;
    constexpr unsigned SL_BYTES = 8 * 9 * 32 * sizeof(float2);
    constexpr unsigned SR_BYTES = P::HALF ? 8 * 9 * 32 * sizeof(short2) : 0;
    extern __shared__ __align__(128) unsigned char smem_raw3[];
    unsigned char *rest = smem_raw3;
    c2 *sE = reinterpret_cast<c2 *>(rest);                             // [NSG][12][32] carries / halo slices (POST != 0)
    float2 *sL = reinterpret_cast<float2 *>(rest + SE_BYTES);          // [8][9][32] link table
    unsigned char *sR = rest + SE_BYTES + SL_BYTES;                    // 16-bit storage: the raw link tile
    unsigned long long *bar = reinterpret_cast<unsigned long long *>(sR + SR_BYTES);   // completion of the link tile's bulk copy
    const int lane = threadIdx.x, sg = threadIdx.y, s0 = sg * S;
    const int Lxh = a.L[0] >> 1, Ly = a.L[1], Lz = a.L[2], Lt = a.L[3];
    const long sy = Lxh, sz = (long)Lxh * Ly, st = (long)Lxh * Ly * Lz;
    long cb0 = (long)blockIdx.x * 32;
    if (a.sweep_nb) {                                    // z-chunked t sweep, see hop_kernels.cuh
        const unsigned c = fdiv(blockIdx.x, a.dchunk), r = blockIdx.x - c * (unsigned)(a.sweep_nb * Lt);
        const unsigned t = fdiv(r, a.dnb), q = r - t * (unsigned)a.sweep_nb;
        cb0 = (long)t * st + (long)c * a.sweep_chunk + (long)q * 32;
    }
    const long cb = cb0 + lane;
    const bool active = cb < a.Vh;

    // ---- one elected thread starts the bulk copy of the link tile of the block's 32 sites (and pulls the own-site slab into L2) ----
    if (lane == 0 && sg == 0) {
        mbar_init(&bar[0], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        const int NK = a.recon >> 1;
        const G *tile = reinterpret_cast<const G *>(a.gauge) + (cb0 >> 5) * (long)(8 * NK * 32);
        mbar_expect_tx(&bar[0], 8 * NK * 32 * sizeof(G));
        if (P::HALF || NK == 9) {
            bulk_g2s(P::HALF ? (void *)sR : (void *)sL, tile, 8 * NK * 32 * sizeof(G), &bar[0]);
        } else {
#pragma unroll
            for (int d = 0; d < 8; d++) bulk_g2s(sL + d * 288, tile + d * 6 * 32, 6 * 32 * sizeof(G), &bar[0]);   // rows 0,1 of each direction
        }
        if (OWN != 0) {     // the own-site slab the epilogue reads: pull it into L2 now
            bulk_prefetch_l2(reinterpret_cast<const V *>(a.own) + (cb0 >> 5) * (long)(L5 * NV * 32), BUF_BYTES);
            if (P::HALF) bulk_prefetch_l2(a.own_norm + (cb0 >> 5) * (long)(L5 * 32), NRM_BYTES);
        }
    }

    c2 acc[S][12];
#pragma unroll
    for (int k = 0; k < S; k++)
#pragma unroll
        for (int q = 0; q < 12; q++) acc[k][q] = mk(0.f, 0.f);

    // neighbour indices (inactive lanes of a ragged last block keep cb = 0 and load nothing)
    const long cbs = active ? cb : 0;
    const unsigned q1 = fdiv((unsigned)cbs, a.dLxh), q2 = fdiv(q1, a.dLy), q3 = fdiv(q2, a.dLz);
    const int xh = (int)((unsigned)cbs - q1 * Lxh), y = (int)(q1 - q2 * Ly), z = (int)(q2 - q3 * Lz), t = (int)q3;
    const int xodd = (a.parity_out + y + z + t) & 1;
    long nb[8];                                                  // link-tile order: 0-3 forward mu, 4-7 backward mu
    nb[0] = xodd ? (xh == Lxh - 1 ? cbs - (Lxh - 1) : cbs + 1) : cbs;
    nb[4] = xodd ? cbs : (xh == 0 ? cbs + (Lxh - 1) : cbs - 1);
    nb[1] = (y == Ly - 1) ? cbs - (Ly - 1) * sy : cbs + sy;
    nb[5] = (y == 0) ? cbs + (Ly - 1) * sy : cbs - sy;
    nb[2] = (z == Lz - 1) ? cbs - (Lz - 1) * sz : cbs + sz;
    nb[6] = (z == 0) ? cbs + (Lz - 1) * sz : cbs - sz;
    nb[3] = (t == Lt - 1) ? cbs - (Lt - 1) * st : cbs + st;
    nb[7] = (t == 0) ? cbs + (Lt - 1) * st : cbs - st;
    const float btp = (t == Lt - 1) ? -1.f : 1.f;               // antiperiodic in t
    const float btm = (t == 0) ? -1.f : 1.f;

    // the loads of the first direction (x+) go out before the link tile is waited for
    const V *gin = reinterpret_cast<const V *>(a.in);
    const int sm = (s0 == 0) ? L5 - 1 : s0 - 1, sp = (s0 + S >= L5) ? 0 : s0 + S;
    // (fp32 storage only: at the 168 registers of the 16-bit kernels the early loads spill and cost more than they hide)
    constexpr bool EARLY = !P::HALF;
    SrcReg<P, PRE, EARLY ? S : 1> first;
    if (EARLY && active) first.load(SrcMem<P, EARLY ? S : 1, true>{gin + sp_off(L5, NV, nb[0], 0), a.in_norm + sp_noff(L5, nb[0], 0), s0, sm, sp});

    // the link tile has landed (its latency ran under the index arithmetic above): warp d mod NSG completes direction d
    __syncthreads();                                             // barrier initialisation visible to every thread
    mbar_wait(&bar[0], 0);
#pragma unroll
    for (int d = 0; d < 8; d++)
        if ((d % NSG) == sg) expand_link<P>(sR, sL, d, lane, a.recon);
    __syncthreads();

    if (active) {
        // neighbour in global memory: chunk 0 of slice 0 / scale of slice 0 of site nb[d];  d = FWD ? MU : 4 + MU
#define MDWF_GDIR(MU, FWD, TD, d, bs) \
        hop_dir3<P, MU, FWD, DAG, PRE, S, TD>(a, L5, s0, sL + (d) * 288 + lane, \
            SrcMem<P, S, true>{gin + sp_off(L5, NV, nb[d], 0), a.in_norm + sp_noff(L5, nb[d], 0), s0, sm, sp}, bs, acc)
        if constexpr (EARLY) hop_dir3<P, 0, true, DAG, PRE, S, false>(a, L5, s0, sL + 0 * 288 + lane, first, 1.f, acc);
        else MDWF_GDIR(0, true, false, 0, 1.f);
        MDWF_GDIR(0, false, false, 4, 1.f);
        MDWF_GDIR(1, true, false, 1, 1.f);
        MDWF_GDIR(1, false, false, 5, 1.f);
        MDWF_GDIR(2, true, false, 2, 1.f);
        MDWF_GDIR(2, false, false, 6, 1.f);
        MDWF_GDIR(3, true, true, 3, btp);
        MDWF_GDIR(3, false, true, 7, btm);
#undef MDWF_GDIR
    }

    epilogue3<P, DAG, POST, OWN, L5, S>(a, acc, sE, lane, sg, s0, cb, active, (int)blockIdx.x);
}

// ---- launchers ----------------------------------------------------------------------------------
template <class P, int DAG, int PRE, int POST, int OWN, int L5, int S>
static int launch_hop3_nst(const HopArgs &a, cudaStream_t st)
{
    constexpr int NSG = L5 / S;
    dim3 block(32, NSG);
    dim3 grid((unsigned)((a.Vh + 31) / 32));
    const size_t smem = ((POST != 0) ? (size_t)NSG * 12 * 32 * sizeof(c2) : 0) + (size_t)8 * 9 * 32 * sizeof(float2) +
                        (P::HALF ? (size_t)8 * 9 * 32 * sizeof(short2) : 0) + 8;
    static bool attr_set = false;                                // once per instantiation, not once per launch
    if (smem > 32 * 1024 && !attr_set) {     // dynamic + the kernel's static shared memory must stay under the 48 KB default
        cudaError_t e = cudaFuncSetAttribute(hop3_kernel<P, DAG, PRE, POST, OWN, L5, S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return (int)e;
        attr_set = true;
    }
    hop3_kernel<P, DAG, PRE, POST, OWN, L5, S><<<grid, block, smem, st>>>(a);
    return (int)cudaGetLastError();
}
template <class P, int DAG, int PRE, int POST, int OWN>
static int launch_hop3_l5(const HopArgs &a, cudaStream_t st)
{
    if (a.L5 == 12) return launch_hop3_nst<P, DAG, PRE, POST, OWN, 12, MDWF_H3_S12>(a, st);
#ifndef MDWF_DEV_FAST
    if (a.L5 == 8) return launch_hop3_nst<P, DAG, PRE, POST, OWN, 8, 2>(a, st);
    if (a.L5 == 16) return launch_hop3_nst<P, DAG, PRE, POST, OWN, 16, 2>(a, st);
#endif
    return (int)cudaErrorInvalidValue;
}
// true when the v3 family covers this launch (fp32 arithmetic, tabulated L5, |kappa| < 1 for the recurrence)
static inline bool hop3_supports(int L5, int post, const HopArgs &a)
{
    if (!(L5 == 8 || L5 == 12 || L5 == 16)) return false;
    if (post == 1 && !(a.r_ok)) return false;
    return true;
}
template <class P>
static int launch_hop3_prec(int dag, int pre, int post, int own, const HopArgs &a, cudaStream_t st)
{
    if (!dag && pre == 1 && post == 1 && own == 0) return launch_hop3_l5<P, 0, 1, 1, 0>(a, st);   // K1
    if (!dag && pre == 0 && post == 1 && own == 0) return launch_hop3_l5<P, 0, 0, 1, 0>(a, st);   // K1 reading a precomputed B psi
    if (!dag && pre == 0 && post == 0 && own == 2) return launch_hop3_l5<P, 0, 0, 0, 2>(a, st);   // K2
    if (!dag && pre == 1 && post == 0 && own == 2) return launch_hop3_l5<P, 0, 1, 0, 2>(a, st);   // D
    if (!dag && pre == 1 && post == 0 && own == 1) return launch_hop3_l5<P, 0, 1, 0, 1>(a, st);   // Schur prep/recon
    if (dag && pre == 0 && post == 1 && own == 0) return launch_hop3_l5<P, 1, 0, 1, 0>(a, st);    // K1^+
    if (dag && pre == 0 && post == 2 && own == 3) return launch_hop3_l5<P, 1, 0, 2, 3>(a, st);    // K2^+, D^+
    if (!dag && pre == 0 && post == 1 && own == 1) return launch_hop3_l5<P, 0, 0, 1, 1>(a, st);   // K2 of Mpc_sym: psi + coef A^{-1} H t
    if (dag && pre == 0 && post == 2 && own == 1) return launch_hop3_l5<P, 1, 0, 2, 1>(a, st);    // K2^+ of Mpc_sym^+: psi + coef B^+ H' u
    return (int)cudaErrorInvalidValue;
}

}   // namespace h3
