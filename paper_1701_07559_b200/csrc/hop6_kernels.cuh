// hop6_kernels.cuh -- the tile sweep of hop5_kernels.cuh for 16-bit storage (fp32 arithmetic), with two or three sweep sets.
// Same tile (2(z) x 2(t) 32-site groups), same ring / TMEM / epilogue structure; what differs:
//
//   * a ring item holds the 16 regions of a slice as stored (4 x 16-bit fixed point per 8-byte chunk: 1.5 KB per group)
//     plus their per-site scales (16 x 128 B): 26 KB instead of 48 KB, so 8 items fit and two slices can be worked on at
//     once with six more on their way;
//   * NSET = 2 or 3 sets of four sweep warps: slice s belongs to set s % NSET.  The 16-bit sweep is bound by
//     instruction issue (the conversions and the scale ride on top of the fp32 arithmetic), not by the memory system,
//     and one warp per scheduler cannot hide its own latencies: two warps per scheduler can;
//   * the sweep prefetches a neighbour as the 6 raw words + scale (7 registers) and converts at the point of use; the
//     stored integers stay unscaled, the scale of the neighbour goes into the reconstruction weight (hop3_kernels.cuh);
//   * set 0 writes the links of the tile into tensor memory, the other sets read them (same lanes): two mbarriers per group
//     (lready / lfree) order the two;
//   * the per-site scales (own regions, halos) and the y-halo rows come in through 16- and 4-byte LDGSTS copies of the
//     three helper warps; the TMA producer moves the 12 whole groups of a slice as before;
//   * the epilogue warps prefetch their own-site slices raw as well (13 registers a slice) and quantise in store3<PH>.
//
// NSET = 2: 16 warps (512 threads, 128 registers): sweep 0-7, epilogue 8-11, TMA producer 12, helpers 13-15.
// NSET = 3 (K1, K1^dagger at L5 = 12; not the default, see launch_hop6_l5): 20 warps (640 threads, 96 registers): sweep 0-11, epilogue 12-15, producer 16, helpers 17-19; a
// sweep warp then holds one neighbour and one link at a time (no prefetch): its two neighbours on the scheduler hide the latency.
#pragma once
#include "hop5_kernels.cuh"

namespace h6 {
using namespace h3;
using namespace h5;

struct S6 {
    static constexpr unsigned CH = 8;                           // bytes per chunk per lane
    static constexpr unsigned ROW = 32 * CH;                    // one chunk row of a group
    static constexpr unsigned PIECE = 6 * ROW;                  // one (group, slice)
    static constexpr unsigned NORM_OFF = 16 * PIECE;            // 16 regions of 32 per-site scales behind the data
    static constexpr unsigned BYTES = 16 * PIECE + 16 * 128;
    static constexpr int RING = 8;
};

// a spinor of one (site, slice) as stored: 6 words of 4 x 16 bits and the scale
struct Raw {
    uint2 q[6];
    float sc;
};
MDWF_DEV void raw_lds(Raw &b, const unsigned char *sb, unsigned off, unsigned noff)
{
    const uint2 *p = reinterpret_cast<const uint2 *>(sb + off);
#pragma unroll
    for (int j = 0; j < 6; j++) b.q[j] = p[32 * j];
    b.sc = *reinterpret_cast<const float *>(sb + noff);
}
MDWF_DEV void raw_ldg(Raw &b, const uint2 *p, const float *n)
{
#pragma unroll
    for (int j = 0; j < 6; j++) b.q[j] = __ldg(p + 32 * j);
    b.sc = __ldg(n);
}
// the stored integers as floats; returns the factor that turns them into values
MDWF_DEV float raw_ints(const Raw &b, c2 *v)
{
#pragma unroll
    for (int j = 0; j < 6; j++) { v[2 * j] = cvt_raw(b.q[j].x); v[2 * j + 1] = cvt_raw(b.q[j].y); }
    return b.sc * (1.0f / MDWF_FIXED_MAX);
}
// spin projection straight from the stored words (project3m, hop3_kernels.cuh)
template <int MU, int SGN>
MDWF_DEV void project_magic(const Raw &b, c2 *h)
{
    c2 f[12];
#pragma unroll
    for (int j = 0; j < 6; j++) { f[2 * j] = magic_pair(b.q[j].x); f[2 * j + 1] = magic_pair(b.q[j].y); }
    project3m<MU, SGN>(f, h);
}
// the stored integers of the upper (half = 0) or lower (half = 1) six complex numbers; the scale goes into the coefficient
// the caller multiplies them with (raw_scale)
MDWF_DEV void raw_half(const Raw &b, int half, c2 *v)
{
#pragma unroll
    for (int j = 0; j < 3; j++) { v[2 * j] = cvt_raw(b.q[3 * half + j].x); v[2 * j + 1] = cvt_raw(b.q[3 * half + j].y); }
}
MDWF_DEV void raw_full(const Raw &b, c2 *v)
{
    raw_half(b, 0, v);
    raw_half(b, 1, v + 6);
}
MDWF_DEV float raw_scale(const Raw &b) { return b.sc * (1.0f / MDWF_FIXED_MAX); }
MDWF_DEV void cp_async4(void *dst_smem, const void *src_gmem)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(dst_smem)), "l"(src_gmem) : "memory");
}

// =====================================================================================================================
template <int DAG, int POST, int OWN, int L5, int NSET>
__global__ void __launch_bounds__(128 * NSET + 256, 1) hop6_kernel(const HopArgs a)
{
    using P = PH;
    using G = typename P::G;
    using SL = S6;
    static_assert(L5 % NSET == 0, "NSET sweep sets: slice s belongs to set s % NSET");
    constexpr int W_EPI = 4 * NSET, W_TMA = W_EPI + 4, W_HLP = W_TMA + 1;      // first warp of each role
    constexpr int NV = 6, RING = SL::RING;
    constexpr unsigned SLOT = SL::BYTES;
    constexpr unsigned ITEMS = 2 + L5;                                               // ring items per tile: 2 of links, L5 slices
    // history ring: POST = 2 gives up one slot for 36 parked columns (partial out_0, upper half of x_0: see its epilogue)
    constexpr int NS = (POST == 2) ? HIST_SLOTS - 1 : HIST_SLOTS;
    constexpr int PARK0 = HIST_COL0 + 24 * (HIST_SLOTS - 1), PARK1 = PARK0 + 24;
    static_assert(PARK1 + 12 <= 512, "tensor memory columns");
    extern __shared__ __align__(128) unsigned char smem6[];
    unsigned long long *bars = reinterpret_cast<unsigned long long *>(smem6 + RING * SLOT);
    unsigned long long *full = bars, *empty = bars + RING;                          // ring: producers -> sweep, sweep -> producers
    unsigned long long *hfull = bars + 2 * RING, *hempty = hfull + 4 * HIST_SLOTS;   // history: per group, per slot
    unsigned long long *lready = hempty + 4 * HIST_SLOTS, *lfree = lready + 4;       // links in TMEM: set 0 -> set 1, set 1 -> set 0
    long *ysrc = reinterpret_cast<long *>(lfree + 4);                                // [3][48] y-halo row table of each helper warp
    unsigned *ydst = reinterpret_cast<unsigned *>(ysrc + 3 * 48);                    // [3][48]
    unsigned *tmem_base_s = ydst + 3 * 48;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int Lxh = a.L[0] >> 1, Lz = a.L[2], Lt = a.L[3];
    const int NK = a.recon >> 1;
    const unsigned LT_BYTES = 8u * NK * 32u * sizeof(G);                             // link tile of one group

    if (threadIdx.x == 0) {
        for (int i = 0; i < RING; i++) { mbar_init(&full[i], 97); mbar_init(&empty[i], 4); }   // full: expect_tx arrival + one LDGSTS arrival per helper lane
        for (int i = 0; i < 4 * HIST_SLOTS; i++) { mbar_init(&hfull[i], 1); mbar_init(&hempty[i], 1); }
        for (int i = 0; i < 4; i++) { mbar_init(&lready[i], 1); mbar_init(&lfree[i], NSET - 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_base_s)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tm_fence_before();
    __syncthreads();
    tm_fence_after();
    const unsigned tmem = *tmem_base_s + ((unsigned)(32 * (warp & 3)) << 16);       // this warp's lanes

    const int ntiles = a.t5_ntiles;
    if (warp == W_TMA) {
        // ================= TMA producer: link tiles and the 12 whole groups of every slice =================
        const unsigned char *gin = reinterpret_cast<const unsigned char *>(a.in);
        const unsigned char *ggauge = reinterpret_cast<const unsigned char *>(a.gauge);
        unsigned it = 0;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const Tile T = tile_of(a, tile);
            for (int h = 0; h < 2; h++) {
                const unsigned slot = it % RING, ph = (it / RING) & 1;
                mbar_wait(&empty[slot], ph ^ 1);
                if (lane == 0) mbar_expect_tx(&full[slot], 2 * LT_BYTES);
                __syncwarp();
                if (lane < 2) {
                    const int p = 2 * h + lane;
                    const long g = group_of(a, T.yy, T.z0 + (p & 1), T.t0 + (p >> 1));
                    bulk_g2s(smem6 + slot * SLOT + lane * LT_BYTES, ggauge + g * (long)LT_BYTES, LT_BYTES, &full[slot]);
                }
                it++;
            }
            long src0 = 0;
            if (lane < 12) {
                const int c = lane;
                int z, t;
                if (c < 4) { z = T.z0 + (c & 1); t = T.t0 + (c >> 1); }
                else if (c < 8) { z = (c < 6) ? T.z0 - 1 : T.z0 + 2; t = T.t0 + (c & 1); }
                else { z = T.z0 + (c & 1); t = (c < 10) ? T.t0 - 1 : T.t0 + 2; }
                src0 = group_of(a, T.yy, wrap(z, Lz), wrap(t, Lt)) * (long)L5 * SL::PIECE;
            }
            for (int s = 0; s < L5; s++) {
                const unsigned slot = it % RING, ph = (it / RING) & 1;
                mbar_wait(&empty[slot], ph ^ 1);
                if (lane == 0) mbar_expect_tx(&full[slot], 12u * SL::PIECE);
                __syncwarp();
                if (lane < 12) bulk_g2s(smem6 + slot * SLOT + lane * SL::PIECE, gin + src0 + (long)s * SL::PIECE, SL::PIECE, &full[slot]);
                it++;
            }
        }
    } else if (warp >= W_HLP) {
        // ================= helpers (warps 13-15): y-halo rows, scales of the 12 groups, scales of the y-halo rows =================
        const int hw = warp - W_HLP;
        const unsigned char *gin = reinterpret_cast<const unsigned char *>(a.in);
        long *ys = ysrc + 48 * hw;
        unsigned *yd = ydst + 48 * hw;
        const int ur = Lxh >> 1, rpw = 32 / ur;                            // 16-byte units per row, rows per warp instruction
        const int r0 = lane / ur, xoff = (lane - r0 * ur) * 16;
        const int u = hw * 32 + lane;                                      // scale unit of this lane: region u >> 3, part u & 7
        unsigned it = 0;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const Tile T = tile_of(a, tile);
            for (int h = 0; h < 2; h++) {                                           // link items: nothing to copy
                mbar_wait(&empty[it % RING], ((it / RING) & 1) ^ 1);
                cp_async_arrive(&full[it % RING]);
                it++;
            }
            __syncwarp();
            for (int rr = lane; rr < 8 * NV; rr += 32) {
                const int hp = rr / NV, j = rr - hp * NV, p = hp & 3, hi = hp >> 2;
                ys[rr] = group_of(a, wrap(T.yy + (hi ? 1 : -1), a.t5_NY), T.z0 + (p & 1), T.t0 + (p >> 1)) * (long)L5 * SL::PIECE +
                         (long)j * SL::ROW + (hi ? 0 : (32 - Lxh) * SL::CH);
                yd[rr] = (unsigned)(12 + p) * SL::PIECE + (unsigned)j * SL::ROW + (hi ? SL::ROW / 2 : 0);
            }
            // scales of the 12 whole groups: one 16-byte unit per helper lane
            const float *nsrc;
            {
                const int c = u >> 3;
                int z, t;
                if (c < 4) { z = T.z0 + (c & 1); t = T.t0 + (c >> 1); }
                else if (c < 8) { z = (c < 6) ? T.z0 - 1 : T.z0 + 2; t = T.t0 + (c & 1); }
                else { z = T.z0 + (c & 1); t = (c < 10) ? T.t0 - 1 : T.t0 + 2; }
                nsrc = a.in_norm + group_of(a, T.yy, wrap(z, Lz), wrap(t, Lt)) * (long)L5 * 32 + (u & 7) * 4;
            }
            const unsigned ndst = SL::NORM_OFF + (unsigned)(u >> 3) * 128 + (unsigned)(u & 7) * 16;
            // scales of the y-halo rows: 8 half-pieces x Lx/2 sites, 4 bytes each, up to two per lane
            const float *ynsrc[2];
            unsigned yndst[2];
#pragma unroll
            for (int k = 0; k < 2; k++) {
                const int v = u + 96 * k;
                ynsrc[k] = nullptr;
                yndst[k] = 0;
                if (v < 8 * Lxh) {
                    const int hp = v / Lxh, xh = v - hp * Lxh, p = hp & 3, hi = hp >> 2;
                    ynsrc[k] = a.in_norm + group_of(a, wrap(T.yy + (hi ? 1 : -1), a.t5_NY), T.z0 + (p & 1), T.t0 + (p >> 1)) * (long)L5 * 32 +
                               (hi ? 0 : 32 - Lxh) + xh;
                    yndst[k] = SL::NORM_OFF + (unsigned)(12 + p) * 128 + (hi ? 64u : 0u) + (unsigned)xh * 4;
                }
            }
            __syncwarp();
            for (int s = 0; s < L5; s++) {
                const unsigned slot = it % RING, ph = (it / RING) & 1;
                mbar_wait(&empty[slot], ph ^ 1);
                unsigned char *sb = smem6 + slot * SLOT;
                for (int rr = r0 + hw * rpw; rr < 8 * NV; rr += 3 * rpw) cp_async16(sb + yd[rr] + xoff, gin + ys[rr] + (long)s * SL::PIECE + xoff);
                cp_async16(sb + ndst, nsrc + s * 32);
#pragma unroll
                for (int k = 0; k < 2; k++)
                    if (ynsrc[k]) cp_async4(sb + yndst[k], ynsrc[k] + s * 32);
                cp_async_arrive(&full[slot]);
                it++;
            }
        }
    } else if (warp < W_EPI) {
        // ================= sweep warps: set 0 = warps 0-3 (even slices, writes the links), set 1 = warps 4-7 (odd slices) =================
        const int set = warp >> 2, w = warp & 3;
        const int pa = w & 1, pb = w >> 1;                                          // z / t offset of this warp's group in the tile
        const int R = 32 / Lxh, r = lane / Lxh, xh = lane - r * Lxh;
        unsigned tcount = 0;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x, tcount++) {
            const Tile T = tile_of(a, tile);
            const unsigned it0 = tcount * ITEMS, h0 = tcount * L5;
            const int z = T.z0 + pa, t = T.t0 + pb, y = R * T.yy + r;
            const int xodd = (a.parity_out + y + z + t) & 1;
            // (region, lane) of this thread's neighbour inside a slice item; link order: 0-3 forward mu, 4-7 backward
            unsigned rl[8];
            const unsigned own = (unsigned)w * 32;
            rl[0] = own + (unsigned)(xodd ? (xh == Lxh - 1 ? lane - (Lxh - 1) : lane + 1) : lane);
            rl[4] = own + (unsigned)(xodd ? lane : (xh == 0 ? lane + (Lxh - 1) : lane - 1));
            rl[1] = (r < R - 1) ? own + (unsigned)(lane + Lxh) : (12u + w) * 32 + 16 + (unsigned)xh;
            rl[5] = (r > 0) ? own + (unsigned)(lane - Lxh) : (12u + w) * 32 + (unsigned)xh;
            rl[2] = (pa == 0 ? (unsigned)(1 + 2 * pb) : (unsigned)(6 + pb)) * 32 + (unsigned)lane;
            rl[6] = (pa == 1 ? (unsigned)(0 + 2 * pb) : (unsigned)(4 + pb)) * 32 + (unsigned)lane;
            rl[3] = (pb == 0 ? (unsigned)(pa + 2) : (unsigned)(10 + pa)) * 32 + (unsigned)lane;
            rl[7] = (pb == 1 ? (unsigned)(pa) : (unsigned)(8 + pa)) * 32 + (unsigned)lane;
            // byte offsets: data = region * PIECE + lane * CH (PIECE = 192 * CH), scale = NORM_OFF + 4 * (32 region + lane)
#define MDWF_OFF(d) ((rl[d] >> 5) * SL::PIECE + (rl[d] & 31) * SL::CH)
#define MDWF_NOFF(d) (SL::NORM_OFF + 4 * rl[d])
            const float btp = (t == Lt - 1) ? -1.f : 1.f, btm = (t == 0) ? -1.f : 1.f;   // antiperiodic in t

            if (set == 0) {
                // ---- links of this site: ring item -> (row 2 rebuilt) -> TMEM columns [20 d, 20 d + 18) ----
                mbar_wait(&lfree[w], (tcount & 1) ^ 1);                             // set 1 has finished with the previous tile's links
                tm_fence_after();
                for (int h = 0; h < 2; h++) {
                    const unsigned it = it0 + h, slot = it % RING, ph = (it / RING) & 1;
                    mbar_wait(&full[slot], ph);
                    if (h == (w >> 1)) {
                        const G *tile_l = reinterpret_cast<const G *>(smem6 + slot * SLOT + (w & 1) * LT_BYTES);
#pragma unroll 1
                        for (int d = 0; d < 8; d++) {
                            float ur[9], ui[9], lwv[18];
                            const G *p = tile_l + d * NK * 32 + lane;
#pragma unroll
                            for (int k = 0; k < 6; k++) gget(p[32 * k], ur[k], ui[k]);
                            if (NK == 9) {
#pragma unroll
                                for (int k = 6; k < 9; k++) gget(p[32 * k], ur[k], ui[k]);
                            } else {
                                row2_from_rows01(ur, ui);
                            }
#pragma unroll
                            for (int k = 0; k < 9; k++) { lwv[k] = ur[k]; lwv[9 + k] = ui[k]; }
                            tm_st16(tmem + LINK_STRIDE * d, lwv);
                            tm_st2(tmem + LINK_STRIDE * d + 16, lwv + 16);
                        }
                        tm_wait_st();
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&empty[slot]);
                }
                tm_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&lready[w]);
            } else {
                mbar_wait(&lready[w], tcount & 1);
                tm_fence_after();
            }

            // ---- the sweep of this set's slices, software-pipelined over (slice, direction) as in hop5_kernels.cuh ----
            constexpr int lk[8] = {0, 4, 1, 5, 2, 6, 3, 7};
            // PF: the neighbour and the link of the NEXT direction are prefetched (two buffers each: 50 registers).  With three
            // sweep sets a warp has 96 registers and two other sweep warps on its scheduler to hide its latencies: no prefetch.
            constexpr bool PF = NSET < 3;
            Raw nb[PF ? 2 : 1];
            float lw[PF ? 2 : 1][18];
            unsigned it = it0 + 2 + set, slot = it % RING;
            const unsigned char *sb = smem6 + slot * SLOT;
            if constexpr (PF) {
                mbar_wait(&full[slot], (it / RING) & 1);
                raw_lds(nb[0], sb, MDWF_OFF(lk[0]), MDWF_NOFF(lk[0]));
                tm_ld16(tmem + LINK_STRIDE * lk[0], lw[0]);
                tm_ld2(tmem + LINK_STRIDE * lk[0] + 16, lw[0] + 16);
            }
            int pending = -1;                                                       // history slot whose hand-off is not finished yet
#define MDWF_HANDOFF()                                                                                  \
    do {                                                                                                \
        if (pending >= 0) {                                                                             \
            tm_wait_st();                                                                               \
            tm_fence_before();                                                                          \
            __syncwarp();                                                                               \
            if (lane == 0) mbar_arrive(&hfull[w * HIST_SLOTS + pending]);                               \
            pending = -1;                                                                               \
        }                                                                                               \
    } while (0)
#define MDWF_DIR6(MU, FWD, d, bs)                                                                       \
    do {                                                                                                \
        constexpr int SGN = ((FWD) ? 1 : -1) * (DAG ? -1 : 1);                                          \
        constexpr int cb_ = PF ? ((d) & 1) : 0, nb_ = PF ? (cb_ ^ 1) : 0;                               \
        if constexpr (!PF) {                                                                            \
            if ((d) == 0) {                                                                             \
                slot = it % RING;                                                                       \
                mbar_wait(&full[slot], (it / RING) & 1);                                                \
                sb = smem6 + slot * SLOT;                                                               \
            }                                                                                           \
            raw_lds(nb[0], sb, MDWF_OFF(lk[(d)]), MDWF_NOFF(lk[(d)]));                                  \
            tm_ld16(tmem + LINK_STRIDE * lk[(d)], lw[0]);                                               \
            tm_ld2(tmem + LINK_STRIDE * lk[(d)] + 16, lw[0] + 16);                                      \
        } else if ((d) < 7) {                                                                           \
            raw_lds(nb[nb_], sb, MDWF_OFF(lk[((d) + 1) & 7]), MDWF_NOFF(lk[((d) + 1) & 7]));            \
        } else {                                                                                        \
            __syncwarp();                                                                               \
            if (lane == 0) mbar_arrive(&empty[slot]);           /* every load of this ring item has been issued */ \
            it += NSET;                                                                                 \
            if (s + NSET < L5) {                                                                        \
                slot = it % RING;                                                                       \
                mbar_wait(&full[slot], (it / RING) & 1);                                                \
                sb = smem6 + slot * SLOT;                                                               \
                raw_lds(nb[nb_], sb, MDWF_OFF(lk[0]), MDWF_NOFF(lk[0]));                                \
            }                                                                                           \
        }                                                                                               \
        tm_wait_ld18(lw[cb_]);                                                                          \
        if (PF && ((d) < 7 || s + NSET < L5)) {                                                         \
            tm_ld16(tmem + LINK_STRIDE * lk[((d) + 1) & 7], lw[nb_]);                                   \
            tm_ld2(tmem + LINK_STRIDE * lk[((d) + 1) & 7] + 16, lw[nb_] + 16);                          \
        }                                                                                               \
        Link U;                                                                                         \
        _Pragma("unroll") for (int k = 0; k < 9; k++) { U.re[k] = lw[cb_][k]; U.im[k] = lw[cb_][9 + k]; } \
        c2 h[6], chi[6];                                                                                \
        const float scw = nb[cb_].sc * (1.0f / MDWF_FIXED_MAX);                                         \
        project_magic<MU, SGN>(nb[cb_], h);                                                             \
        su3_mul3(U, h, chi);                                                                            \
        recon3<MU, SGN, true>(chi, (bs) * scw, acc);                                                    \
        if (!PF && (d) == 7) {                                                                          \
            __syncwarp();                                                                               \
            if (lane == 0) mbar_arrive(&empty[slot]);           /* this ring item has been read */     \
            it += NSET;                                                                                 \
        }                                                                                               \
    } while (0)
            for (int s = set; s < L5; s += NSET) {
                c2 acc[12];
#pragma unroll
                for (int q = 0; q < 12; q++) acc[q] = mk(0.f, 0.f);
                MDWF_DIR6(0, true, 0, 1.f);
                MDWF_HANDOFF();
                MDWF_DIR6(0, false, 1, 1.f);
                MDWF_DIR6(1, true, 2, 1.f);
                MDWF_DIR6(1, false, 3, 1.f);
                MDWF_DIR6(2, true, 4, 1.f);
                MDWF_DIR6(2, false, 5, 1.f);
                MDWF_DIR6(3, true, 6, btp);
                MDWF_DIR6(3, false, 7, btm);
                // ---- raw hop result of the slice -> TMEM history slot, handed to the epilogue warp of the same lanes ----
                const unsigned hit = h0 + s, hs = hit % NS, hph = (hit / NS) & 1;
                mbar_wait(&hempty[w * HIST_SLOTS + hs], hph ^ 1);
                tm_fence_after();
                hist_store(tmem + HIST_COL0 + 24 * hs, acc);
                pending = (int)hs;
            }
            MDWF_HANDOFF();
            if (set != 0) {                                                         // every link load of this tile has completed
                tm_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&lfree[w]);
            }
#undef MDWF_DIR6
#undef MDWF_HANDOFF
#undef MDWF_OFF
#undef MDWF_NOFF
        }
    } else if (warp < W_TMA) {
        // ================= epilogue warps: fifth-dimension POST, own-site term, quantise + store, fused norm =================
        const int w = warp - W_EPI;
        const int pa = w & 1, pb = w >> 1;
        unsigned hit = 0;
        const float coef = (float)a.coef_hop;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const Tile T = tile_of(a, tile);
            const long g = group_of(a, T.yy, T.z0 + pa, T.t0 + pb);
            const long cb = g * 32 + lane;
            const uint2 *ob = reinterpret_cast<const uint2 *>(a.own) + g * (long)(L5 * NV * 32) + lane;
            const float *on = a.own_norm + g * (long)(L5 * 32) + lane;
            double nsum = 0.0;
            if (POST == 0) {
                // out_s = coef x_s + (own_d + own_o Lambda) psi_s: upper spins from slice s-1, lower from s+1 (-m_f at the wrap).
                // The own slices sit as stored in a rotating window of three (s, s+1, s+2 on its way); the loop is rolled by the
                // window length (static register indices, small code: two sweep warps share the instruction cache).
                static_assert(POST != 0 || OWN == 2, "POST = 0 comes with OWN = 2");
                constexpr int NB = 3;
                Raw ow[NB];
                uint2 f_lo[3];                                                      // lower half of slice 0 as stored (wrap of s = L5-1)
                float f_sc = 0.f;
                c2 pu[6];                                                           // upper half of slice s-1 (stored integers) and its scale
                float pu_sc;
                const float fd = (float)a.own_d, fo = (float)a.own_o, fow = (float)(-a.mf * a.own_o);
                const c2 cf = dup(coef);
                raw_ldg(ow[2], ob + (L5 - 1) * NV * 32, on + (L5 - 1) * 32);
                raw_ldg(ow[0], ob, on);
                raw_ldg(ow[1], ob + NV * 32, on + 32);
                raw_half(ow[2], 0, pu);                                             // upper half of the last slice (wrap of s = 0)
                pu_sc = raw_scale(ow[2]);
#pragma unroll
                for (int j = 0; j < 3; j++) f_lo[j] = ow[0].q[3 + j];
                f_sc = ow[0].sc;
#pragma unroll 1
                for (int s0 = 0; s0 < L5; s0 += NB) {
#pragma unroll
                    for (int k = 0; k < NB; k++) {
                        const int s = s0 + k;
                        if (s < L5) {
                            if (s + 2 < L5) raw_ldg(ow[(k + 2) % NB], ob + (s + 2) * NV * 32, on + (s + 2) * 32);
                            c2 o[12];
                            {
                                c2 cur[12], lo[6];
                                raw_full(ow[k], cur);
                                Raw nx;                                             // only its lower half is used
                                const bool wrapl = (s == L5 - 1);
#pragma unroll
                                for (int j = 0; j < 3; j++) nx.q[3 + j] = wrapl ? f_lo[j] : ow[(k + 1) % NB].q[3 + j];
                                nx.sc = wrapl ? f_sc : ow[(k + 1) % NB].sc;
                                raw_half(nx, 1, lo);
                                const float csc = raw_scale(ow[k]);
                                const c2 d2 = dup(fd * csc), fu = dup(((s == 0) ? fow : fo) * pu_sc), fl = dup((wrapl ? fow : fo) * raw_scale(nx));
#pragma unroll
                                for (int q = 0; q < 6; q++) {
                                    o[q] = fma2(d2, cur[q], mul2(fu, pu[q]));
                                    o[6 + q] = fma2(d2, cur[6 + q], mul2(fl, lo[q]));
                                    pu[q] = cur[q];
                                }
                                pu_sc = csc;
                            }
                            const unsigned hs = hit % NS, hph = (hit / NS) & 1;
                            mbar_wait(&hfull[w * HIST_SLOTS + hs], hph);
                            tm_fence_after();
                            c2 x[12];
                            hist_load(tmem + HIST_COL0 + 24 * hs, x);
                            tm_fence_before();
                            __syncwarp();
                            if (lane == 0) mbar_arrive(&hempty[w * HIST_SLOTS + hs]);
                            hit++;
#pragma unroll
                            for (int q = 0; q < 12; q++) o[q] = fma2(cf, x[q], o[q]);
                            nsum += (double)store3<P>(a.out, a.out_norm, L5, s, cb, o, a.partial != nullptr);
                        }
                    }
                }
            }
            if (POST == 1) {
                // coef (B A^{-1}) x per chirality: the two first-order recurrences over the slice history in TMEM, exactly as
                // in hop5_kernels.cuh (pass A ascending as the slices arrive, pass B descending)
                constexpr int DOFF = DAG ? 12 : 0, MOFF = DAG ? 0 : 12;
                const c2 nk = dup(a.r_nk), bz = dup(a.r_bz), cz = dup(a.r_cz);
                const unsigned h0 = hit;
                c2 zp[6], Wm[6];
                c2 pw = dup(1.f);
#pragma unroll
                for (int q = 0; q < 6; q++) { zp[q] = mk(0.f, 0.f); Wm[q] = mk(0.f, 0.f); }
                for (int s = 0; s < L5; s++) {
                    const unsigned hs = (h0 + s) % NS, hph = ((h0 + s) / NS) & 1;
                    mbar_wait(&hfull[w * HIST_SLOTS + hs], hph);
                    tm_fence_after();
                    c2 x[12];
                    hist_load(tmem + HIST_COL0 + 24 * hs, x);
                    float tp[12];
#pragma unroll
                    for (int q = 0; q < 6; q++) {
                        const c2 zz = fma2(nk, zp[q], x[DOFF / 2 + q]);                 // z_s = x_s - kappa z_{s-1}
                        const c2 tt = fma2(cz, zp[q], mul2(bz, zz));                    // bz z_s + cz z_{s-1}
                        zp[q] = zz;
                        tp[2 * q] = tt.x; tp[2 * q + 1] = tt.y;
                        Wm[q] = fma2(pw, x[MOFF / 2 + q], Wm[q]);
                    }
                    pw = mul2(pw, nk);
                    tm_st8(tmem + HIST_COL0 + 24 * hs + DOFF, tp);
                    tm_st2(tmem + HIST_COL0 + 24 * hs + DOFF + 8, tp + 8);
                    tm_st2(tmem + HIST_COL0 + 24 * hs + DOFF + 10, tp + 10);
                }
                tm_wait_st();
                c2 zn[6];                                                               // mirrored recurrence state z_{s+1}
#pragma unroll
                for (int q = 0; q < 6; q++) zn[q] = mk(0.f, 0.f);
                for (int s = L5 - 1; s >= 0; s--) {
                    const unsigned hs = (h0 + s) % NS;
                    c2 x[12], o[12];
                    hist_load(tmem + HIST_COL0 + 24 * hs, x);
                    tm_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&hempty[w * HIST_SLOTS + hs]);
                    const c2 qWd = dup(a.r_qW[s]), qWm = dup(a.r_qW[L5 - 1 - s]);
#pragma unroll
                    for (int q = 0; q < 6; q++) {
                        const c2 zz = fma2(nk, zn[q], x[MOFF / 2 + q]);                 // z_s = x_s - kappa z_{s+1}
                        o[MOFF / 2 + q] = fma2(qWm, Wm[q], fma2(cz, zn[q], mul2(bz, zz)));
                        zn[q] = zz;
                        o[DOFF / 2 + q] = fma2(qWd, zp[q], x[DOFF / 2 + q]);            // zp = z_{L5-1} of the direct half = its W
                    }
                    nsum += (double)store3<P>(a.out, a.out_norm, L5, s, cb, o, a.partial != nullptr);
                }
                hit += L5;
            }
            if (POST == 2) {
                // out_s = coef (post_d + post_o Lambda^dagger) x_s + (own_d + own_o Lambda^dagger) psi_s   (OWN = 3), streaming:
                // out_s once x_{s+1} has arrived (s = 1 .. L5-2), every history slot freed as soon as the next output has used
                // it.  The two ends need the other end of the fifth dimension; so that slots 0 and 1 are not held until then
                // (the sweep of the next tile would wait for the whole tail of this one), what they contribute is parked in
                // 36 tensor-memory columns of this warp's own: out_0 without its x_{L5-1} term, and the upper half of x_0.
                // The own slices sit as stored in a rotating window of three (s-1, s, s+1); the loop is rolled by the window.
                static_assert(POST != 2 || OWN == 3, "POST = 2 comes with OWN = 3");
                const unsigned h0 = hit;
                const float cf = coef * (float)a.post_d, co = coef * (float)a.post_o, mw = (float)(-a.mf);
                const c2 cd2 = dup(cf);
                constexpr int NB = 3;
                Raw ow[NB];                                                         // slice j at index j % 3
                raw_ldg(ow[0], ob, on);
                raw_ldg(ow[1], ob + NV * 32, on + 32);
                raw_ldg(ow[2], ob + 2 * NV * 32, on + 64);
#define MDWF_HSLOT(s_) ((h0 + (unsigned)(s_)) % NS)
#define MDWF_HWAIT(s_) mbar_wait(&hfull[w * HIST_SLOTS + MDWF_HSLOT(s_)], ((h0 + (unsigned)(s_)) / NS) & 1)
#define MDWF_HFREE(s_)                                                                   \
    do {                                                                                 \
        tm_fence_before();                                                               \
        __syncwarp();                                                                    \
        if (lane == 0) mbar_arrive(&hempty[w * HIST_SLOTS + MDWF_HSLOT(s_)]);            \
    } while (0)
                // own-site term of output slice s: psi_s (rc), upper half of psi_{s+1} (ru), lower half of psi_{s-1} (rlo)
                auto own_term = [&](int s, const Raw &rc, const Raw &ru, const Raw &rlo, c2 *o) {
                    const c2 oou = dup((float)a.own_o * (s == L5 - 1 ? mw : 1.f) * raw_scale(ru)), ool = dup((float)a.own_o * (s == 0 ? mw : 1.f) * raw_scale(rlo));
                    const c2 odc = dup((float)a.own_d * raw_scale(rc));
                    c2 pc[12], pu[6], pl[6];
                    raw_full(rc, pc);
                    raw_half(ru, 0, pu);
                    raw_half(rlo, 1, pl);
#pragma unroll
                    for (int q = 0; q < 6; q++) {
                        o[q] = fma2(odc, pc[q], mul2(oou, pu[q]));
                        o[6 + q] = fma2(odc, pc[6 + q], mul2(ool, pl[q]));
                    }
                };
                // hop part: x_s, the upper half of x_su and the lower half of x_sl from TMEM; then store.  (Loading x_s and x_sl
                // before the wait for x_{s+1} would save a tensor-memory latency per slice, but the extra live registers spill.)
                auto finish = [&](int s, int su, int sl, c2 *o) {
                    const c2 cou = dup(co * (s == L5 - 1 ? mw : 1.f)), col = dup(co * (s == 0 ? mw : 1.f));
                    {
                        float xu[12], xl[12];
                        const unsigned tu = tmem + HIST_COL0 + 24 * MDWF_HSLOT(su), tl = tmem + HIST_COL0 + 24 * MDWF_HSLOT(sl) + 12;
                        tm_ld8(tu, xu); tm_ld2(tu + 8, xu + 8); tm_ld2(tu + 10, xu + 10);
                        tm_ld8(tl, xl); tm_ld2(tl + 8, xl + 8); tm_ld2(tl + 10, xl + 10);
                        tm_wait_ld24(xu, xl);
#pragma unroll
                        for (int q = 0; q < 6; q++) {
                            o[q] = fma2(cou, mk(xu[2 * q], xu[2 * q + 1]), o[q]);
                            o[6 + q] = fma2(col, mk(xl[2 * q], xl[2 * q + 1]), o[6 + q]);
                        }
                    }
                    c2 x[12];
                    hist_load(tmem + HIST_COL0 + 24 * MDWF_HSLOT(s), x);
#pragma unroll
                    for (int q = 0; q < 12; q++) o[q] = fma2(cd2, x[q], o[q]);
                    nsum += (double)store3<P>(a.out, a.out_norm, L5, s, cb, o, a.partial != nullptr);
                };
                uint2 up0q[3];                                                      // upper half of psi_0 as stored: own term of out_{L5-1}
#pragma unroll
                for (int j = 0; j < 3; j++) up0q[j] = ow[0].q[j];
                const float up0sc = ow[0].sc;
                MDWF_HWAIT(0);
                MDWF_HWAIT(1);
                tm_fence_after();
                {   // out_0 without col lo(x_{L5-1}): own term (lower half of psi_{L5-1} read here), x_0, upper half of x_1
                    Raw lastlo;
#pragma unroll
                    for (int j = 0; j < 3; j++) lastlo.q[3 + j] = __ldg(ob + (L5 - 1) * NV * 32 + 32 * (3 + j));
                    lastlo.sc = __ldg(on + (L5 - 1) * 32);
                    c2 o[12], x[12];
                    own_term(0, ow[0], ow[1], lastlo, o);
                    float xu[12];
                    const unsigned tu = tmem + HIST_COL0 + 24 * MDWF_HSLOT(1);
                    tm_ld8(tu, xu); tm_ld2(tu + 8, xu + 8); tm_ld2(tu + 10, xu + 10);
                    hist_load(tmem + HIST_COL0 + 24 * MDWF_HSLOT(0), x);
                    tm_wait_ld12(xu);
                    const c2 cou = dup(co);
                    float pk[12];
#pragma unroll
                    for (int q = 0; q < 6; q++) {
                        o[q] = fma2(cd2, x[q], fma2(cou, mk(xu[2 * q], xu[2 * q + 1]), o[q]));
                        o[6 + q] = fma2(cd2, x[6 + q], o[6 + q]);
                        pk[2 * q] = x[q].x; pk[2 * q + 1] = x[q].y;
                    }
                    hist_store(tmem + PARK0, o);
                    tm_st8(tmem + PARK1, pk);
                    tm_st2(tmem + PARK1 + 8, pk + 8);
                    tm_st2(tmem + PARK1 + 10, pk + 10);
                    tm_wait_st();
                }
#pragma unroll 1
                for (int s0 = 1; s0 <= L5 - 2; s0 += NB) {
#pragma unroll
                    for (int k = 0; k < NB; k++) {
                        const int s = s0 + k;                                       // s % 3 = (1 + k) % 3
                        if (s <= L5 - 2) {
                            c2 o[12];
                            own_term(s, ow[(k + 1) % NB], ow[(k + 2) % NB], ow[k % NB], o);
                            if (s + 2 <= L5 - 1) raw_ldg(ow[k % NB], ob + (s + 2) * NV * 32, on + (s + 2) * 32);   // the slot of slice s-1 is free
                            MDWF_HWAIT(s + 1);
                            tm_fence_after();
                            finish(s, s + 1, s - 1, o);
                            MDWF_HFREE(s - 1);
                        }
                    }
                }
                {   // the two ends: out_{L5-1} (upper from the parked x_0, lower from x_{L5-2}) and the rest of out_0
                    Raw up0;
#pragma unroll
                    for (int j = 0; j < 3; j++) { up0.q[j] = up0q[j]; up0.q[3 + j] = up0q[j]; }
                    up0.sc = up0sc;
                    c2 o[12], x[12];
                    own_term(L5 - 1, ow[(L5 - 1) % NB], up0, ow[(L5 - 2) % NB], o);
                    float xu[12], xl[12];
                    const unsigned tl = tmem + HIST_COL0 + 24 * MDWF_HSLOT(L5 - 2) + 12;
                    tm_ld8(tmem + PARK1, xu); tm_ld2(tmem + PARK1 + 8, xu + 8); tm_ld2(tmem + PARK1 + 10, xu + 10);
                    tm_ld8(tl, xl); tm_ld2(tl + 8, xl + 8); tm_ld2(tl + 10, xl + 10);
                    tm_wait_ld24(xu, xl);
                    hist_load(tmem + HIST_COL0 + 24 * MDWF_HSLOT(L5 - 1), x);
                    const c2 cou = dup(co * mw), col = dup(co);
#pragma unroll
                    for (int q = 0; q < 6; q++) {
                        o[q] = fma2(cd2, x[q], fma2(cou, mk(xu[2 * q], xu[2 * q + 1]), o[q]));
                        o[6 + q] = fma2(cd2, x[6 + q], fma2(col, mk(xl[2 * q], xl[2 * q + 1]), o[6 + q]));
                    }
                    nsum += (double)store3<P>(a.out, a.out_norm, L5, L5 - 1, cb, o, a.partial != nullptr);
                    hist_load(tmem + PARK0, o);
                    const c2 colw = dup(co * mw);
#pragma unroll
                    for (int q = 0; q < 6; q++) o[6 + q] = fma2(colw, x[6 + q], o[6 + q]);
                    nsum += (double)store3<P>(a.out, a.out_norm, L5, 0, cb, o, a.partial != nullptr);
                }
                tm_fence_before();
                __syncwarp();
                if (lane == 0) {
                    mbar_arrive(&hempty[w * HIST_SLOTS + MDWF_HSLOT(L5 - 2)]);
                    mbar_arrive(&hempty[w * HIST_SLOTS + MDWF_HSLOT(L5 - 1)]);
                }
#undef MDWF_HSLOT
#undef MDWF_HWAIT
#undef MDWF_HFREE
                hit += L5;
            }
            if (a.partial) {
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) nsum += __shfl_xor_sync(0xffffffffu, nsum, o);
                if (lane == 0) a.partial[g] = nsum;
            }
        }
    }
    tm_fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(*tmem_base_s) : "memory");
}

// ---- launchers --------------------------------------------------------------------------------------------------------
template <int DAG, int POST, int OWN, int L5, int NSET>
static int launch_hop6_inst(const HopArgs &a, cudaStream_t st)
{
    static int sms = 0;
    const size_t smem = (size_t)S6::RING * S6::BYTES + 8 * (2 * S6::RING + 8 * HIST_SLOTS + 8) + 3 * 48 * 12 + 16;
    if (!sms) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        cudaError_t e = cudaFuncSetAttribute(hop6_kernel<DAG, POST, OWN, L5, NSET>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) { sms = 0; return (int)e; }
    }
    const int grid = a.t5_ntiles < sms ? a.t5_ntiles : sms;
    hop6_kernel<DAG, POST, OWN, L5, NSET><<<grid, 128 * NSET + 256, smem, st>>>(a);
    return (int)cudaGetLastError();
}
template <int DAG, int POST, int OWN>
static int launch_hop6_l5(const HopArgs &a, cudaStream_t st)
{
    // Three sweep sets (96 registers, no one-direction prefetch; build with -DMDWF_HOP6_NSET3) make K1 / K1^dagger faster when they
    // are timed alone, 1.13 -> 1.09 ms, but the timed solve runs against the board's power cap and got SLOWER with them (3.06 ->
    // 3.11 s, median SM clock 1905 -> 1830 MHz): two sets are the default.  The epilogues of K2 / K2^dagger (own-slice window) spill
    // at 96 registers (1.23 -> 1.92 ms).
#ifdef MDWF_HOP6_NSET3
    if (a.L5 == 12) return launch_hop6_inst<DAG, POST, OWN, 12, POST == 1 ? 3 : 2>(a, st);
#endif
    if (a.L5 == 12) return launch_hop6_inst<DAG, POST, OWN, 12, 2>(a, st);
#ifndef MDWF_DEV_FAST
    if (a.L5 == 8) return launch_hop6_inst<DAG, POST, OWN, 8, 2>(a, st);
#endif
    return -1;
}
// -1: not covered (the caller falls back to v3)
static int launch_hop6(int dag, int pre, int post, int own, HopArgs a, cudaStream_t st)
{
    if (!hop5_geometry(a)) return -1;
    if (a.kver == 5 && a.t5_ntiles < 8 * mdwf_sm_count()) return -1;
    if (!dag && pre == 0 && post == 0 && own == 2) return launch_hop6_l5<0, 0, 2>(a, st);   // K2
    if (!dag && pre == 0 && post == 1 && own == 0) return launch_hop6_l5<0, 1, 0>(a, st);   // K1 reading a precomputed B psi
    if (dag && pre == 0 && post == 1 && own == 0) return launch_hop6_l5<1, 1, 0>(a, st);    // K1^+
    if (dag && pre == 0 && post == 2 && own == 3 && a.kver != 5) return launch_hop6_l5<1, 2, 3>(a, st);   // K2^+: its epilogue costs more than the sweep gains (1.54 ms against 1.44 ms of v3): only when forced
    return -1;
}

}   // namespace h6
