// hop5_kernels.cuh -- v5 of the fused Wilson-hopping + fifth-dimension kernels (fp32 arithmetic): a persistent,
// warp-specialised TILE SWEEP.  One CTA per SM owns a 4D tile of 2(z) x 2(t) 32-site groups (128 output sites) and sweeps
// it through the fifth dimension, one s-slice per step:
//
//   producer warp (1)   streams the tile's input through a shared-memory ring with the TMA engine (cp.async.bulk +
//                       mbarrier): first the link tiles of the 4 groups (two ring items), then per slice 12 whole
//                       neighbour groups (the 4 own positions, 4 z-halo, 4 t-halo: 3 KB each in fp32) and 8 y-halo
//                       rows.  A staged group serves every output site that touches it (x+-, the inner y hops, the
//                       in-tile z / t hops): 16 group-slices enter the SM per 4 output group-slices instead of the ~6 per
//                       output group that the per-group kernels pull through L1.
//   sweep warps (4)     one warp per group, one thread per 4D site.  They never touch global memory: links live in
//                       TENSOR MEMORY (TMEM, 144 columns per lane, written once per tile), neighbour spinors come out of
//                       the ring with conflict-free LDS.128, and the raw hop result of the slice (24 words) goes into
//                       a TMEM ring of slice slots.  All arithmetic is packed f32x2 (hop3_kernels.cuh).
//   epilogue warps (4)  warp 4+w reads what sweep warp w left in TMEM (same lanes), applies the fifth-dimension POST
//                       operator (B A^{-1} by its two first-order recurrences, or the bidiagonal Lambda^dagger form),
//                       adds the own-site term (own slices loaded from global memory exactly once, prefetched a slice
//                       ahead), stores, and accumulates the fused norm.  Their global latency hides behind the sweep.
//
// TMEM is used as a per-thread scratchpad (tcgen05.st / tcgen05.ld, shape 32x32b: lane = thread), not as an MMA
// accumulator: it is the only on-chip memory left once the ring takes the shared memory, and it lets the s-recurrences
// of A^{-1} (one forward, one backward in s) run over a slice history without registers.
//
// Geometry: Lx/2 in {2,4,8,16} (a 32-site group = 32/(Lx/2) whole x-rows of one (z,t) plane), Ly a multiple of that
// row count, L5 in {8, 12}.  Everything else falls back to the v3 family.
#pragma once
#include "hop3_kernels.cuh"

namespace h5 {
using namespace h3;

constexpr int RING = 4;                  // ring items of SLOT_BYTES in shared memory
constexpr int LINK_STRIDE = 20;          // TMEM columns [20 d, 20 d + 18): link d (9 real parts, 9 imaginary parts)
constexpr int HIST_COL0 = 160;           // TMEM columns 160..: history ring of 24-column slice slots
constexpr int HIST_SLOTS = 14;           // (512 - 160) / 24

// ---- mbarrier / TMEM helpers ----------------------------------------------------------------------------------------
MDWF_DEV void mbar_arrive(unsigned long long *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// 16-byte asynchronous copy (LDGSTS) and the arrival it triggers on an mbarrier once this thread's copies have landed
MDWF_DEV void cp_async16(void *dst_smem, const void *src_gmem)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst_smem)), "l"(src_gmem) : "memory");
}
MDWF_DEV void cp_async_arrive(unsigned long long *bar)
{
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
MDWF_DEV void tm_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
MDWF_DEV void tm_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
MDWF_DEV void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
MDWF_DEV void tm_st16(unsigned ta, const float *r)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(ta),
                 "f"(r[0]), "f"(r[1]), "f"(r[2]), "f"(r[3]), "f"(r[4]), "f"(r[5]), "f"(r[6]), "f"(r[7]), "f"(r[8]), "f"(r[9]), "f"(r[10]),
                 "f"(r[11]), "f"(r[12]), "f"(r[13]), "f"(r[14]), "f"(r[15])
                 : "memory");
}
MDWF_DEV void tm_st8(unsigned ta, const float *r)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(ta), "f"(r[0]), "f"(r[1]), "f"(r[2]),
                 "f"(r[3]), "f"(r[4]), "f"(r[5]), "f"(r[6]), "f"(r[7])
                 : "memory");
}
MDWF_DEV void tm_st2(unsigned ta, const float *r)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1,%2};" ::"r"(ta), "f"(r[0]), "f"(r[1]) : "memory");
}
MDWF_DEV void tm_ld16(unsigned ta, float *r)
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3]), "=f"(r[4]), "=f"(r[5]), "=f"(r[6]), "=f"(r[7]), "=f"(r[8]), "=f"(r[9]),
                   "=f"(r[10]), "=f"(r[11]), "=f"(r[12]), "=f"(r[13]), "=f"(r[14]), "=f"(r[15])
                 : "r"(ta));
}
MDWF_DEV void tm_ld8(unsigned ta, float *r)
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3]), "=f"(r[4]), "=f"(r[5]), "=f"(r[6]), "=f"(r[7])
                 : "r"(ta));
}
MDWF_DEV void tm_ld2(unsigned ta, float *r)
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0,%1}, [%2];" : "=f"(r[0]), "=f"(r[1]) : "r"(ta));
}
// tcgen05.wait::ld with the loaded registers threaded through it, so that no use is scheduled above the wait
MDWF_DEV void tm_wait_ld18(float *r)
{
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+f"(r[0]), "+f"(r[1]), "+f"(r[2]), "+f"(r[3]), "+f"(r[4]), "+f"(r[5]), "+f"(r[6]), "+f"(r[7]), "+f"(r[8]), "+f"(r[9]),
                   "+f"(r[10]), "+f"(r[11]), "+f"(r[12]), "+f"(r[13]), "+f"(r[14]), "+f"(r[15]), "+f"(r[16]), "+f"(r[17])
                 :);
}
MDWF_DEV void tm_wait_ld24(float *r)
{
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+f"(r[0]), "+f"(r[1]), "+f"(r[2]), "+f"(r[3]), "+f"(r[4]), "+f"(r[5]), "+f"(r[6]), "+f"(r[7]), "+f"(r[8]), "+f"(r[9]),
                   "+f"(r[10]), "+f"(r[11]), "+f"(r[12]), "+f"(r[13]), "+f"(r[14]), "+f"(r[15]), "+f"(r[16]), "+f"(r[17]), "+f"(r[18]),
                   "+f"(r[19]), "+f"(r[20]), "+f"(r[21]), "+f"(r[22]), "+f"(r[23])
                 :);
}
MDWF_DEV void tm_wait_ld24(float *a, float *b)
{
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+f"(a[0]), "+f"(a[1]), "+f"(a[2]), "+f"(a[3]), "+f"(a[4]), "+f"(a[5]), "+f"(a[6]), "+f"(a[7]), "+f"(a[8]), "+f"(a[9]),
                   "+f"(a[10]), "+f"(a[11]), "+f"(b[0]), "+f"(b[1]), "+f"(b[2]), "+f"(b[3]), "+f"(b[4]), "+f"(b[5]), "+f"(b[6]), "+f"(b[7]),
                   "+f"(b[8]), "+f"(b[9]), "+f"(b[10]), "+f"(b[11])
                 :);
}
MDWF_DEV void tm_wait_ld12(float *a)
{
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+f"(a[0]), "+f"(a[1]), "+f"(a[2]), "+f"(a[3]), "+f"(a[4]), "+f"(a[5]), "+f"(a[6]), "+f"(a[7]), "+f"(a[8]), "+f"(a[9]),
                   "+f"(a[10]), "+f"(a[11])
                 :);
}
// 24 words of one slice slot <-> 12 complex pairs
MDWF_DEV void hist_store(unsigned ta, const c2 *x)
{
    float r[24];
#pragma unroll
    for (int q = 0; q < 12; q++) { r[2 * q] = x[q].x; r[2 * q + 1] = x[q].y; }
    tm_st16(ta, r);
    tm_st8(ta + 16, r + 16);
}
MDWF_DEV void hist_load(unsigned ta, c2 *x)
{
    float r[24];
    tm_ld16(ta, r);
    tm_ld8(ta + 16, r + 16);
    tm_wait_ld24(r);
#pragma unroll
    for (int q = 0; q < 12; q++) x[q] = mk(r[2 * q], r[2 * q + 1]);
}
// ---- tile geometry ---------------------------------------------------------------------------------------------------
struct Tile {
    int yy, z0, t0;
};
MDWF_DEV Tile tile_of(const HopArgs &a, int idx)
{
    // order: y-group fastest, then the z-pairs of a chunk, then t-pairs, then z-chunks (t-halo reuse out of L2)
    const unsigned q1 = fdiv((unsigned)idx, a.t5_dNY), yy = idx - q1 * a.t5_NY;
    const unsigned q2 = fdiv(q1, a.t5_dnzq), zq = q1 - q2 * a.t5_nzq;
    const unsigned q3 = fdiv(q2, a.t5_dNT), tp = q2 - q3 * a.t5_NT;
    Tile t;
    t.yy = (int)yy;
    t.z0 = 2 * (int)(q3 * a.t5_nzq + zq);
    t.t0 = 2 * (int)tp;
    return t;
}
MDWF_DEV long group_of(const HopArgs &a, int yy, int z, int t) { return ((long)t * a.L[2] + z) * a.t5_NY + yy; }
MDWF_DEV int wrap(int v, int n) { return v < 0 ? v + n : (v >= n ? v - n : v); }

// Shared-memory ring item of one slice: 16 regions of PIECE bytes.
//   regions 0..3   own positions p = a + 2 b (a = z offset, b = t offset of the group in the tile)
//   regions 4..7   z halo: 4 + b: (z0-1, t0+b),  6 + b: (z0+2, t0+b)
//   regions 8..11  t halo: 8 + a: (z0+a, t0-1), 10 + a: (z0+a, t0+2)
//   regions 12..15 y halo of own position p: per chunk row (512 B) bytes [0,256) hold the last x-row of the group below,
//                  bytes [256,512) the first x-row of the group above
template <class P> struct Slot {
    using V = typename P::V;
    static constexpr unsigned CH = sizeof(V);                  // bytes per chunk per lane (16 fp32, 8 16-bit)
    static constexpr unsigned ROW = 32 * CH;                   // one chunk row of a group
    static constexpr unsigned PIECE = P::NV * ROW;             // one (group, slice)
    static constexpr unsigned BYTES = 16 * PIECE;
};

// =====================================================================================================================
template <class P, int DAG, int PRE, int POST, int OWN, int L5>
__global__ void __launch_bounds__(384, 1) hop5_kernel(const HopArgs a)
{
    using V = typename P::V;
    using G = typename P::G;
    using SL = Slot<P>;
    static_assert(!P::HALF, "v5: fp32 storage only so far");
    static_assert(PRE == 0, "v5: B-on-load not yet");
    constexpr int NV = P::NV;
    constexpr unsigned SLOT = SL::BYTES;
    // history ring: POST = 2 gives up one slot for 36 parked columns (out_0 without its x_{L5-1} term, upper half of x_0)
    constexpr int NS = (POST == 2) ? HIST_SLOTS - 1 : HIST_SLOTS;
    constexpr int PARK0 = HIST_COL0 + 24 * (HIST_SLOTS - 1), PARK1 = PARK0 + 24;
    static_assert(PARK1 + 12 <= 512, "tensor memory columns");
    extern __shared__ __align__(128) unsigned char smem5[];
    unsigned long long *bars = reinterpret_cast<unsigned long long *>(smem5 + RING * SLOT);
    unsigned long long *full = bars, *empty = bars + RING;                          // ring: producer -> sweep, sweep -> producer
    unsigned long long *hfull = bars + 2 * RING, *hempty = hfull + 4 * HIST_SLOTS;   // history: per warp pair, per slot
    unsigned long long *lfree = hempty + 4 * HIST_SLOTS;                             // unused (links ride in the ring)
    long *ysrc = reinterpret_cast<long *>(lfree + 4);                                // [3][48] y-halo row table, one per helper warp (they may be a tile apart)
    unsigned *ydst = reinterpret_cast<unsigned *>(ysrc + 3 * 48);                    // [3][48]
    unsigned *tmem_base_s = ydst + 3 * 48;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int Lxh = a.L[0] >> 1, Ly = a.L[1], Lz = a.L[2], Lt = a.L[3];
    const int NK = a.recon >> 1;
    const unsigned LT_BYTES = 8u * NK * 32u * sizeof(G);                             // link tile of one group

    if (threadIdx.x == 0) {
        for (int i = 0; i < RING; i++) { mbar_init(&full[i], 97); mbar_init(&empty[i], 4); }   // full: expect_tx arrival + one cp.async arrival per producer lane
        for (int i = 0; i < 4 * HIST_SLOTS; i++) { mbar_init(&hfull[i], 1); mbar_init(&hempty[i], 1); }
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
    if (warp == 8) {
        // ================= producer 1: TMA stream of link tiles and whole groups =================
        const unsigned char *gin = reinterpret_cast<const unsigned char *>(a.in);
        const unsigned char *ggauge = reinterpret_cast<const unsigned char *>(a.gauge);
        unsigned it = 0;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const Tile T = tile_of(a, tile);
            // ---- links: two ring items of two groups each ----
            for (int h = 0; h < 2; h++) {
                const unsigned slot = it % RING, ph = (it / RING) & 1;
                mbar_wait(&empty[slot], ph ^ 1);
                if (lane == 0) mbar_expect_tx(&full[slot], 2 * LT_BYTES);
                __syncwarp();
                if (lane < 2) {
                    const int p = 2 * h + lane;
                    const long g = group_of(a, T.yy, T.z0 + (p & 1), T.t0 + (p >> 1));
                    bulk_g2s(smem5 + slot * SLOT + lane * LT_BYTES, ggauge + g * (long)LT_BYTES, LT_BYTES, &full[slot]);
                }
                it++;
            }
            // ---- the 12 whole groups of a slice: lane c < 12 issues one bulk copy (source offset at s = 0) ----
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
                if (lane < 12) bulk_g2s(smem5 + slot * SLOT + lane * SL::PIECE, gin + src0 + (long)s * SL::PIECE, SL::PIECE, &full[slot]);
                it++;
            }
        }
    } else if (warp >= 9) {
        // ================= producers 2-4 (warps 9-11, a third of the rows each): the 8 y-halo rows of every slice (6 chunk rows of Lx/2 lanes each) =================
        // 16-byte asynchronous copies (LDGSTS) spread over the lanes, completion signalled on the same mbarrier: bulk
        // copies of 256 B cost the TMA engine as much as whole groups (measured: 48 of them per slice double the kernel time).
        const unsigned char *gin = reinterpret_cast<const unsigned char *>(a.in);
        const int nyu = (8 * NV * Lxh) / 32;                              // copies per lane per slice
        const int xoff = (lane & (Lxh - 1)) * SL::CH, rpw = 32 / Lxh, r0 = lane / Lxh;   // rows per warp instruction, this lane's row
        unsigned it = 0;
        ysrc += 48 * (warp - 9);
        ydst += 48 * (warp - 9);
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const Tile T = tile_of(a, tile);
            for (int h = 0; h < 2; h++) {                                           // link items: nothing to copy
                mbar_wait(&empty[it % RING], ((it / RING) & 1) ^ 1);
                cp_async_arrive(&full[it % RING]);
                it++;
            }
            // row table of the tile (8 half-pieces x NV chunk rows): source offset at s = 0, offset inside the ring item
            __syncwarp();
            for (int rr = lane; rr < 8 * NV; rr += 32) {
                const int hp = rr / NV, j = rr - hp * NV, p = hp & 3, hi = hp >> 2;
                ysrc[rr] = group_of(a, wrap(T.yy + (hi ? 1 : -1), a.t5_NY), T.z0 + (p & 1), T.t0 + (p >> 1)) * (long)L5 * SL::PIECE +
                           (long)j * SL::ROW + (hi ? 0 : (32 - Lxh) * SL::CH);
                ydst[rr] = (unsigned)(12 + p) * SL::PIECE + (unsigned)j * SL::ROW + (hi ? SL::ROW / 2 : 0);
            }
            __syncwarp();
            for (int s = 0; s < L5; s++) {
                const unsigned slot = it % RING, ph = (it / RING) & 1;
                mbar_wait(&empty[slot], ph ^ 1);
                unsigned char *sb = smem5 + slot * SLOT;
                for (int i = warp - 9, rr = r0 + (warp - 9) * rpw; i < nyu; i += 3, rr += 3 * rpw)
                    cp_async16(sb + ydst[rr] + xoff, gin + ysrc[rr] + (long)s * SL::PIECE + xoff);
                cp_async_arrive(&full[slot]);
                it++;
            }
        }
    } else if (warp < 4) {
        // ================= sweep warps: the hop, out of shared memory and TMEM =================
        const int pa = warp & 1, pb = warp >> 1;                                    // z / t offset of this warp's group in the tile
        const int R = 32 / Lxh, r = lane / Lxh, xh = lane - r * Lxh;
        unsigned it = 0, hit = 0;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const Tile T = tile_of(a, tile);
            const int z = T.z0 + pa, t = T.t0 + pb, y = R * T.yy + r;
            const int xodd = (a.parity_out + y + z + t) & 1;
            // byte offset of chunk 0 of this thread's neighbour inside a slice item; link order: 0-3 forward mu, 4-7 backward
            unsigned off[8];
            const unsigned own = (unsigned)warp * SL::PIECE;
            off[0] = own + (unsigned)(xodd ? (xh == Lxh - 1 ? lane - (Lxh - 1) : lane + 1) : lane) * SL::CH;
            off[4] = own + (unsigned)(xodd ? lane : (xh == 0 ? lane + (Lxh - 1) : lane - 1)) * SL::CH;
            off[1] = (r < R - 1) ? own + (unsigned)(lane + Lxh) * SL::CH : (12u + warp) * SL::PIECE + SL::ROW / 2 + (unsigned)xh * SL::CH;
            off[5] = (r > 0) ? own + (unsigned)(lane - Lxh) * SL::CH : (12u + warp) * SL::PIECE + (unsigned)xh * SL::CH;
            off[2] = (pa == 0 ? (unsigned)(1 + 2 * pb) : (unsigned)(6 + pb)) * SL::PIECE + (unsigned)lane * SL::CH;
            off[6] = (pa == 1 ? (unsigned)(0 + 2 * pb) : (unsigned)(4 + pb)) * SL::PIECE + (unsigned)lane * SL::CH;
            off[3] = (pb == 0 ? (unsigned)(pa + 2) : (unsigned)(10 + pa)) * SL::PIECE + (unsigned)lane * SL::CH;
            off[7] = (pb == 1 ? (unsigned)(pa) : (unsigned)(8 + pa)) * SL::PIECE + (unsigned)lane * SL::CH;
            const float btp = (t == Lt - 1) ? -1.f : 1.f, btm = (t == 0) ? -1.f : 1.f;   // antiperiodic in t

            // ---- links of this site: ring item -> (row 2 rebuilt) -> TMEM columns [20 d, 20 d + 18) ----
            for (int h = 0; h < 2; h++) {
                const unsigned slot = it % RING, ph = (it / RING) & 1;
                mbar_wait(&full[slot], ph);
                if (h == (warp >> 1)) {
                    const G *tile_l = reinterpret_cast<const G *>(smem5 + slot * SLOT + (warp & 1) * LT_BYTES);
#pragma unroll 1
                    for (int d = 0; d < 8; d++) {
                        float ur[9], ui[9], w[18];
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
                        for (int k = 0; k < 9; k++) { w[k] = ur[k]; w[9 + k] = ui[k]; }
                        tm_st16(tmem + LINK_STRIDE * d, w);
                        tm_st2(tmem + LINK_STRIDE * d + 16, w + 16);
                    }
                    tm_wait_st();
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[slot]);
                it++;
            }

            // ---- the sweep, software-pipelined over (slice, direction): the neighbour spinor and the link of the NEXT
            //      direction are on their way (LDS / tcgen05.ld) while the current one is multiplied; the hand-off of a
            //      slice's result to the epilogue warp completes under the first direction of the next slice ----
            // processing order d = 0..7 -> link index lk[d] (0-3 forward mu, 4-7 backward mu): x+ x- y+ y- z+ z- t+ t-
            constexpr int lk[8] = {0, 4, 1, 5, 2, 6, 3, 7};
            c2 vb[2][12];
            float lw[2][18];
            unsigned slot = it % RING;
            mbar_wait(&full[slot], (it / RING) & 1);
            const unsigned char *sb = smem5 + slot * SLOT;
            Ld<P>::template chunks<12, false>(reinterpret_cast<const V *>(sb + off[lk[0]]), 1.f, vb[0]);
            tm_ld16(tmem + LINK_STRIDE * lk[0], lw[0]);
            tm_ld2(tmem + LINK_STRIDE * lk[0] + 16, lw[0] + 16);
            int pending = -1;                                                       // history slot whose hand-off is not finished yet
#define MDWF_HANDOFF()                                                                                  \
    do {                                                                                                \
        if (pending >= 0) {                                                                             \
            tm_wait_st();                                                                               \
            tm_fence_before();                                                                          \
            __syncwarp();                                                                               \
            if (lane == 0) mbar_arrive(&hfull[warp * HIST_SLOTS + pending]);                            \
            pending = -1;                                                                               \
        }                                                                                               \
    } while (0)
#define MDWF_DIR5(MU, FWD, TD, d, bs)                                                                   \
    do {                                                                                                \
        constexpr int SGN = ((FWD) ? 1 : -1) * (DAG ? -1 : 1);                                          \
        constexpr int cb_ = (d) & 1, nb_ = cb_ ^ 1;                                                     \
        if ((d) < 7) {                                                                                  \
            Ld<P>::template chunks<12, false>(reinterpret_cast<const V *>(sb + off[lk[((d) + 1) & 7]]), 1.f, vb[nb_]); \
        } else {                                                                                        \
            __syncwarp();                                                                               \
            if (lane == 0) mbar_arrive(&empty[slot]);           /* every load of this ring item has been issued */ \
            it++;                                                                                       \
            if (s + 1 < L5) {                                                                           \
                slot = it % RING;                                                                       \
                mbar_wait(&full[slot], (it / RING) & 1);                                                \
                sb = smem5 + slot * SLOT;                                                               \
                Ld<P>::template chunks<12, false>(reinterpret_cast<const V *>(sb + off[lk[0]]), 1.f, vb[nb_]); \
            }                                                                                           \
        }                                                                                               \
        tm_wait_ld18(lw[cb_]);                                                                          \
        if ((d) < 7 || s + 1 < L5) {                                                                    \
            tm_ld16(tmem + LINK_STRIDE * lk[((d) + 1) & 7], lw[nb_]);                                   \
            tm_ld2(tmem + LINK_STRIDE * lk[((d) + 1) & 7] + 16, lw[nb_] + 16);                          \
        }                                                                                               \
        Link U;                                                                                         \
        _Pragma("unroll") for (int k = 0; k < 9; k++) { U.re[k] = lw[cb_][k]; U.im[k] = lw[cb_][9 + k]; } \
        c2 h[6], chi[6];                                                                                \
        project3<MU, SGN>(vb[cb_], h);                                                                  \
        su3_mul3(U, h, chi);                                                                            \
        recon3<MU, SGN, TD>(chi, bs, acc);                                                              \
    } while (0)
            for (int s = 0; s < L5; s++) {
                c2 acc[12];
#pragma unroll
                for (int q = 0; q < 12; q++) acc[q] = mk(0.f, 0.f);
                MDWF_DIR5(0, true, false, 0, 1.f);
                MDWF_HANDOFF();
                MDWF_DIR5(0, false, false, 1, 1.f);
                MDWF_DIR5(1, true, false, 2, 1.f);
                MDWF_DIR5(1, false, false, 3, 1.f);
                MDWF_DIR5(2, true, false, 4, 1.f);
                MDWF_DIR5(2, false, false, 5, 1.f);
                MDWF_DIR5(3, true, true, 6, btp);
                MDWF_DIR5(3, false, true, 7, btm);
                // ---- raw hop result of the slice -> TMEM history slot, handed to the epilogue warp of the same lanes ----
                const unsigned hs = hit % NS, hph = (hit / NS) & 1;
                mbar_wait(&hempty[warp * HIST_SLOTS + hs], hph ^ 1);
                tm_fence_after();
                hist_store(tmem + HIST_COL0 + 24 * hs, acc);
                pending = (int)hs;
                hit++;
            }
            MDWF_HANDOFF();
#undef MDWF_DIR5
#undef MDWF_HANDOFF
        }
    } else if (warp < 8) {
        // ================= epilogue warps: fifth-dimension POST, own-site term, store, fused norm =================
        const int w = warp - 4;
        const int pa = w & 1, pb = w >> 1;
        unsigned hit = 0;
        const float coef = (float)a.coef_hop;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const Tile T = tile_of(a, tile);
            const long g = group_of(a, T.yy, T.z0 + pa, T.t0 + pb);
            const long cb = g * 32 + lane;
            double nsum = 0.0;
            if (POST == 0) {
                // out_s = coef x_s + own term; OWN = 2: (own_d + own_o Lambda) psi: upper from s-1, lower from s+1 (-m_f at the wrap)
                const V *ob = reinterpret_cast<const V *>(a.own) + g * (long)(L5 * NV * 32) + lane;
                constexpr int NB = 3;                                               // own slices in flight (registers): s .. s+2
                c2 ow[NB][12], pu[6], first_lo[6];
                const c2 d2 = dup((float)a.own_d), o2 = dup((float)a.own_o), ow2 = dup((float)(-a.mf * a.own_o)), cf = dup(coef);
                if (OWN == 2) Ld<P>::template chunks<6>(ob + (L5 - 1) * NV * 32, 1.f, pu);   // upper half of the last slice (wrap of s = 0)
                if (OWN != 0) {
#pragma unroll
                    for (int k = 0; k < NB - 1; k++) Ld<P>::template chunks<12>(ob + k * NV * 32, 1.f, ow[k]);
                }
#pragma unroll
                for (int s = 0; s < L5; s++) {
                    if (OWN != 0 && s + NB - 1 < L5) Ld<P>::template chunks<12>(ob + (s + NB - 1) * NV * 32, 1.f, ow[(s + NB - 1) % NB]);
                    const c2 *cur = ow[s % NB], *nxt = ow[(s + 1) % NB];
                    if (OWN == 2 && s == 0) {
#pragma unroll
                        for (int q = 0; q < 6; q++) first_lo[q] = cur[6 + q];
                    }
                    const unsigned hs = hit % NS, hph = (hit / NS) & 1;
                    mbar_wait(&hfull[w * HIST_SLOTS + hs], hph);
                    tm_fence_after();
                    c2 x[12], o[12];
                    hist_load(tmem + HIST_COL0 + 24 * hs, x);
                    tm_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&hempty[w * HIST_SLOTS + hs]);
                    hit++;
                    if (OWN == 0) {
#pragma unroll
                        for (int q = 0; q < 12; q++) o[q] = mul2(cf, x[q]);
                    } else if (OWN == 1) {
#pragma unroll
                        for (int q = 0; q < 12; q++) o[q] = fma2(cf, x[q], cur[q]);
                    } else {
                        const c2 fu = (s == 0) ? ow2 : o2, fl = (s == L5 - 1) ? ow2 : o2;
#pragma unroll
                        for (int q = 0; q < 6; q++) {
                            const c2 lo = (s == L5 - 1) ? first_lo[q] : nxt[6 + q];
                            o[q] = fma2(cf, x[q], fma2(d2, cur[q], mul2(fu, pu[q])));
                            o[6 + q] = fma2(cf, x[6 + q], fma2(d2, cur[6 + q], mul2(fl, lo)));
                        }
#pragma unroll
                        for (int q = 0; q < 6; q++) pu[q] = cur[q];
                    }
                    nsum += (double)store3<P>(a.out, a.out_norm, L5, s, cb, o, a.partial != nullptr);
                }
            }
            if (POST == 1) {
                // coef (B A^{-1}) x per chirality (DAG: the transposed pattern), two first-order recurrences over the slice
                // history in TMEM.  "direct" half (upper spins; lower for the dagger): z_s = x_s - kappa z_{s-1}, W = z_{L5-1};
                // "mirrored" half: z_s = x_s - kappa z_{s+1}, W = z_0;  t_s = bz z_s + cz z_{s -+ 1} + qW W  (hop3_kernels.cuh).
                // Pass A runs as the slices arrive (ascending): direct recurrence, partial result written back in place, and
                // the mirrored wall term W = sum_s (-kappa)^s x_s.  Pass B (descending) finishes both halves and stores.
                constexpr int DOFF = DAG ? 12 : 0, MOFF = DAG ? 0 : 12;               // word offsets of the direct / mirrored half
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
                        const c2 z = fma2(nk, zp[q], x[DOFF / 2 + q]);                  // z_s = x_s - kappa z_{s-1}
                        const c2 t = fma2(cz, zp[q], mul2(bz, z));                      // bz z_s + cz z_{s-1}
                        zp[q] = z;
                        tp[2 * q] = t.x; tp[2 * q + 1] = t.y;
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
                        const c2 z = fma2(nk, zn[q], x[MOFF / 2 + q]);                  // z_s = x_s - kappa z_{s+1}
                        o[MOFF / 2 + q] = fma2(qWm, Wm[q], fma2(cz, zn[q], mul2(bz, z)));
                        zn[q] = z;
                        o[DOFF / 2 + q] = fma2(qWd, zp[q], x[DOFF / 2 + q]);            // zp = z_{L5-1} of the direct half = its W
                    }
                    nsum += (double)store3<P>(a.out, a.out_norm, L5, s, cb, o, a.partial != nullptr);
                }
                hit += L5;
            }
            if (POST == 2) {
                // out_s = coef (post_d + post_o Lambda^dagger) x_s + (own_d + own_o Lambda^dagger) psi_s   (OWN = 3):
                // upper spins take slice s+1, lower spins slice s-1, factor -m_f at the wrap.  Streaming: out_s is finished as
                // soon as x_{s+1} has arrived (s = 1 .. L5-2) and every history slot is freed as soon as the next output has used it;
                // then s = L5-1 and s = 0, which need the other end of the fifth dimension.  The own slices sit in a rotating
                // register window (s-1 .. s+2), each loaded from global memory once.
                static_assert(POST != 2 || OWN == 3, "POST = 2 comes with OWN = 3");
                const V *ob = reinterpret_cast<const V *>(a.own) + g * (long)(L5 * NV * 32) + lane;
                const unsigned h0 = hit;
                const float cf = coef * (float)a.post_d, co = coef * (float)a.post_o, mw = (float)(-a.mf);
                const c2 cd2 = dup(cf), od2 = dup((float)a.own_d);
                constexpr int NB = 4;
                c2 ow[NB][12];
                Ld<P>::template chunks<12>(ob, 1.f, ow[0]);
                Ld<P>::template chunks<12>(ob + NV * 32, 1.f, ow[1]);
                Ld<P>::template chunks<12>(ob + 2 * NV * 32, 1.f, ow[2]);
#define MDWF_HSLOT(s_) ((h0 + (unsigned)(s_)) % NS)
#define MDWF_HWAIT(s_) mbar_wait(&hfull[w * HIST_SLOTS + MDWF_HSLOT(s_)], ((h0 + (unsigned)(s_)) / NS) & 1)
#define MDWF_HFREE(s_)                                                                   \
    do {                                                                                 \
        tm_fence_before();                                                               \
        __syncwarp();                                                                    \
        if (lane == 0) mbar_arrive(&hempty[w * HIST_SLOTS + MDWF_HSLOT(s_)]);            \
    } while (0)
                // one output slice: x_s, the upper half of x_su and the lower half of x_sl from TMEM; own slices from registers
                auto finish = [&](int s, int su, int sl, const c2 *pc, const c2 *pu, const c2 *pl) {
                    const c2 fu = dup(s == L5 - 1 ? mw : 1.f), fl = dup(s == 0 ? mw : 1.f);
                    const c2 cou = mul2(dup(co), fu), col = mul2(dup(co), fl), oou = mul2(dup((float)a.own_o), fu), ool = mul2(dup((float)a.own_o), fl);
                    c2 x[12], o[12];
                    float xu[12], xl[12];
                    hist_load(tmem + HIST_COL0 + 24 * MDWF_HSLOT(s), x);
                    const unsigned tu = tmem + HIST_COL0 + 24 * MDWF_HSLOT(su), tl = tmem + HIST_COL0 + 24 * MDWF_HSLOT(sl) + 12;
                    tm_ld8(tu, xu); tm_ld2(tu + 8, xu + 8); tm_ld2(tu + 10, xu + 10);
                    tm_ld8(tl, xl); tm_ld2(tl + 8, xl + 8); tm_ld2(tl + 10, xl + 10);
                    tm_wait_ld24(xu, xl);
#pragma unroll
                    for (int q = 0; q < 6; q++) {
                        o[q] = fma2(cd2, x[q], fma2(cou, mk(xu[2 * q], xu[2 * q + 1]), fma2(od2, pc[q], mul2(oou, pu[q]))));
                        o[6 + q] = fma2(cd2, x[6 + q], fma2(col, mk(xl[2 * q], xl[2 * q + 1]), fma2(od2, pc[6 + q], mul2(ool, pl[6 + q]))));
                    }
                    nsum += (double)store3<P>(a.out, a.out_norm, L5, s, cb, o, a.partial != nullptr);
                };
                MDWF_HWAIT(0);
                MDWF_HWAIT(1);
                tm_fence_after();
                // So that slots 0 and 1 are not held until the two ends are done (the sweep of the next tile would wait for the
                // whole tail of this one), what they contribute there is parked in 36 tensor-memory columns of this warp's own:
                // out_0 without its x_{L5-1} term, and the upper half of x_0.
                {
                    c2 lastlo[6], o[12], x[12];
                    Ld<P>::template chunks<6>(ob + (L5 - 1) * NV * 32 + 32 * (NV / 2), 1.f, lastlo);   // lower half of psi_{L5-1}
                    float xu[12], pk[12];
                    const unsigned tu = tmem + HIST_COL0 + 24 * MDWF_HSLOT(1);
                    tm_ld8(tu, xu); tm_ld2(tu + 8, xu + 8); tm_ld2(tu + 10, xu + 10);
                    hist_load(tmem + HIST_COL0 + 24 * MDWF_HSLOT(0), x);
                    tm_wait_ld12(xu);
                    const c2 cou = dup(co), oou = dup((float)a.own_o), ool = dup((float)a.own_o * mw);
#pragma unroll
                    for (int q = 0; q < 6; q++) {
                        o[q] = fma2(cd2, x[q], fma2(cou, mk(xu[2 * q], xu[2 * q + 1]), fma2(od2, ow[0][q], mul2(oou, ow[1][q]))));
                        o[6 + q] = fma2(cd2, x[6 + q], fma2(od2, ow[0][6 + q], mul2(ool, lastlo[q])));
                        pk[2 * q] = x[q].x; pk[2 * q + 1] = x[q].y;
                    }
                    hist_store(tmem + PARK0, o);
                    tm_st8(tmem + PARK1, pk);
                    tm_st2(tmem + PARK1 + 8, pk + 8);
                    tm_st2(tmem + PARK1 + 10, pk + 10);
                    tm_wait_st();
                }
                c2 up0[6];                                                          // upper half of psi_0 (own term of out_{L5-1}), read again late
#pragma unroll
                for (int s = 1; s <= L5 - 2; s++) {
                    if (s + 2 <= L5 - 1) Ld<P>::template chunks<12>(ob + (s + 2) * NV * 32, 1.f, ow[(s + 2) % NB]);
                    if (s == L5 - 2) Ld<P>::template chunks<6>(ob, 1.f, up0);
                    MDWF_HWAIT(s + 1);
                    tm_fence_after();
                    finish(s, s + 1, s - 1, ow[s % NB], ow[(s + 1) % NB], ow[(s - 1) % NB]);
                    MDWF_HFREE(s - 1);
                }
                {   // the two ends: out_{L5-1} (upper from the parked x_0, lower from x_{L5-2}) and the rest of out_0
                    const c2 *pc = ow[(L5 - 1) % NB], *pl = ow[(L5 - 2) % NB];
                    c2 o[12], x[12];
                    float xu[12], xl[12];
                    const unsigned tl = tmem + HIST_COL0 + 24 * MDWF_HSLOT(L5 - 2) + 12;
                    tm_ld8(tmem + PARK1, xu); tm_ld2(tmem + PARK1 + 8, xu + 8); tm_ld2(tmem + PARK1 + 10, xu + 10);
                    tm_ld8(tl, xl); tm_ld2(tl + 8, xl + 8); tm_ld2(tl + 10, xl + 10);
                    tm_wait_ld24(xu, xl);
                    hist_load(tmem + HIST_COL0 + 24 * MDWF_HSLOT(L5 - 1), x);
                    const c2 cou = dup(co * mw), col = dup(co), oou = dup((float)a.own_o * mw), ool = dup((float)a.own_o);
#pragma unroll
                    for (int q = 0; q < 6; q++) {
                        o[q] = fma2(cd2, x[q], fma2(cou, mk(xu[2 * q], xu[2 * q + 1]), fma2(od2, pc[q], mul2(oou, up0[q]))));
                        o[6 + q] = fma2(cd2, x[6 + q], fma2(col, mk(xl[2 * q], xl[2 * q + 1]), fma2(od2, pc[6 + q], mul2(ool, pl[6 + q]))));
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
static inline int mdwf_sm_count()
{
    static int sms = 0;
    if (!sms) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) sms = 148;
    }
    return sms;
}
static inline bool hop5_geometry(HopArgs &a)
{
    const int Lxh = a.L[0] >> 1;
    if (!(Lxh == 2 || Lxh == 4 || Lxh == 8 || Lxh == 16)) return false;
    const int R = 32 / Lxh;
    if (a.L[1] % R != 0) return false;
    if (!(a.L5 == 8 || a.L5 == 12)) return false;
    a.t5_NY = a.L[1] / R;
    const int nzp = a.L[2] / 2;
    // z-pairs per chunk: the input planes of a chunk's t-pair (4 t-planes with halo) should stay in L2 until the next t-pair
    int nzq = nzp;
    const long pair_bytes = (long)a.t5_NY * 2 * 2 * a.L5 * 3072 * 3;      // groups of one z-pair x t-pair, 3 streams, fp32
    const long budget = (a.t5_l2mb > 0 ? (long)a.t5_l2mb : 48L) << 20;
    while (nzq > 1 && (nzq % 2 == 0) && nzq * pair_bytes > budget) nzq /= 2;
    a.t5_nzq = nzq;
    a.t5_NT = a.L[3] / 2;
    a.t5_ntiles = a.t5_NY * nzp * a.t5_NT;
    a.t5_dNY = mdwf_fastdiv((unsigned)a.t5_NY);
    a.t5_dnzq = mdwf_fastdiv((unsigned)a.t5_nzq);
    a.t5_dNT = mdwf_fastdiv((unsigned)a.t5_NT);
    return true;
}
template <class P, int DAG, int PRE, int POST, int OWN, int L5>
static int launch_hop5_inst(const HopArgs &a, cudaStream_t st)
{
    static int sms = 0;
    const size_t smem = (size_t)RING * Slot<P>::BYTES + 8 * (2 * RING + 8 * HIST_SLOTS + 4) + 3 * 48 * 12 + 16;
    if (!sms) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        cudaError_t e = cudaFuncSetAttribute(hop5_kernel<P, DAG, PRE, POST, OWN, L5>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) { sms = 0; return (int)e; }
    }
    const int grid = a.t5_ntiles < sms ? a.t5_ntiles : sms;
    hop5_kernel<P, DAG, PRE, POST, OWN, L5><<<grid, 384, smem, st>>>(a);
    return (int)cudaGetLastError();
}
template <class P, int DAG, int PRE, int POST, int OWN>
static int launch_hop5_l5(const HopArgs &a, cudaStream_t st)
{
    if (a.L5 == 12) return launch_hop5_inst<P, DAG, PRE, POST, OWN, 12>(a, st);
#ifndef MDWF_DEV_FAST
    if (a.L5 == 8) return launch_hop5_inst<P, DAG, PRE, POST, OWN, 8>(a, st);
#endif
    return -1;
}
// -1: not covered by the v5 family (the caller falls back to v3)
template <class P>
static int launch_hop5_prec(int dag, int pre, int post, int own, HopArgs a, cudaStream_t st)
{
    if (!hop5_geometry(a)) return -1;
    if (a.kver == 5 && a.t5_ntiles < 8 * mdwf_sm_count()) return -1;     // default (auto): a persistent CTA per SM needs several tiles per SM to pay; "kernels=v5" forces it
    if (!dag && pre == 0 && post == 0 && own == 2) return launch_hop5_l5<P, 0, 0, 0, 2>(a, st);   // K2
    if (!dag && pre == 0 && post == 1 && own == 0) return launch_hop5_l5<P, 0, 0, 1, 0>(a, st);   // K1 reading a precomputed B psi
    if (dag && pre == 0 && post == 1 && own == 0) return launch_hop5_l5<P, 1, 0, 1, 0>(a, st);    // K1^+
    if (dag && pre == 0 && post == 2 && own == 3) return launch_hop5_l5<P, 1, 0, 2, 3>(a, st);    // K2^+
    return -1;
}

}   // namespace h5
