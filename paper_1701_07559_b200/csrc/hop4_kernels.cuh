// hop4_kernels.cuh -- v4 of the fused hop kernels for fp32 arithmetic: the neighbour spinors are STAGED IN SHARED
// MEMORY BY BULK-ASYNCHRONOUS COPIES (cp.async.bulk + mbarrier, the TMA engine), one whole 32-site group (all L5
// slices: L5 * NV * 512 B contiguous in the warp-blob layout) per stage, two stages in flight per block.
//
// Why: ncu on the v3 kernels (profiles/r01_v3_hop_kernels_ncu.md) shows every warp stalling once per direction on
// its first global load, with no unit saturated; registers (236-254) leave no room for a second direction in
// flight.  Here loads hold no registers at all: while the block multiplies direction d out of one shared-memory
// buffer, the copy engine fills the other with the group of direction d+1.
//
// Geometry (requires Lx = 32, i.e. 16 checkerboard sites per x-row, so that a 32-site group is the two rows
// y0, y0+1 of one (z,t)): the 32 neighbours of the block are
//   x+-      : the block's own group index g on the other parity (lane permuted inside the group),
//   z+-, t+- : one other group each, same lane,
//   y+-      : rows y0+1 / y0 are in g again (pass Y1: lanes 0-15 hop forward, lanes 16-31 hop backward, both
//              reading lane ^ 16 of g); rows y0+2 / y0-1 are half of the groups g+1 / g-1 (passes Y2A, Y2B, each
//              with half of the lanes masked -- 1/8 more issue slots, which these kernels have to spare).
// Stage order g, z+, z-, t+, t-, y+, y- : 7 bulk copies of L5*NV*512 B per block, each consumed by 1-3 passes.
// The B-on-load halo slices (PRE = 1) come out of the same staged group for free.
#pragma once
#include "hop3_kernels.cuh"

namespace h4 {
using namespace h3;

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
        asm volatile("{\n\t.reg .pred P1;\n\tmbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2;\n\tselp.u32 %0, 1, 0, P1;\n\t}"
                     : "=r"(ok)
                     : "r"(addr), "r"(phase)
                     : "memory");
    }
}
MDWF_DEV void bulk_g2s(void *dst_smem, const void *src_gmem, unsigned bytes, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
MDWF_DEV void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ---- chunk loads from the staged group -----------------------------------------------------------------
template <class P> struct Ls;
template <> struct Ls<PS> {
    template <int NC> static MDWF_DEV void chunks(const float4 *p, float, c2 *v)      // p: chunk 0 of this lane, stride 32
    {
#pragma unroll
        for (int j = 0; j < NC / 2; j++) {
            const float4 q = p[32 * j];
            v[2 * j] = mk(q.x, q.y);
            v[2 * j + 1] = mk(q.z, q.w);
        }
    }
};
template <> struct Ls<PH> {
    template <int NC> static MDWF_DEV void chunks(const short4 *p, float norm, c2 *v)
    {
        const c2 s2 = dup(norm * (1.0f / MDWF_FIXED_MAX));
#pragma unroll
        for (int j = 0; j < NC / 2; j++) {
            const uint2 q = reinterpret_cast<const uint2 *>(p)[32 * j];
            v[2 * j] = cvt_pair(q.x, s2);
            v[2 * j + 1] = cvt_pair(q.y, s2);
        }
    }
};

// projection / reconstruction with a RUN-TIME sign S (= +-1) and weight p (= boundary sign, or 0 for a masked lane)
template <int MU>
MDWF_DEV void project4(float S, const c2 *v, c2 *h)
{
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
template <int MU>
MDWF_DEV void recon4(float S0, float p, const c2 *chi, c2 *acc)
{
    const float S = S0 * p;
    const c2 pp = mk(p, p), mp = mk(-S, S), pm = mk(S, -S), ss = mk(S, S), mm = mk(-S, -S);
#pragma unroll
    for (int c = 0; c < 3; c++) {
        acc[c] = fma2(chi[c], pp, acc[c]);
        acc[3 + c] = fma2(chi[3 + c], pp, acc[3 + c]);
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

// One pass over the S slices of this thread out of a staged group.
//   buf / nrm : staged group (chunk (s, j) of lane l at buf[(s*NV + j)*32 + l], scale at nrm[s*32 + l])
//   ln        : lane of this thread's neighbour inside the group
//   sl        : this thread's link for this pass (shared-memory link table)
//   SG        : sign of the gamma_mu term, (fwd ? 1 : -1) * (DAG ? -1 : 1);  p: boundary sign, 0 = lane masked
template <class P, int MU, int PRE, int L5, int S>
MDWF_DEV void hop_pass4(const HopArgs &a, int s0, const typename P::V *buf, const float *nrm, int ln, const float2 *sl,
                        float SG, float p, c2 (*acc)[12])
{
    using V = typename P::V;
    constexpr int NV = P::NV;
    Link U;
    load_link3(sl, U);
    const V *p0 = buf + (s0 * NV) * 32 + ln;
    if (PRE == 0) {
#pragma unroll
        for (int k = 0; k < S; k++) {
            c2 v[12], h[6], chi[6];
            Ls<P>::template chunks<12>(p0 + k * NV * 32, P::HALF ? nrm[(s0 + k) * 32 + ln] : 1.f, v);
            project4<MU>(SG, v, h);
            su3_mul3(U, h, chi);
            recon4<MU>(SG, p, chi, acc[k]);
        }
    } else {
        const float f = (float)(a.pre_o / a.pre_d), fw = (float)(-a.mf * a.pre_o / a.pre_d);
        const int sm = (s0 == 0) ? L5 - 1 : s0 - 1;
        const int sp = (s0 + S >= L5) ? 0 : s0 + S;
        c2 prev_up[6], cur[12], nxt[12];
        Ls<P>::template chunks<6>(buf + (sm * NV) * 32 + ln, P::HALF ? nrm[sm * 32 + ln] : 1.f, prev_up);
        Ls<P>::template chunks<12>(p0, P::HALF ? nrm[s0 * 32 + ln] : 1.f, cur);
#pragma unroll
        for (int k = 0; k < S; k++) {
            if (k < S - 1) Ls<P>::template chunks<12>(p0 + (k + 1) * NV * 32, P::HALF ? nrm[(s0 + k + 1) * 32 + ln] : 1.f, nxt);
            else Ls<P>::template chunks<6>(buf + (sp * NV + NV / 2) * 32 + ln, P::HALF ? nrm[sp * 32 + ln] : 1.f, nxt + 6);
            const c2 fu = dup((s0 + k == 0) ? fw : f);
            const c2 fl = dup((s0 + k == L5 - 1) ? fw : f);
            c2 w[12], h[6], chi[6];
#pragma unroll
            for (int q = 0; q < 6; q++) {
                w[q] = fma2(fu, prev_up[q], cur[q]);
                w[6 + q] = fma2(fl, nxt[6 + q], cur[6 + q]);
            }
            project4<MU>(SG, w, h);
            su3_mul3(U, h, chi);
            recon4<MU>(SG, p, chi, acc[k]);
#pragma unroll
            for (int q = 0; q < 6; q++) prev_up[q] = cur[q];
            if (k < S - 1) {
#pragma unroll
                for (int q = 0; q < 12; q++) cur[q] = nxt[q];
            }
        }
    }
}

template <class P, int DAG, int PRE, int POST, int OWN, int L5, int S>
__global__ void __launch_bounds__(32 * (L5 / S), 2) hop4_kernel(const HopArgs a)
{
    constexpr int NSG = L5 / S, NV = P::NV;
    using V = typename P::V;
    constexpr unsigned BUF_BYTES = L5 * NV * 32 * sizeof(V);          // one staged group
    constexpr unsigned NRM_BYTES = P::HALF ? L5 * 32 * sizeof(float) : 0;
    extern __shared__ __align__(128) unsigned char smem_raw4[];
    V *buf[2] = {reinterpret_cast<V *>(smem_raw4), reinterpret_cast<V *>(smem_raw4 + BUF_BYTES)};
    float *nrm[2] = {reinterpret_cast<float *>(smem_raw4 + 2 * BUF_BYTES),
                     reinterpret_cast<float *>(smem_raw4 + 2 * BUF_BYTES + NRM_BYTES)};
    unsigned char *rest = smem_raw4 + 2 * BUF_BYTES + 2 * NRM_BYTES;
    c2 *sE = reinterpret_cast<c2 *>(rest);                                                  // [NSG][12][32] (POST != 0)
    float2 *sL = reinterpret_cast<float2 *>(rest + (POST != 0 ? NSG * 12 * 32 * sizeof(c2) : 0));   // [8][9][32] links
    unsigned long long *bar = reinterpret_cast<unsigned long long *>(
        rest + (POST != 0 ? NSG * 12 * 32 * sizeof(c2) : 0) + 8 * 9 * 32 * sizeof(float2));  // [2] mbarriers

    const int lane = threadIdx.x, sg = threadIdx.y, s0 = sg * S;
    const bool leader = (lane == 0 && sg == 0);
    long cb0 = (long)blockIdx.x * 32;
    if (a.sweep_nb) {                                    // z-chunked t sweep, see hop_kernels.cuh
        const int Lt = a.L[3];
        const int per_chunk = a.sweep_nb * Lt;
        const int c = blockIdx.x / per_chunk, r = blockIdx.x - c * per_chunk;
        const int t = r / a.sweep_nb, q = r - t * a.sweep_nb;
        cb0 = (long)t * ((long)a.Vh / Lt) + (long)c * a.sweep_chunk + (long)q * 32;
    }
    const long cb = cb0 + lane;

    // coordinates of the block (all 32 sites share z, t; rows y0 = even, y0 + 1) and of this lane
    constexpr int Lxh = 16;
    const int Ly = a.L[1], Lz = a.L[2], Lt = a.L[3];
    int r = (int)cb;
    const int xh = r % Lxh; r /= Lxh;
    const int y = r % Ly;   r /= Ly;
    const int z = r % Lz;
    const int t = r / Lz;
    const int y0 = y & ~1;
    const int xodd = (a.parity_out + y + z + t) & 1;
    const long sz = (long)Lxh * Ly, st = (long)Lxh * Ly * Lz;
    // first site of the group staged in each stage: g, z+, z-, t+, t-, y+ (rows y0+2, y0+3), y- (rows y0-2, y0-1)
    long gs[7];
    gs[0] = cb0;
    gs[1] = (z == Lz - 1) ? cb0 - (Lz - 1) * sz : cb0 + sz;
    gs[2] = (z == 0) ? cb0 + (Lz - 1) * sz : cb0 - sz;
    gs[3] = (t == Lt - 1) ? cb0 - (Lt - 1) * st : cb0 + st;
    gs[4] = (t == 0) ? cb0 + (Lt - 1) * st : cb0 - st;
    gs[5] = (y0 + 2 == Ly) ? cb0 - (long)(Ly - 2) * Lxh : cb0 + 32;
    gs[6] = (y0 == 0) ? cb0 + (long)(Ly - 2) * Lxh : cb0 - 32;
    const float btp = (t == Lt - 1) ? -1.f : 1.f;               // antiperiodic in t
    const float btm = (t == 0) ? -1.f : 1.f;

    auto issue = [&](int stage) {                                // leader only: start the bulk copy of one stage
        const int b = stage & 1;
        mbar_expect_tx(&bar[b], BUF_BYTES + NRM_BYTES);
        bulk_g2s(buf[b], reinterpret_cast<const V *>(a.in) + (gs[stage] >> 5) * (long)(L5 * NV * 32), BUF_BYTES, &bar[b]);
        if (P::HALF) bulk_g2s(nrm[b], a.in_norm + (gs[stage] >> 5) * (long)(L5 * 32), NRM_BYTES, &bar[b]);
    };
    if (leader) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_proxy_async();
        issue(0);
        issue(1);
    }

    c2 acc[S][12];
#pragma unroll
    for (int k = 0; k < S; k++)
#pragma unroll
        for (int q = 0; q < 12; q++) acc[k][q] = mk(0.f, 0.f);

    // neighbour lanes inside the own group (x hops) and the sites whose links the backward hops need
    const long cb_xp = xodd ? (xh == Lxh - 1 ? cb - (Lxh - 1) : cb + 1) : cb;
    const long cb_xm = xodd ? cb : (xh == 0 ? cb + (Lxh - 1) : cb - 1);
    const long cb_ym = (y == 0) ? cb + (long)(Ly - 1) * Lxh : cb - Lxh;
    const long cb_zm = gs[2] + lane, cb_tm = gs[4] + lane;
    // the 8 links of the block's 32 sites, built once (hop3_kernels.cuh): warp d mod NSG builds direction d
#pragma unroll
    for (int d = 0; d < 8; d++)
        if ((d % NSG) == sg) {
            if ((d & 1) == 0) stage_link<P, false>(a.gauge_same, d >> 1, cb, a.recon, sL + d * 288 + lane);
            else stage_link<P, true>(a.gauge_other, d >> 1, d == 1 ? cb_xm : (d == 3 ? cb_ym : (d == 5 ? cb_zm : cb_tm)), a.recon,
                                     sL + d * 288 + lane);
        }
    __syncthreads();                                             // links and barrier initialisation visible

    constexpr float SF = DAG ? -1.f : 1.f, SB = DAG ? 1.f : -1.f;       // sign of the gamma term: forward / backward hop
    const bool lo = lane < 16;                                   // row y0 (lanes 0-15) or y0 + 1 (lanes 16-31)
#pragma unroll
    for (int stage = 0; stage < 7; stage++) {
        const int b = stage & 1;
        mbar_wait(&bar[b], (stage >> 1) & 1);
        const V *B = buf[b];
        const float *N = nrm[b];
        if (stage == 0) {
            hop_pass4<P, 0, PRE, L5, S>(a, s0, B, N, (int)(cb_xp - cb0), sL + 0 * 288 + lane, SF, 1.f, acc);
            hop_pass4<P, 0, PRE, L5, S>(a, s0, B, N, (int)(cb_xm - cb0), sL + 1 * 288 + lane, SB, 1.f, acc);
            // Y1: row y0 hops forward to row y0+1, row y0+1 hops backward to row y0: both are lane ^ 16 of g
            hop_pass4<P, 1, PRE, L5, S>(a, s0, B, N, lane ^ 16, sL + (lo ? 2 : 3) * 288 + lane, lo ? SF : SB, 1.f, acc);
        } else if (stage == 1) {
            hop_pass4<P, 2, PRE, L5, S>(a, s0, B, N, lane, sL + 4 * 288 + lane, SF, 1.f, acc);
        } else if (stage == 2) {
            hop_pass4<P, 2, PRE, L5, S>(a, s0, B, N, lane, sL + 5 * 288 + lane, SB, 1.f, acc);
        } else if (stage == 3) {
            hop_pass4<P, 3, PRE, L5, S>(a, s0, B, N, lane, sL + 6 * 288 + lane, SF, btp, acc);
        } else if (stage == 4) {
            hop_pass4<P, 3, PRE, L5, S>(a, s0, B, N, lane, sL + 7 * 288 + lane, SB, btm, acc);
        } else if (stage == 5) {
            // Y2A: row y0+1 hops forward to row y0+2 = lanes 0-15 of the next group; row y0 is masked
            hop_pass4<P, 1, PRE, L5, S>(a, s0, B, N, lane ^ 16, sL + 2 * 288 + lane, SF, lo ? 0.f : 1.f, acc);
        } else {
            // Y2B: row y0 hops backward to row y0-1 = lanes 16-31 of the previous group; row y0+1 is masked
            hop_pass4<P, 1, PRE, L5, S>(a, s0, B, N, lane ^ 16, sL + 3 * 288 + lane, SB, lo ? 1.f : 0.f, acc);
        }
        if (stage + 2 < 7) {
            __syncthreads();                                     // every warp is done reading buf[b]
            if (leader) {
                fence_proxy_async();
                issue(stage + 2);
            }
        }
    }
    epilogue3<P, DAG, POST, OWN, L5, S>(a, acc, sE, lane, sg, s0, cb, true);
}

// ---- launchers ----------------------------------------------------------------------------------
template <class P, int DAG, int PRE, int POST, int OWN, int L5, int S>
static int launch_hop4_inst(const HopArgs &a, cudaStream_t st)
{
    constexpr int NSG = L5 / S;
    using V = typename P::V;
    dim3 block(32, NSG);
    dim3 grid((unsigned)(a.Vh / 32));
    const size_t smem = 2 * (size_t)L5 * P::NV * 32 * sizeof(V) + (P::HALF ? 2 * (size_t)L5 * 32 * sizeof(float) : 0) +
                        ((POST != 0) ? (size_t)NSG * 12 * 32 * sizeof(c2) : 0) + (size_t)8 * 9 * 32 * sizeof(float2) + 16;
    cudaError_t e = cudaFuncSetAttribute(hop4_kernel<P, DAG, PRE, POST, OWN, L5, S>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return (int)e;
    hop4_kernel<P, DAG, PRE, POST, OWN, L5, S><<<grid, block, smem, st>>>(a);
    return (int)cudaGetLastError();
}
template <class P, int DAG, int PRE, int POST, int OWN>
static int launch_hop4_l5(const HopArgs &a, cudaStream_t st)
{
    if (a.L5 == 12) return launch_hop4_inst<P, DAG, PRE, POST, OWN, 12, 3>(a, st);
#ifndef MDWF_DEV_FAST
    if (a.L5 == 8) return launch_hop4_inst<P, DAG, PRE, POST, OWN, 8, 2>(a, st);
#endif
    return (int)cudaErrorInvalidValue;
}
// the staged family covers Lx = 32 (two x-rows per 32-site group), L5 in {8, 12}, and the recurrence form of B A^-1
static inline bool hop4_supports(const HopArgs &a, int post)
{
    if (a.L[0] != 32 || (a.L[1] & 1) || a.Vh % 32 != 0) return false;
    if (!(a.L5 == 8 || a.L5 == 12)) return false;
    if (post == 1 && !a.r_ok) return false;
    return true;
}
template <class P>
static int launch_hop4_prec(int dag, int pre, int post, int own, const HopArgs &a, cudaStream_t st)
{
    if (!dag && pre == 1 && post == 1 && own == 0) return launch_hop4_l5<P, 0, 1, 1, 0>(a, st);   // K1
    if (!dag && pre == 0 && post == 1 && own == 0) return launch_hop4_l5<P, 0, 0, 1, 0>(a, st);   // K1 reading a precomputed B psi
    if (!dag && pre == 0 && post == 0 && own == 2) return launch_hop4_l5<P, 0, 0, 0, 2>(a, st);   // K2
    if (!dag && pre == 1 && post == 0 && own == 2) return launch_hop4_l5<P, 0, 1, 0, 2>(a, st);   // D
    if (!dag && pre == 1 && post == 0 && own == 1) return launch_hop4_l5<P, 0, 1, 0, 1>(a, st);   // Schur prep/recon
    if (dag && pre == 0 && post == 1 && own == 0) return launch_hop4_l5<P, 1, 0, 1, 0>(a, st);    // K1^+
    if (dag && pre == 0 && post == 2 && own == 3) return launch_hop4_l5<P, 1, 0, 2, 3>(a, st);    // K2^+, D^+
    return (int)cudaErrorInvalidValue;
}

}   // namespace h4
