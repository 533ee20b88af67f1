// hop3b_kernels.cuh -- NEXT-2 ("propagators": 12 spin-colour columns per source): the fused hop
// kernels of hop3_kernels.cuh applied to a BATCH of right-hand sides in one launch.
//
// A block still owns one 32-site group.  Its link tile (8 directions, 12- or 18-real, by one TMA bulk copy) is brought into shared
// memory and completed (row 2, 16-bit conversion) ONCE and then serves all nrhs vectors: the links and their reconstruction are
// amortised over nrhs x L5 slices instead of L5, and nrhs applications cost one launch.  The arithmetic per right-hand side is
// the code of the single-vector kernel (hop_dir3, epilogue3), so a batched application is bit-identical to nrhs single ones.
//
// Batch layout: the nrhs parity vectors are one spinor array over nrhs * Vp sites (Vp = Vh rounded up to 32): right-hand side r
// occupies the site indices [r Vp, (r + 1) Vp).  The device functions address spinors by site index, so the batch kernel only
// shifts the indices it hands them (a.batch_sites = Vp).
#pragma once
#include "hop3_kernels.cuh"

namespace h3 {

template <class P, int DAG, int PRE, int POST, int OWN, int L5, int S>
__global__ void __launch_bounds__(32 * (L5 / S), Hop3Cfg<P, S>::WARPS / (L5 / S) > 0 ? Hop3Cfg<P, S>::WARPS / (L5 / S) : 1)
hop3_batch_kernel(const HopArgs a)
{
    constexpr int NSG = L5 / S, NV = P::NV;
    using V = typename P::V;
    using G = typename P::G;
    constexpr unsigned SE_BYTES = (POST != 0) ? NSG * 12 * 32 * sizeof(c2) : 0;
    constexpr unsigned SL_BYTES = 8 * 9 * 32 * sizeof(float2);
    constexpr unsigned SR_BYTES = P::HALF ? 8 * 9 * 32 * sizeof(short2) : 0;
    extern __shared__ __align__(128) unsigned char smem_raw3b[];
    c2 *sE = reinterpret_cast<c2 *>(smem_raw3b);                               // [NSG][12][32] carries / halo slices (POST != 0)
    float2 *sL = reinterpret_cast<float2 *>(smem_raw3b + SE_BYTES);            // [8][9][32] link table
    unsigned char *sR = smem_raw3b + SE_BYTES + SL_BYTES;                      // 16-bit storage: the raw link tile
    unsigned long long *bar = reinterpret_cast<unsigned long long *>(sR + SR_BYTES);
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

    // ---- the link tile of the block's 32 sites: once for the whole batch ----
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
    }
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
    const V *gin = reinterpret_cast<const V *>(a.in);
    const int sm = (s0 == 0) ? L5 - 1 : s0 - 1, sp = (s0 + S >= L5) ? 0 : s0 + S;

    __syncthreads();                                             // barrier initialisation visible to every thread
    mbar_wait(&bar[0], 0);
#pragma unroll
    for (int d = 0; d < 8; d++)
        if ((d % NSG) == sg) expand_link<P>(sR, sL, d, lane, a.recon);
    __syncthreads();

    // ---- the right-hand sides, one after the other, on the staged links ----
#pragma unroll 1
    for (int r = 0; r < a.nrhs; r++) {
        const long roff = (long)r * a.batch_sites;               // site-index shift of right-hand side r
        c2 acc[S][12];
#pragma unroll
        for (int k = 0; k < S; k++)
#pragma unroll
            for (int q = 0; q < 12; q++) acc[k][q] = mk(0.f, 0.f);
        if (active) {
#define MDWF_GDIRB(MU, FWD, TD, d, bs) \
            hop_dir3<P, MU, FWD, DAG, PRE, S, TD>(a, L5, s0, sL + (d) * 288 + lane, \
                SrcMem<P, S, true>{gin + sp_off(L5, NV, nb[d] + roff, 0), a.in_norm + sp_noff(L5, nb[d] + roff, 0), s0, sm, sp}, bs, acc)
            MDWF_GDIRB(0, true, false, 0, 1.f);
            MDWF_GDIRB(0, false, false, 4, 1.f);
            MDWF_GDIRB(1, true, false, 1, 1.f);
            MDWF_GDIRB(1, false, false, 5, 1.f);
            MDWF_GDIRB(2, true, false, 2, 1.f);
            MDWF_GDIRB(2, false, false, 6, 1.f);
            MDWF_GDIRB(3, true, true, 3, btp);
            MDWF_GDIRB(3, false, true, 7, btm);
#undef MDWF_GDIRB
        }
        epilogue3<P, DAG, POST, OWN, L5, S>(a, acc, sE, lane, sg, s0, cb + roff, active, (int)(blockIdx.x + r * gridDim.x));
        __syncthreads();                                         // the epilogue's shared-memory carries are reused by the next right-hand side
    }
}

template <class P, int DAG, int PRE, int POST, int OWN, int L5, int S>
static int launch_hop3_batch_inst(const HopArgs &a, cudaStream_t st)
{
    constexpr int NSG = L5 / S;
    dim3 block(32, NSG);
    dim3 grid((unsigned)((a.Vh + 31) / 32));
    const size_t smem = ((POST != 0) ? (size_t)NSG * 12 * 32 * sizeof(c2) : 0) + (size_t)8 * 9 * 32 * sizeof(float2) +
                        (P::HALF ? (size_t)8 * 9 * 32 * sizeof(short2) : 0) + 8;
    static bool attr_set = false;
    if (smem > 32 * 1024 && !attr_set) {
        cudaError_t e = cudaFuncSetAttribute(hop3_batch_kernel<P, DAG, PRE, POST, OWN, L5, S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return (int)e;
        attr_set = true;
    }
    hop3_batch_kernel<P, DAG, PRE, POST, OWN, L5, S><<<grid, block, smem, st>>>(a);
    return (int)cudaGetLastError();
}
template <class P, int DAG, int PRE, int POST, int OWN>
static int launch_hop3_batch_l5(const HopArgs &a, cudaStream_t st)
{
    if (a.L5 == 12) return launch_hop3_batch_inst<P, DAG, PRE, POST, OWN, 12, MDWF_H3_S12>(a, st);
    if (a.L5 == 8) return launch_hop3_batch_inst<P, DAG, PRE, POST, OWN, 8, 2>(a, st);
    if (a.L5 == 16) return launch_hop3_batch_inst<P, DAG, PRE, POST, OWN, 16, 2>(a, st);
    return -1;
}
// the four kernels of Mpc and Mpc^dagger; -1: not covered (other L5, |kappa| >= 0.98, other variants)
template <class P>
static int launch_hop3_batch_prec(int dag, int pre, int post, int own, const HopArgs &a, cudaStream_t st)
{
    if (!hop3_supports(a.L5, post, a) || a.nrhs < 1) return -1;
    if (!dag && pre == 1 && post == 1 && own == 0) return launch_hop3_batch_l5<P, 0, 1, 1, 0>(a, st);   // K1
    if (!dag && pre == 0 && post == 0 && own == 2) return launch_hop3_batch_l5<P, 0, 0, 0, 2>(a, st);   // K2
    if (dag && pre == 0 && post == 1 && own == 0) return launch_hop3_batch_l5<P, 1, 0, 1, 0>(a, st);    // K1^+
    if (dag && pre == 0 && post == 2 && own == 3) return launch_hop3_batch_l5<P, 1, 0, 2, 3>(a, st);    // K2^+
    return -1;
}

}   // namespace h3
