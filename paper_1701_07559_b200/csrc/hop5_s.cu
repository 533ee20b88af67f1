// v5 tile-sweep hop kernels (TMA ring, TMEM links and slice history, warp-specialised) instantiated for precision PS
#include "hop5_kernels.cuh"
int mdwf_launch_hop5_S(int dag, int pre, int post, int own, const HopArgs &a, cudaStream_t st)
{
    if (post == 1 && !a.r_ok) return -1;
    return h5::launch_hop5_prec<PS>(dag, pre, post, own, a, st);     // -1: not covered, the caller falls back to v3
}
