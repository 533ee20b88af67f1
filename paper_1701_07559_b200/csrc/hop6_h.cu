// tile-sweep hop kernels for 16-bit storage (two sweep sets, hop6_kernels.cuh)
#include "hop6_kernels.cuh"
int mdwf_launch_hop6_H(int dag, int pre, int post, int own, const HopArgs &a, cudaStream_t st)
{
    if (post == 1 && !a.r_ok) return -1;
    return h6::launch_hop6(dag, pre, post, own, a, st);     // -1: not covered, the caller falls back to v3
}
