// v4 hop kernels (neighbour groups staged in shared memory by bulk-asynchronous copies) for precision PS
#include "hop4_kernels.cuh"
int mdwf_launch_hop4_S(int dag, int pre, int post, int own, const HopArgs &a, cudaStream_t st)
{
    if (!h4::hop4_supports(a, post)) return -1;      // caller falls back to the v3 family
    return h4::launch_hop4_prec<PS>(dag, pre, post, own, a, st);
}
