// v3 hop kernels (packed f32x2 arithmetic, recurrence form of B A^{-1}) instantiated for precision PS
#include "hop3_kernels.cuh"
int mdwf_launch_hop3_S(int dag, int pre, int post, int own, const HopArgs &a, cudaStream_t st)
{
    if (!h3::hop3_supports(a.L5, post, a)) return -1;      // caller falls back to the v2 family
    return h3::launch_hop3_prec<PS>(dag, pre, post, own, a, st);
}
