// batched (multi-right-hand-side) v3 hop kernels, 16-bit storage (hop3b_kernels.cuh)
#include "hop3b_kernels.cuh"
int mdwf_launch_hop3_batch_H(int dag, int pre, int post, int own, const HopArgs &a, cudaStream_t st)
{
    return h3::launch_hop3_batch_prec<PH>(dag, pre, post, own, a, st);      // -1: not covered
}
