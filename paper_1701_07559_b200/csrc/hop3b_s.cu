// batched (multi-right-hand-side) v3 hop kernels, fp32 storage (hop3b_kernels.cuh)
#include "hop3b_kernels.cuh"
int mdwf_launch_hop3_batch_S(int dag, int pre, int post, int own, const HopArgs &a, cudaStream_t st)
{
    return h3::launch_hop3_batch_prec<PS>(dag, pre, post, own, a, st);      // -1: not covered
}
