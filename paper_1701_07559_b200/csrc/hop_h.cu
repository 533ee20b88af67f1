// hop kernels instantiated for precision PH (see hop_kernels.cuh)
#include "hop_kernels.cuh"
int mdwf_launch_hop_H(int dag, int pre, int post, int own, const HopArgs &a, cudaStream_t st)
{
    return launch_hop_prec<PH>(dag, pre, post, own, a, st);
}
int mdwf_launch_sdense_H(int L5, int Vh, const SpinorBuf &in, const SpinorBuf &out, const void *dense, cudaStream_t st)
{
    return launch_sdense_prec<PH>(L5, Vh, in, out, dense, st);
}
