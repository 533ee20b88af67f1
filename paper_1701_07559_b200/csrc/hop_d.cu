// hop kernels instantiated for precision PD (see hop_kernels.cuh)
#include "hop_kernels.cuh"
int mdwf_launch_hop_D(int dag, int pre, int post, int own, const HopArgs &a, cudaStream_t st)
{
    return launch_hop_prec<PD>(dag, pre, post, own, a, st);
}
int mdwf_launch_sdense_D(int L5, int Vh, const SpinorBuf &in, const SpinorBuf &out, const void *dense, cudaStream_t st)
{
    return launch_sdense_prec<PD>(L5, Vh, in, out, dense, st);
}
