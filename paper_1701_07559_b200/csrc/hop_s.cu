// hop kernels instantiated for precision PS (see hop_kernels.cuh)
#include "hop_kernels.cuh"
int mdwf_launch_hop_S(int dag, int pre, int post, int own, const HopArgs &a, cudaStream_t st)
{
    return launch_hop_prec<PS>(dag, pre, post, own, a, st);
}
int mdwf_launch_sdense_S(int L5, int Vh, const SpinorBuf &in, const SpinorBuf &out, const void *dense, cudaStream_t st)
{
    return launch_sdense_prec<PS>(L5, Vh, in, out, dense, st);
}
