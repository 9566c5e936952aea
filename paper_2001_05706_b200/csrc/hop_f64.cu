/* fp64 instantiations of the hopping-term kernel (outer / reliable-update precision). */
#include "hop_kernel.cuh"

cudaError_t hop_launch_f64(const qcd_gauge* g, const HopLaunch& L, cudaStream_t st)
{
    HopArgs<double> A = make_hop_args<double>(g, L);
    return hop_dispatch<double>(A, g->reconstruct, L.dagger, L.mode, st);
}
