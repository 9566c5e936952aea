/* fp64 instantiations of the hopping-term kernel (outer / reliable-update precision). */
#include "hop_kernel.cuh"

cudaError_t hop_launch_f64(const qcd_gauge* g, const HopLaunch& L, cudaStream_t st)
{
    HopArgs<double> A = make_hop_args<double>(g, L);
    return hop_dispatch<double>(A, g->reconstruct, L.dagger, L.mode, st);
}

cudaError_t clover_site_launch_f64(void* out, const void* in, const void* clov, int Vh, cudaStream_t st)
{
    return clover_site_launch<double>(out, in, clov, Vh, st);
}
