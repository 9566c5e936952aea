/* fp32 instantiations of the hopping-term kernel (single precision). */
#include "hop_kernel.cuh"

cudaError_t hop_tile_launch_f32(const qcd_gauge* g, const HopLaunch& L, cudaStream_t st, bool* handled); /* hop_tile.cu */

cudaError_t hop_launch_f32(const qcd_gauge* g, const HopLaunch& L, cudaStream_t st)
{
    if (L.mode == HOP_CHEB) {
        bool handled = false;
        const cudaError_t e = hop_tile_launch_f32(g, L, st, &handled);
        if (handled || e != cudaSuccess) return e;
    }
    HopArgs<float> A = make_hop_args<float>(g, L);
    return hop_dispatch<float>(A, g->reconstruct, L.dagger, L.mode, st);
}

cudaError_t clover_site_launch_f32(void* out, const void* in, const void* clov, int Vh, cudaStream_t st)
{
    return clover_site_launch<float>(out, in, clov, Vh, st);
}
