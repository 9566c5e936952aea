/* hop.cu -- precision dispatch of the hopping-term launch. */
#include "qcd_internal.h"

cudaError_t hop_launch_f32(const qcd_gauge* g, const HopLaunch& L, cudaStream_t st);
cudaError_t hop_launch_f64(const qcd_gauge* g, const HopLaunch& L, cudaStream_t st);

int hop_launch(qcd_ctx* ctx, const qcd_gauge* g, const HopLaunch& L)
{
    if (L.out_parity != 0 && L.out_parity != 1) return qcd_set_error(QCD_EINVAL, "hop: parity must be 0|1");
    cudaError_t e = (g->precision == 4) ? hop_launch_f32(g, L, ctx->stream) : hop_launch_f64(g, L, ctx->stream);
    if (e != cudaSuccess) return qcd_set_error(QCD_ECUDA, "hop launch: %s", cudaGetErrorString(e));
    ctx->launches++;
    return QCD_OK;
}
