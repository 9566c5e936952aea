/* hop.cu -- precision dispatch of the hopping-term launch. */
#include "qcd_internal.h"

cudaError_t hop_launch_f32(const qcd_gauge* g, const HopLaunch& L, cudaStream_t st);
cudaError_t hop_launch_f64(const qcd_gauge* g, const HopLaunch& L, cudaStream_t st);

int hop_launch(qcd_ctx* ctx, const qcd_gauge* g, const HopLaunch& L)
{
    if (L.out_parity != 0 && L.out_parity != 1) return qcd_set_error(QCD_EINVAL, "hop: parity must be 0|1");
    if (g->precision != 4 && g->precision != 8) return qcd_set_error(QCD_EINVAL, "hop: needs an fp32 or fp64 gauge handle");
    if (L.norm_out) {
        /* one partial per block of the fused norm; blocks of >= 64 threads (grown on demand, never in a solver loop:
         * qcd_set_operator sizes it) */
        const size_t need = ((size_t)g->geo.Vh + 63) / 64;
        if (ctx->hop_partial_cap < need) {
            if (ctx->d_hop_partial) cudaFree(ctx->d_hop_partial);
            ctx->d_hop_partial = nullptr;
            ctx->hop_partial_cap = 0;
            cudaError_t ea = cudaMalloc(&ctx->d_hop_partial, need * sizeof(double));
            if (ea != cudaSuccess) return qcd_set_error(QCD_EALLOC, "hop: norm partials: %s", cudaGetErrorString(ea));
            ctx->hop_partial_cap = need;
        }
    }
    cudaError_t e = (g->precision == 4) ? hop_launch_f32(g, L, ctx->stream) : hop_launch_f64(g, L, ctx->stream);
    if (e != cudaSuccess) return qcd_set_error(QCD_ECUDA, "hop launch: %s", cudaGetErrorString(e));
    ctx->launches++;
    return QCD_OK;
}
