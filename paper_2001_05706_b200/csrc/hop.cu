/* hop.cu -- precision dispatch of the hopping-term launch. */
#include "qcd_internal.h"

cudaError_t hop_launch_f32(const qcd_gauge* g, const HopLaunch& L, cudaStream_t st);
cudaError_t hop_launch_f64(const qcd_gauge* g, const HopLaunch& L, cudaStream_t st);

cudaError_t clover_site_launch_f32(void* out, const void* in, const void* clov, int Vh, cudaStream_t st);
cudaError_t clover_site_launch_f64(void* out, const void* in, const void* clov, int Vh, cudaStream_t st);

/* out = C in on one parity; block = 0,1: A of parity 0,1; 2,3: A^-1 of parity 0,1 */
int clover_site_apply(qcd_ctx* ctx, void* out, const void* in, const qcd_clover* c, int block)
{
    const void* clov = (const char*)c->data + (size_t)block * c->block_bytes;
    const cudaError_t e = (c->precision == 4) ? clover_site_launch_f32(out, in, clov, c->geo.Vh, ctx->stream)
                                              : clover_site_launch_f64(out, in, clov, c->geo.Vh, ctx->stream);
    if (e != cudaSuccess) return qcd_set_error(QCD_ECUDA, "clover apply launch: %s", cudaGetErrorString(e));
    ctx->launches++;
    return QCD_OK;
}

int hop_norm_scratch(qcd_ctx* ctx, size_t nblocks)
{
    if (ctx->hop_partial_cap >= nblocks) return QCD_OK;
    if (ctx->d_hop_partial) cudaFree(ctx->d_hop_partial);
    if (ctx->d_hop_ticket) cudaFree(ctx->d_hop_ticket);
    ctx->d_hop_partial = nullptr;
    ctx->d_hop_ticket = nullptr;
    ctx->hop_partial_cap = 0;
    const size_t ngroups = (nblocks + HOP_NORM_GROUP - 1) / HOP_NORM_GROUP;
    cudaError_t e = cudaMalloc(&ctx->d_hop_partial, (nblocks + ngroups) * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_hop_ticket, (ngroups + 1) * sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaMemset(ctx->d_hop_ticket, 0, (ngroups + 1) * sizeof(unsigned int));
    if (e != cudaSuccess) return qcd_set_error(QCD_EALLOC, "hop: fused-norm scratch: %s", cudaGetErrorString(e));
    ctx->hop_partial_cap = nblocks;
    return QCD_OK;
}

int hop_launch(qcd_ctx* ctx, const qcd_gauge* g, const HopLaunch& L)
{
    if (L.out_parity != 0 && L.out_parity != 1) return qcd_set_error(QCD_EINVAL, "hop: parity must be 0|1");
    if (g->precision != 4 && g->precision != 8) return qcd_set_error(QCD_EINVAL, "hop: needs an fp32 or fp64 gauge handle");
    if (L.norm_out) { /* sized by qcd_set_operator; grown here only for a first use outside a solver */
        const int rc = hop_norm_scratch(ctx, ((size_t)g->geo.Vh + 63) / 64);
        if (rc) return rc;
    }
    cudaError_t e = (g->precision == 4) ? hop_launch_f32(g, L, ctx->stream) : hop_launch_f64(g, L, ctx->stream);
    if (e != cudaSuccess) return qcd_set_error(QCD_ECUDA, "hop launch: %s", cudaGetErrorString(e));
    ctx->launches++;
    return QCD_OK;
}
