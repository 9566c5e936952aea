/*
 * solver.cu -- CG on N = M^dag M (reading O6/S13), the
 * reliable-update mixed-precision CG (a12, reading O7/S15; PAPER.md:163 ref. [1]) and
 * the Chebyshev polynomial driver (a14, reading O8/S16).
 *
 * alpha and beta never leave the device: reductions write rho, <p,Np> and beta to
 * device slots and the update kernels read them there.  The host reads back two
 * doubles per iteration for the stopping test.
 */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "qcd_internal.h"

#define RC(expr)               \
    do {                       \
        int rc__ = (expr);     \
        if (rc__) return rc__; \
    } while (0)

namespace {

qcd_ctx* g_last_ctx = nullptr;

/* device scalar slots: rho before iteration k lives in slot S_RHO + ((k-1) & 1), the update of
 * iteration k writes rho' to S_RHO + (k & 1) */
enum { S_RHO = 0, S_PQ = 2, S_NTMP = 3, S_AUX = 6 };
inline int rho_slot(int k) { return S_RHO + (k & 1); }

struct Op {
    qcd_ctx* ctx;
    const qcd_gauge* g;
    const qcd_clover* c;
    double kappa;
    int parity;
    size_t nreal;
    size_t bytes;
};

Op make_op(qcd_ctx* ctx, const qcd_gauge* g, const qcd_clover* c)
{
    Op o;
    o.ctx = ctx; o.g = g; o.c = c; o.kappa = ctx->kappa; o.parity = ctx->op_parity;
    o.nreal = (size_t)(ctx->op_parity == 2 ? g->geo.V : g->geo.Vh) * 24;
    o.bytes = o.nreal * g->precision;
    return o;
}

/* q = M^dag M p, t = M p (kept), tmp = hop temporary.  With ex: the launches are gated by
 * ex->halt and |t|^2 = <p, M^dag M p> is accumulated in the epilogue of the launch(es) writing t
 * (no separate pass over t). */
int apply_N(const Op& o, void* q, const void* p, void* t, void* tmp, const OpExtra* ex = nullptr)
{
    int rc = op_apply_M(o.ctx, t, p, tmp, o.g, o.c, o.kappa, o.parity, 0, ex);
    if (rc) return rc;
    OpExtra gate = {ex ? ex->halt : nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    return op_apply_M(o.ctx, q, t, tmp, o.g, o.c, o.kappa, o.parity, 1, ex ? &gate : nullptr);
}

/* One CG iteration n on the device, the BLAS fused into the operator (SURVEY.md 8(a) a10 "fused CG BLAS"):
 *   t = M p, <p,Np> = |t|^2 in the epilogue of the launch writing t;
 *   q = M^dag t is never stored: the launch that computes it does r -= alpha q, rho' = |r|^2 and the stop /
 *   reliable-update decision (cg_decide) in its epilogue;
 *   x += alpha p ; p = r + beta p in one pass (blas_cg_xp), the p update only while the solver runs.
 * Per iteration and site this moves 3 vectors less than separate  |t|^2, (x, r, rho') and p passes. */
int cg_iteration(const Op& o, int n, void* x, void* r, void* p, void* q, void* t, void* tmp)
{
    qcd_ctx* ctx = o.ctx;
    double* d = ctx->d_scalar;
    double *rho = d + rho_slot(n - 1), *rho2 = d + rho_slot(n);
    const int* halt = &ctx->d_ctl->halt;
    const int P = o.g->precision;
    const OpExtra ex1 = {halt, d + S_PQ, d + S_NTMP, nullptr, nullptr, nullptr, nullptr, nullptr};
    RC(op_apply_M(ctx, t, p, tmp, o.g, o.c, o.kappa, o.parity, 0, &ex1));
    const OpExtra ex2 = {halt, rho2, d + S_NTMP, r, rho, d + S_PQ, ctx->d_ctl, ctx->d_status};
    RC(op_apply_M(ctx, q, t, tmp, o.g, o.c, o.kappa, o.parity, 1, &ex2));
    return blas_cg_xp(ctx, dev_ratio(rho, d + S_PQ), dev_ratio(rho2, rho), r, x, p, o.nreal, P, ctx->d_ctl, n);
}

int fetch(qcd_ctx* ctx, int slot, int n)
{
    QCD_CHECK_CUDA(cudaMemcpyAsync(ctx->h_scalar + slot, ctx->d_scalar + slot, sizeof(double) * n, cudaMemcpyDeviceToHost, ctx->stream));
    QCD_CHECK_CUDA(cudaStreamSynchronize(ctx->stream));
    return QCD_OK;
}

/* ---- device-side control (CgCtl) ----------------------------------------------------------
 * The host enqueues iterations ahead of the device; the CG update kernel decides on the device
 * whether the iteration converged / needs a reliable update / broke down, sets ctl->halt and
 * mirrors (iterations done, halt) into two mapped host words.  While halt is set every further
 * kernel of the iteration returns at once, so nothing enqueued ahead changes x, r or p.  The host
 * only polls the mapped words (no stream synchronisation per iteration). */
int ctl_start(qcd_ctx* ctx, double thresh, double delta, double rmax)
{
    CgCtl* h = reinterpret_cast<CgCtl*>(ctx->h_scalar + 8); /* pinned staging (h_scalar has SC_COUNT = 16 doubles) */
    memset(h, 0, sizeof(CgCtl));
    h->thresh = thresh; h->delta = delta; h->rmax = rmax; h->rnorm = rmax;
    ctx->h_status[0] = 0;
    ctx->h_status[1] = 0;
    QCD_CHECK_CUDA(cudaMemcpyAsync(ctx->d_ctl, h, sizeof(CgCtl), cudaMemcpyHostToDevice, ctx->stream));
    return QCD_OK;
}

int ctl_read(qcd_ctx* ctx, CgCtl* out)
{
    CgCtl* h = reinterpret_cast<CgCtl*>(ctx->h_scalar + 8);
    QCD_CHECK_CUDA(cudaMemcpyAsync(h, ctx->d_ctl, sizeof(CgCtl), cudaMemcpyDeviceToHost, ctx->stream));
    QCD_CHECK_CUDA(cudaStreamSynchronize(ctx->stream));
    *out = *h;
    return QCD_OK;
}

/* block until iteration `need` has been executed or the solver halted */
int ctl_wait(qcd_ctx* ctx, int need)
{
    volatile int* hs = ctx->h_status;
    unsigned spins = 0;
    while (hs[0] < need && hs[1] == 0) {
        if ((++spins & 0x3ff) == 0) {
            const cudaError_t e = cudaStreamQuery(ctx->stream);
            if (e == cudaSuccess) return QCD_OK; /* drained: the caller reads the state */
            if (e != cudaErrorNotReady) return qcd_set_error(QCD_ECUDA, "cg: %s", cudaGetErrorString(e));
        }
    }
    return QCD_OK;
}

int run_ahead()
{
    /* iterations the host may be ahead of the device; each one enqueued past a halt costs a few
     * skipped launches, each one less risks an idle device */
    const char* e = getenv("QCD_CG_RUNAHEAD"); /* read per solve: tests sweep it */
    int d = e ? atoi(e) : 0; /* 0: enqueue iteration n + 1 as soon as iteration n's residual update has reported (the x / p pass of
                               * iteration n is still running then, so the device never idles); measured on B200, 32^3x64: mixed CG 56.7 /
                               * 57.7 / 58.2 ms for 0 / 1 / 2 (every launch enqueued past a reliable update is a skipped launch), pure
                               * fp64 CG 92.4 - 93.0 ms for all three */
    if (d < 0) d = 0;
    if (d > 64) d = 64;
    return d;
}

int true_residual(const Op& o, const void* x, const void* b, void* q, void* t, void* tmp, double bnorm, double* r_true)
{
    qcd_ctx* ctx = o.ctx;
    const int P = o.g->precision;
    RC(apply_N(o, q, x, t, tmp));
    RC(blas_axpby(ctx, host_scalar(1.0), b, host_scalar(-1.0), q, o.nreal, P)); /* q = b - q */
    RC(blas_norm2(ctx, q, o.nreal, P, ctx->d_scalar + S_AUX));
    RC(fetch(ctx, S_AUX, 1));
    *r_true = bnorm > 0 ? sqrt(ctx->h_scalar[S_AUX]) / bnorm : 0.0;
    return QCD_OK;
}

int cg_pure(qcd_ctx* ctx, void* x, const void* b, double tol, int maxiter, qcd_stats* st)
{
    const Op o = make_op(ctx, ctx->g_hi, ctx->c_hi);
    const int P = o.g->precision;
    QCD_REQUIRE(P == 4 || P == 8, "cg: the operator needs an fp32 or fp64 gauge handle");
    const int nfields = o.parity == 2 ? 4 : 5;
    QCD_REQUIRE(ctx->ws && ctx->ws_bytes >= nfields * o.bytes, "cg: workspace too small (need %zu bytes)", nfields * o.bytes);
    char* w = (char*)ctx->ws;
    void *r = w, *p = w + o.bytes, *q = w + 2 * o.bytes, *t = w + 3 * o.bytes, *tmp = w + 4 * o.bytes;
    double* d = ctx->d_scalar;
    double* h = ctx->h_scalar;

    RC(blas_zero(ctx, x, o.bytes));
    RC(blas_copy(ctx, r, b, o.bytes));
    RC(blas_copy(ctx, p, b, o.bytes));
    RC(blas_norm2(ctx, b, o.nreal, P, d + rho_slot(0)));
    RC(fetch(ctx, rho_slot(0), 1));
    const double bnorm = sqrt(h[rho_slot(0)]);
    double rnorm = bnorm;
    int k = 0, conv = (bnorm == 0.0), brk = 0;
    if (!conv && maxiter > 0) {
        RC(ctl_start(ctx, tol * bnorm, 0.0, bnorm));
        const int ahead = run_ahead();
        int n = 0;
        while (n < maxiter) {
            n++;
            RC(cg_iteration(o, n, x, r, p, q, t, tmp));
            if (n > ahead) RC(ctl_wait(ctx, n - ahead));
            if (ctx->h_status[1]) break;
        }
        CgCtl c;
        RC(ctl_read(ctx, &c));
        conv = c.halt == CG_CONVERGED;
        brk = c.halt == CG_BREAKDOWN;
        k = c.iter + brk;
        rnorm = c.rnorm;
    }
    double r_true = 0.0;
    RC(true_residual(o, x, b, q, t, tmp, bnorm, &r_true));
    if (st) {
        st->iters = k; st->reliable_updates = 0; st->converged = conv; st->breakdown = brk;
        st->r_iter = bnorm > 0 ? rnorm / bnorm : 0.0;
        st->r_true = r_true;
    }
    if (brk) return qcd_set_error(QCD_EBREAKDOWN, "cg: <p,Np> <= 0 or NaN at iteration %d", k);
    return conv ? QCD_OK : QCD_NOCONV;
}

int cg_mixed(qcd_ctx* ctx, void* y, const void* b, double tol, int maxiter, qcd_stats* st)
{
    const Op oh = make_op(ctx, ctx->g_hi, ctx->c_hi);
    Op ol = make_op(ctx, ctx->g_lo, ctx->c_lo);
    QCD_REQUIRE(oh.g->precision == 8 && (ol.g->precision == 4 || ol.g->precision == 2),
                "mixed cg: needs an fp64 high and an fp32 or 16-bit low operator");
    /* 16-bit low operator (reading H1): the inner vectors stay fp32, the operator streams 16-bit fields */
    const bool half = ol.g->precision == 2;
    ol.bytes = ol.nreal * 4;
    const int nblocks = ol.parity == 2 ? 2 : 1;
    const size_t need = 4 * oh.bytes + 6 * ol.bytes;
    QCD_REQUIRE(ctx->ws && ctx->ws_bytes >= need, "mixed cg: workspace too small (need %zu bytes)", need);
    char* w = (char*)ctx->ws;
    void *rh = w, *th = w + oh.bytes, *h1 = w + 2 * oh.bytes, *h2 = w + 3 * oh.bytes;
    char* wl = w + 4 * oh.bytes;
    void *x = wl, *r = wl + ol.bytes, *p = wl + 2 * ol.bytes, *q = wl + 3 * ol.bytes, *tl = wl + 4 * ol.bytes, *l2 = wl + 5 * ol.bytes;
    /* 16-bit operator buffers share the tl/l2 region: 3 x 52 B/site < 2 x 96 B/site */
    const size_t hbytes = (size_t)nblocks * ol.g->geo.Vh * 52;
    char *ph = (char*)tl, *th16 = ph + hbytes, *tmp16 = th16 + hbytes;
    double* d = ctx->d_scalar;
    double* h = ctx->h_scalar;
    const size_t n = oh.nreal, Vh = (size_t)oh.g->geo.Vh;

    RC(blas_zero(ctx, y, oh.bytes));
    RC(blas_zero(ctx, x, ol.bytes));
    RC(blas_convert(ctx, r, 4, b, 8, n, Vh));
    if (half) RC(half_xpay_store(ctx, host_scalar(1.0), r, host_scalar(0.0), 1, p, ph, Vh, nblocks));
    else RC(blas_copy(ctx, p, r, ol.bytes));
    RC(blas_norm2(ctx, b, n, 8, d + S_AUX));
    RC(blas_norm2(ctx, r, n, 4, d + rho_slot(0)));
    RC(fetch(ctx, 0, 8));
    const double bnorm = sqrt(h[S_AUX]);
    double rhnorm = bnorm;
    int k = 0, conv = (bnorm == 0.0), brk = 0, nup = 0;
    const bool trace = getenv("QCD_TRACE") != nullptr;
    if (!conv && maxiter > 0) {
        RC(ctl_start(ctx, tol * bnorm, ctx->delta, sqrt(h[rho_slot(0)])));
        const int* halt = &ctx->d_ctl->halt;
        const int ahead = run_ahead();
        int nq = 0; /* iterations enqueued (== executed whenever the device is not halted) */
        for (;;) {
            while (nq < maxiter) {
                nq++;
                if (half) {
                    double *rho = d + rho_slot(nq - 1), *rho2 = d + rho_slot(nq);
                    /* q = M^dag store16(M store16(p)); <p, q> taken as written */
                    RC(op_apply_M_half(ctx, th16, 0, ph, tmp16, ol.g, ol.c, ol.kappa, ol.parity, 0, halt));
                    RC(op_apply_M_half(ctx, q, 1, th16, tmp16, ol.g, ol.c, ol.kappa, ol.parity, 1, halt));
                    RC(blas_redot(ctx, p, q, n, 4, d + S_PQ, halt));
                    RC(blas_cg_update(ctx, dev_ratio(rho, d + S_PQ), p, q, x, r, n, 4, rho2, ctx->d_ctl, ctx->d_status));
                    /* p = r + beta p, beta = (float)(rho'/rho); skipped when the update halted the iteration */
                    RC(half_xpay_store(ctx, host_scalar(1.0), r, dev_ratio(rho2, rho), 0, p, ph, Vh, nblocks, halt));
                } else {
                    RC(cg_iteration(ol, nq, x, r, p, q, tl, l2));
                }
                if (nq > ahead) RC(ctl_wait(ctx, nq - ahead));
                if (ctx->h_status[1]) break;
            }
            CgCtl c;
            RC(ctl_read(ctx, &c));
            k = c.iter;
            if (c.halt == CG_RUN) break; /* maxiter */
            if (c.halt == CG_BREAKDOWN) { brk = 1; k++; break; }
            /* reliable update due after iteration k (reading O7) */
            double *rho = d + rho_slot(k - 1), *rho2 = d + rho_slot(k);
            RC(blas_accumulate_hi(ctx, y, x, n, Vh));                          /* y += x ; x = 0          */
            RC(apply_N(oh, th, y, h1, h2));                                    /* th = N_hi y             */
            RC(blas_residual_hi(ctx, rh, r, b, th, n, Vh, rho2, ctx->d_ctl));  /* rh = b - th ; r = (f)rh ; rho' = |rh|^2 */
            RC(ctl_read(ctx, &c));
            rhnorm = c.rnorm;
            nup++;
            if (trace) fprintf(stderr, "mixed   reliable update %d after iteration %d: |r_hi|/|b| = %.6e\n", nup, k, rhnorm / bnorm);
            if (c.halt == CG_CONVERGED) { conv = 1; break; }
            if (k >= maxiter) break;
            ctx->h_status[1] = 0;
            ctx->h_status[0] = k;
            if (half) RC(half_xpay_store(ctx, host_scalar(1.0), r, dev_ratio(rho2, rho), 0, p, ph, Vh, nblocks));
            else RC(blas_axpby(ctx, host_scalar(1.0), r, dev_ratio(rho2, rho), p, n, 4));
            nq = k;
        }
    }
    if (!conv) RC(blas_accumulate_hi(ctx, y, x, n, Vh));
    double r_true = 0.0;
    /* Convergence is only ever declared by a reliable update, whose rh = b - N_hi y is the fp64
     * residual of the returned y recomputed from scratch (O6): it is the true residual; recompute
     * only on the other exits (maxiter, breakdown, b = 0). */
    if (conv && nup > 0 && bnorm > 0.0) r_true = rhnorm / bnorm;
    else RC(true_residual(oh, y, b, th, h1, h2, bnorm, &r_true));
    if (st) {
        st->iters = k; st->reliable_updates = nup; st->converged = conv; st->breakdown = brk;
        st->r_iter = bnorm > 0 ? rhnorm / bnorm : 0.0;
        st->r_true = r_true;
    }
    if (brk) return qcd_set_error(QCD_EBREAKDOWN, "mixed cg: <p,Np> <= 0 or NaN at iteration %d", k);
    return conv ? QCD_OK : QCD_NOCONV;
}

/* The scalar side of the multi-shift CG (B. Jegerlehner, hep-lat/9612014): zeta_s of the previous, current and next
 * iteration for every shift, relative to the base shift. */
struct ShiftRecurrence {
    double zm[QCD_MAX_SHIFTS], z0[QCD_MAX_SHIFTS], zp[QCD_MAX_SHIFTS];
    double alpha_old, beta_old;
    const double* shifts;
    /* x_s += c_s p_s, c_s = alpha zeta_s' / zeta_s, for the first nact shifts */
    MultiShiftCoef x_coef(double alpha, int nact)
    {
        MultiShiftCoef cx;
        cx.ns = nact; cx.alpha = alpha;
        for (int s = 0; s < nact; s++) {
            const double sh = shifts[s] - shifts[0];
            zp[s] = z0[s] * zm[s] * alpha_old / (alpha * beta_old * (zm[s] - z0[s]) + zm[s] * alpha_old * (1.0 + sh * alpha));
            cx.c[s] = alpha * zp[s] / z0[s];
        }
        return cx;
    }
    /* p_s = zeta_s' r + beta_s p_s, beta_s = beta (zeta_s' / zeta_s)^2; advances the recurrence */
    void p_coef(double alpha, double beta, int nact, MultiShiftCoef* cz, MultiShiftCoef* cb)
    {
        cz->ns = cb->ns = nact; cz->alpha = cb->alpha = 0.0;
        for (int s = 0; s < nact; s++) {
            const double ratio = zp[s] / z0[s];
            cz->c[s] = zp[s];
            cb->c[s] = beta * ratio * ratio;
            zm[s] = z0[s];
            z0[s] = zp[s];
        }
        alpha_old = alpha; beta_old = beta;
    }
};

double hop_flops_per_apply_M(const Op& o)
{
    /* nominal (reading S18): 1320 per output site per hop, +504 per clover / clover-inverse apply */
    const double Vh = (double)o.g->geo.Vh;
    const double hops = 2.0; /* both forms launch two single-parity hops per M */
    double f = hops * 1320.0 * Vh;
    if (o.c) f += 2.0 * 504.0 * Vh;
    return f;
}

} // namespace

void solver_forget_ctx(const qcd_ctx* ctx)
{
    if (g_last_ctx == ctx) g_last_ctx = nullptr;
}

extern "C" {

int qcd_set_operator(qcd_ctx* ctx, const qcd_gauge* g_hi, const qcd_gauge* g_lo, const qcd_clover* c_hi, const qcd_clover* c_lo,
                     double kappa, double csw, int parity, double delta)
{
    QCD_REQUIRE(ctx && g_hi, "set_operator: NULL ctx or gauge");
    QCD_REQUIRE(parity == 0 || parity == 1 || parity == 2, "set_operator: parity must be 0|1|2");
    QCD_REQUIRE(g_hi->ctx == ctx, "set_operator: g_hi belongs to another ctx");
    QCD_REQUIRE(g_hi->precision == 4 || g_hi->precision == 8, "set_operator: g_hi must be an fp32 or fp64 gauge handle");
    if (c_hi) {
        QCD_REQUIRE(c_hi->precision == g_hi->precision && c_hi->geo.V == g_hi->geo.V, "set_operator: c_hi does not match g_hi");
        QCD_REQUIRE(c_hi->kappa == kappa && c_hi->csw == csw, "set_operator: kappa/csw differ from the clover's");
    }
    if (g_lo) {
        QCD_REQUIRE(g_lo->ctx == ctx, "set_operator: g_lo belongs to another ctx");
        QCD_REQUIRE(g_lo->precision == 2 || g_lo->precision == 4, "set_operator: g_lo must be an fp32 or 16-bit gauge handle");
        QCD_REQUIRE(g_lo->geo.V == g_hi->geo.V && g_lo->tb == g_hi->tb, "set_operator: g_lo does not match g_hi");
        QCD_REQUIRE((c_lo != nullptr) == (c_hi != nullptr), "set_operator: c_lo and c_hi must both be given or both NULL");
        if (c_lo) {
            QCD_REQUIRE(c_lo->precision == g_lo->precision && c_lo->geo.V == g_lo->geo.V, "set_operator: c_lo does not match g_lo");
            QCD_REQUIRE(c_lo->kappa == kappa && c_lo->csw == csw, "set_operator: kappa/csw differ from c_lo's");
        }
        QCD_REQUIRE(delta > 0.0 && delta < 1.0, "set_operator: delta must be in (0,1)");
    }
    ctx->g_hi = g_hi; ctx->g_lo = g_lo; ctx->c_hi = c_hi; ctx->c_lo = g_lo ? c_lo : nullptr;
    ctx->kappa = kappa; ctx->csw = csw; ctx->op_parity = parity; ctx->delta = delta;
    ctx->op_set = 1;
    g_last_ctx = ctx;
    /* size the scratch of the norm fused into the hop epilogue now, not inside a solve */
    QCD_CHECK_CUDA(cudaSetDevice(ctx->device));
    {
        const int rc = hop_norm_scratch(ctx, ((size_t)g_hi->geo.Vh + 63) / 64);
        if (rc) return rc;
    }
    return QCD_OK;
}

int qcd_apply_operator(qcd_ctx* ctx, void* out, const void* in, int flags)
{
    QCD_REQUIRE(ctx && ctx->op_set, "apply_operator: no operator set");
    return qcd_dslash_ex(out, in, ctx->g_hi, ctx->c_hi, ctx->kappa, ctx->csw, ctx->op_parity, flags, nullptr);
}

/* Even-odd source preparation and solution reconstruction (reading O5) in the high precision of the
 * operator of qcd_set_operator; p = its parity, pb = 1 - p; full fields hold the even block, then the odd one. */
static inline size_t eo_block_bytes(const qcd_ctx* ctx) { return (size_t)ctx->g_hi->geo.Vh * 24 * ctx->g_hi->precision; }

int qcd_eo_prepare(qcd_ctx* ctx, void* bhat, const void* b)
{
    QCD_REQUIRE(ctx && ctx->op_set, "eo_prepare: no operator set (qcd_set_operator)");
    QCD_REQUIRE(ctx->op_parity == 0 || ctx->op_parity == 1, "eo_prepare: the operator set is the full-lattice one");
    QCD_REQUIRE(bhat && b && (((uintptr_t)bhat | (uintptr_t)b) & 15u) == 0, "eo_prepare: pointers must be non-NULL, 16-byte aligned");
    const size_t blk = eo_block_bytes(ctx);
    const char* bc = (const char*)b;
    QCD_REQUIRE((const char*)bhat + blk <= bc || bc + 2 * blk <= (const char*)bhat, "eo_prepare: bhat and b alias");
    QCD_ON_DEVICE(ctx);
    const int p = ctx->op_parity, pb = 1 - p;
    const void* t = bc + (size_t)pb * blk;
    if (ctx->c_hi) { /* t = Ainv_pb b_pb */
        QCD_REQUIRE(ctx->ws && ctx->ws_bytes >= blk, "eo_prepare: workspace missing (qcd_set_workspace)");
        QCD_REQUIRE((const char*)ctx->ws + blk <= (const char*)bhat || (const char*)bhat + blk <= (const char*)ctx->ws, "eo_prepare: bhat lies in the workspace");
        RC(clover_site_apply(ctx, ctx->ws, t, ctx->c_hi, 2 + pb));
        t = ctx->ws;
    }
    HopLaunch L;
    memset(&L, 0, sizeof(L));
    L.out = bhat; L.in = t; L.z = bc + (size_t)p * blk; L.a = 1.0; L.b = ctx->kappa; L.out_parity = p; L.mode = HOP_XPAY;
    return hop_launch(ctx, ctx->g_hi, L);
}

int qcd_eo_reconstruct(qcd_ctx* ctx, void* x, const void* b)
{
    QCD_REQUIRE(ctx && ctx->op_set, "eo_reconstruct: no operator set (qcd_set_operator)");
    QCD_REQUIRE(ctx->op_parity == 0 || ctx->op_parity == 1, "eo_reconstruct: the operator set is the full-lattice one");
    QCD_REQUIRE(x && b && (((uintptr_t)x | (uintptr_t)b) & 15u) == 0, "eo_reconstruct: pointers must be non-NULL, 16-byte aligned");
    const size_t blk = eo_block_bytes(ctx);
    QCD_REQUIRE((char*)x + 2 * blk <= (const char*)b || (const char*)b + 2 * blk <= (char*)x, "eo_reconstruct: x and b alias");
    QCD_ON_DEVICE(ctx);
    const int p = ctx->op_parity, pb = 1 - p;
    char* x_pb = (char*)x + (size_t)pb * blk;
    HopLaunch L;
    memset(&L, 0, sizeof(L)); /* x_pb = b_pb + kappa H_{pb,p} x_p */
    L.out = x_pb; L.in = (char*)x + (size_t)p * blk; L.z = (const char*)b + (size_t)pb * blk; L.a = 1.0; L.b = ctx->kappa;
    L.out_parity = pb; L.mode = HOP_XPAY;
    RC(hop_launch(ctx, ctx->g_hi, L));
    if (ctx->c_hi) RC(clover_site_apply(ctx, x_pb, x_pb, ctx->c_hi, 2 + pb)); /* site-local: in place */
    return QCD_OK;
}

int qcd_clover_apply(qcd_ctx* ctx, void* out, const void* in, const qcd_clover* c, int inverse, int parity)
{
    QCD_REQUIRE(ctx && c && c->ctx == ctx, "clover_apply: NULL handle or clover of another context");
    QCD_REQUIRE(c->precision == 4 || c->precision == 8, "clover_apply: needs an fp32 or fp64 clover handle");
    QCD_REQUIRE(parity == 0 || parity == 1, "clover_apply: parity must be 0|1");
    QCD_REQUIRE(out && in && (((uintptr_t)out | (uintptr_t)in) & 15u) == 0, "clover_apply: pointers must be non-NULL, 16-byte aligned");
    const size_t blk = (size_t)c->geo.Vh * 24 * c->precision;
    QCD_REQUIRE(out == in || (char*)out + blk <= (const char*)in || (const char*)in + blk <= (char*)out, "clover_apply: out and in overlap partially");
    QCD_ON_DEVICE(ctx);
    return clover_site_apply(ctx, out, in, c, (inverse ? 2 : 0) + parity);
}

int qcd_cg_solve_ex(qcd_ctx* ctx, void* x, const void* b, double tol, int maxiter, qcd_stats* stats)
{
    QCD_REQUIRE(ctx && ctx->op_set, "cg_solve: no operator set (qcd_set_operator)");
    QCD_REQUIRE(x && b && (((uintptr_t)x | (uintptr_t)b) & 15u) == 0, "cg_solve: x/b must be non-NULL, 16-byte aligned");
    QCD_REQUIRE(x != b, "cg_solve: x and b alias");
    QCD_REQUIRE(tol > 0.0 && maxiter >= 0, "cg_solve: tol must be > 0 and maxiter >= 0");
    QCD_ON_DEVICE(ctx);
    qcd_stats st;
    memset(&st, 0, sizeof(st));
    cudaEvent_t e0, e1;
    QCD_CHECK_CUDA(cudaEventCreate(&e0));
    QCD_CHECK_CUDA(cudaEventCreate(&e1));
    QCD_CHECK_CUDA(cudaEventRecord(e0, ctx->stream));
    const int rc = ctx->g_lo ? cg_mixed(ctx, x, b, tol, maxiter, &st) : cg_pure(ctx, x, b, tol, maxiter, &st);
    cudaEventRecord(e1, ctx->stream);
    cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    st.seconds = ms * 1e-3;
    {
        const Op o = make_op(ctx, ctx->g_lo ? ctx->g_lo : ctx->g_hi, ctx->g_lo ? ctx->c_lo : ctx->c_hi);
        st.flops = 2.0 * hop_flops_per_apply_M(o) * st.iters;
        const double w = o.g->precision;
        const double Vh = (double)o.g->geo.Vh;
        const double hop_bytes = (48.0 + 8.0 * o.g->reconstruct) * w * Vh;
        double per_M = 2.0 * hop_bytes + 24.0 * w * Vh + (o.c ? 2.0 * 72.0 * w * Vh : 0.0);
        const double blas = (2.0 + 6.0 + 3.0) * w * (double)o.nreal; /* redot + cg_update + xpay */
        st.bytes = (2.0 * per_M + blas) * st.iters;
    }
    if (stats) *stats = st;
    return rc;
}

int qcd_cg_solve(void* x, const void* b, double tol, int maxiter)
{
    QCD_REQUIRE(g_last_ctx, "cg_solve: qcd_set_operator has not been called");
    return qcd_cg_solve_ex(g_last_ctx, x, b, tol, maxiter, nullptr);
}

int qcd_cg_multishift(qcd_ctx* ctx, void* x, const void* b, const double* shifts, int nshift, double tol, int maxiter,
                      qcd_stats* stats, double* r_true)
{
    QCD_REQUIRE(ctx && ctx->op_set, "cg_multishift: no operator set (qcd_set_operator)");
    QCD_REQUIRE(!ctx->g_lo, "cg_multishift: pure-precision operator only");
    QCD_REQUIRE(x && b && shifts && (((uintptr_t)x | (uintptr_t)b) & 15u) == 0, "cg_multishift: bad pointer");
    QCD_REQUIRE(nshift >= 1 && nshift <= QCD_MAX_SHIFTS, "cg_multishift: 1 <= nshift <= %d", (int)QCD_MAX_SHIFTS);
    QCD_REQUIRE(tol > 0.0 && maxiter >= 0, "cg_multishift: tol must be > 0 and maxiter >= 0");
    QCD_ON_DEVICE(ctx);
    for (int i = 0; i < nshift; i++)
        QCD_REQUIRE(shifts[i] >= 0.0 && (i == 0 || shifts[i] > shifts[i - 1]), "cg_multishift: shifts must be >= 0 and strictly ascending");
    const Op o = make_op(ctx, ctx->g_hi, ctx->c_hi);
    const int P = o.g->precision;
    const size_t need = (size_t)(4 + nshift) * o.bytes;
    QCD_REQUIRE(ctx->ws && ctx->ws_bytes >= need, "cg_multishift: workspace too small (need %zu bytes)", need);
    {
        const uintptr_t a0 = (uintptr_t)x, a1 = (uintptr_t)b;
        QCD_REQUIRE(a0 + nshift * o.bytes <= a1 || a1 + o.bytes <= a0, "cg_multishift: x and b alias");
    }
    char* w = (char*)ctx->ws;
    void *r = w, *q = w + o.bytes, *t = w + 2 * o.bytes, *tmp = w + 3 * o.bytes;
    char* p = w + 4 * o.bytes;
    double* d = ctx->d_scalar;
    double* h = ctx->h_scalar;
    cudaEvent_t e0, e1;
    QCD_CHECK_CUDA(cudaEventCreate(&e0));
    QCD_CHECK_CUDA(cudaEventCreate(&e1));
    QCD_CHECK_CUDA(cudaEventRecord(e0, ctx->stream));

    RC(blas_zero(ctx, x, nshift * o.bytes));
    RC(blas_copy(ctx, r, b, o.bytes));
    for (int s = 0; s < nshift; s++) RC(blas_copy(ctx, p + s * o.bytes, b, o.bytes));
    RC(blas_norm2(ctx, b, o.nreal, P, d + S_RHO));
    RC(fetch(ctx, S_RHO, 1));
    const double bnorm = sqrt(h[S_RHO]);
    double rho = h[S_RHO], rnorm = bnorm;
    ShiftRecurrence rec;
    rec.alpha_old = 1.0; rec.beta_old = 0.0; rec.shifts = shifts;
    for (int s = 0; s < nshift; s++) rec.zm[s] = rec.z0[s] = 1.0;
    /* a shifted system whose residual |zeta_s| |r| has reached tol |b| is frozen (reading M1): the
     * shifts ascend, so the active systems are always the first nact */
    int k = 0, conv = (bnorm == 0.0), brk = 0, nact = nshift;
    /* Base shift 0: the iteration runs like the plain CG's (cg_iteration): <p,Np> = |t|^2 from the epilogue of the
     * launch writing t, q = M^dag t never stored, r -= alpha q and rho' = |r|^2 in the epilogue of the launch that
     * computes it, then ONE pass over the shifted systems (x_s += c_s p_s ; p_s = zeta_s r + beta_s p_s) once the host
     * has turned <p,Np> and rho' into this iteration's coefficients: one host round trip per iteration instead of
     * two, 2 + 3 per shift fewer vector streams.  A base shift > 0 needs |p|^2 as well and takes the loop below. */
    const bool fused = (shifts[0] == 0.0);
    while (fused && !conv && k < maxiter) {
        k++;
        double *d_rho = d + rho_slot(k - 1), *d_rho2 = d + rho_slot(k);
        const OpExtra ex1 = {nullptr, d + S_PQ, d + S_NTMP, nullptr, nullptr, nullptr, nullptr, nullptr};
        RC(op_apply_M(ctx, t, p, tmp, o.g, o.c, o.kappa, o.parity, 0, &ex1));
        const OpExtra ex2 = {nullptr, d_rho2, d + S_NTMP, r, d_rho, d + S_PQ, nullptr, nullptr};
        RC(op_apply_M(ctx, q, t, tmp, o.g, o.c, o.kappa, o.parity, 1, &ex2));
        RC(fetch(ctx, 0, 3));
        const double pq = h[S_PQ];
        if (!(pq > 0.0)) { brk = 1; break; } /* the launch computing q has written nothing in this case */
        const double alpha = rho / pq;
        const MultiShiftCoef cx = rec.x_coef(alpha, nact);
        const double rho2 = h[rho_slot(k)];
        rnorm = sqrt(rho2);
        conv = (rnorm <= tol * bnorm);
        if (!conv) while (nact > 1 && fabs(rec.zp[nact - 1]) * rnorm <= tol * bnorm) nact--;
        MultiShiftCoef cz, cb;
        rec.p_coef(alpha, rho2 / rho, conv ? 0 : nact, &cz, &cb); /* the converging iteration updates x only */
        RC(blas_multishift_xp(ctx, cx, cz, cb, x, p, r, o.nreal, P));
        rho = rho2;
    }
    while (!fused && !conv && k < maxiter) {
        k++;
        RC(apply_N(o, q, p, t, tmp));
        if (shifts[0] != 0.0) RC(blas_axpby(ctx, host_scalar(shifts[0]), p, host_scalar(1.0), q, o.nreal, P));
        RC(blas_redot(ctx, p, q, o.nreal, P, d + S_PQ));
        RC(fetch(ctx, S_PQ, 1));
        const double pq = h[S_PQ];
        if (!(pq > 0.0)) { brk = 1; break; }
        const double alpha = rho / pq;
        const MultiShiftCoef cx = rec.x_coef(alpha, nact);
        RC(blas_multishift_x(ctx, cx, x, p, q, r, o.nreal, P, d + (S_RHO + 1)));
        RC(fetch(ctx, (S_RHO + 1), 1));
        const double rho2 = h[(S_RHO + 1)];
        rnorm = sqrt(rho2);
        if (rnorm <= tol * bnorm) { conv = 1; break; }
        while (nact > 1 && fabs(rec.zp[nact - 1]) * rnorm <= tol * bnorm) nact--;
        MultiShiftCoef cz, cb;
        rec.p_coef(alpha, rho2 / rho, nact, &cz, &cb);
        RC(blas_multishift_p(ctx, cz, cb, p, r, o.nreal, P));
        rho = rho2;
    }
    cudaEventRecord(e1, ctx->stream);
    cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    double rt0 = 0.0;
    for (int s = 0; s < nshift && (r_true || s == 0); s++) {
        const char* xs = (const char*)x + s * o.bytes;
        RC(apply_N(o, q, xs, t, tmp));
        if (shifts[s] != 0.0) RC(blas_axpby(ctx, host_scalar(shifts[s]), xs, host_scalar(1.0), q, o.nreal, P));
        RC(blas_axpby(ctx, host_scalar(1.0), b, host_scalar(-1.0), q, o.nreal, P));
        RC(blas_norm2(ctx, q, o.nreal, P, d + S_AUX));
        RC(fetch(ctx, S_AUX, 1));
        const double rt = bnorm > 0 ? sqrt(h[S_AUX]) / bnorm : 0.0;
        if (r_true) r_true[s] = rt;
        if (s == 0) rt0 = rt;
    }
    if (stats) {
        memset(stats, 0, sizeof(*stats));
        stats->iters = k; stats->converged = conv; stats->breakdown = brk;
        stats->r_iter = bnorm > 0 ? rnorm / bnorm : 0.0;
        stats->r_true = rt0;
        stats->seconds = ms * 1e-3;
        stats->flops = 2.0 * hop_flops_per_apply_M(o) * k;
    }
    if (brk) return qcd_set_error(QCD_EBREAKDOWN, "cg_multishift: <p,(N+s)p> <= 0 or NaN at iteration %d", k);
    return conv ? QCD_OK : QCD_NOCONV;
}

int qcd_cheb_apply_multi(qcd_ctx* ctx, void* y, const void* v, int nvec, const qcd_gauge* g, double kappa, const double* coeff,
                         int degree, double scale)
{
    QCD_REQUIRE(ctx && g && y && v && coeff, "cheb_apply: NULL argument");
    QCD_REQUIRE(g->precision == 4 || g->precision == 8, "cheb_apply: needs an fp32 or fp64 gauge handle");
    QCD_REQUIRE(g->ctx == ctx, "cheb_apply: the gauge handle belongs to another ctx");
    QCD_ON_DEVICE(ctx);
    QCD_REQUIRE(degree >= 0 && scale > 0.0 && nvec >= 1, "cheb_apply: degree must be >= 0, scale > 0, nvec >= 1");
    QCD_REQUIRE((((uintptr_t)y | (uintptr_t)v) & 15u) == 0, "cheb_apply: y/v must be 16-byte aligned");
    const int P = g->precision;
    const size_t blk = (size_t)g->geo.Vh * 24 * P, full = 2 * blk, nreal = (size_t)g->geo.V * 24;
    const size_t batch = (size_t)nvec * full;
    {
        const uintptr_t a0 = (uintptr_t)y, a1 = (uintptr_t)v;
        QCD_REQUIRE(a0 + batch <= a1 || a1 + batch <= a0, "cheb_apply: y and v alias");
    }
    if (degree == 0) {
        RC(blas_copy(ctx, y, v, batch));
        return blas_axpby(ctx, host_scalar(0.0), v, host_scalar(coeff[0]), y, nreal * nvec, P);
    }
    QCD_REQUIRE(ctx->ws && ctx->ws_bytes >= 2 * batch, "cheb_apply: workspace too small (need %zu bytes)", 2 * batch);
    /* Clenshaw: b_{d+1} = b_{d+2} = 0; b_k = c_k v + 2 X b_{k+1} - b_{k+2}; y = c_0 v + X b_1 - b_2,
     * X = g5 (1 - kappa H) / scale.  b_d = c_d v needs no operator apply. */
    char* bk1 = (char*)ctx->ws;  /* b_{k+1} */
    char* bk2 = bk1 + batch;     /* b_{k+2}, overwritten by b_k */
    RC(blas_copy(ctx, bk1, v, batch));
    RC(blas_axpby(ctx, host_scalar(0.0), v, host_scalar(coeff[degree]), bk1, nreal * nvec, P));
    for (int k = degree - 1; k >= 0; k--) {
        const bool first = (k == degree - 1), last = (k == 0);
        char* out = last ? (char*)y : bk2;
        for (int p = 0; p < 2; p++) {
            HopLaunch L;
            memset(&L, 0, sizeof(L));
            L.mode = HOP_CHEB;
            L.in = bk1 + (1 - p) * blk;
            L.z = bk1 + p * blk;
            L.tm = bk2 + p * blk;
            L.v = (const char*)v + p * blk;
            L.out = out + p * blk;
            L.b = -kappa;
            L.c1 = (last ? 1.0 : 2.0) / scale;
            L.c2 = first ? 0.0 : -1.0;
            L.c3 = coeff[k];
            L.vstride = nreal;
            L.nvec = nvec;
            L.out_parity = p;
            L.dagger = 0;
            RC(hop_launch(ctx, g, L));
        }
        if (!last) { char* s = bk1; bk1 = bk2; bk2 = s; }
    }
    return QCD_OK;
}

/* out_j = D_W in_j = (1 - kappa H) in_j, or gamma5 D_W in_j, for nvec full-lattice vectors: two
 * launches of the multi-rhs kernel (one per output parity), each link fetched once per block. */
int qcd_wilson_multi(qcd_ctx* ctx, void* out, const void* in, int nvec, const qcd_gauge* g, double kappa, int gamma5)
{
    QCD_REQUIRE(ctx && g && out && in, "wilson_multi: NULL argument");
    QCD_REQUIRE(g->precision == 4 || g->precision == 8, "wilson_multi: needs an fp32 or fp64 gauge handle");
    QCD_REQUIRE(nvec >= 1, "wilson_multi: nvec must be >= 1");
    QCD_REQUIRE(g->ctx == ctx, "wilson_multi: the gauge handle belongs to another ctx");
    QCD_ON_DEVICE(ctx);
    QCD_REQUIRE((((uintptr_t)out | (uintptr_t)in) & 15u) == 0, "wilson_multi: out/in must be 16-byte aligned");
    const int P = g->precision;
    const size_t blk = (size_t)g->geo.Vh * 24 * P, nreal = (size_t)g->geo.V * 24;
    const size_t batch = (size_t)nvec * 2 * blk;
    {
        const uintptr_t a0 = (uintptr_t)out, a1 = (uintptr_t)in;
        QCD_REQUIRE(a0 + batch <= a1 || a1 + batch <= a0, "wilson_multi: out and in alias");
    }
    for (int p = 0; p < 2; p++) {
        HopLaunch L;
        memset(&L, 0, sizeof(L));
        L.mode = HOP_CHEB;
        L.in = (const char*)in + (1 - p) * blk;
        L.z = (const char*)in + p * blk;
        L.out = (char*)out + p * blk;
        L.b = -kappa;
        L.c1 = 1.0;
        L.s5 = gamma5 ? -1.0 : 1.0;
        L.vstride = nreal;
        L.nvec = nvec;
        L.out_parity = p;
        RC(hop_launch(ctx, g, L));
    }
    return QCD_OK;
}

int qcd_cheb_apply(qcd_ctx* ctx, void* y, const void* v, const qcd_gauge* g, double kappa, const double* coeff, int degree, double scale)
{
    return qcd_cheb_apply_multi(ctx, y, v, 1, g, kappa, coeff, degree, scale);
}

} /* extern "C" */
