/*
 * api.cu -- the C ABI of include/qcd.h: handles, argument checking, layout and operator
 * entry points.  Solvers and the Chebyshev driver are in solver.cu.
 */
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "qcd_internal.h"

static thread_local char g_err[512] = "";

int qcd_set_error(int code, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

static int make_geom(const int dims[4], Geom* g)
{
    if (!dims) return qcd_set_error(QCD_EINVAL, "dims is NULL");
    for (int i = 0; i < 4; i++)
        if (dims[i] < 2 || (dims[i] & 1)) return qcd_set_error(QCD_EINVAL, "dims[%d]=%d must be even and >= 2", i, dims[i]);
    g->X = dims[0]; g->Y = dims[1]; g->Z = dims[2]; g->T = dims[3];
    g->X2 = g->X / 2;
    g->V = (long long)g->X * g->Y * g->Z * g->T;
    if (g->V / 2 > 0x3fffffffLL) return qcd_set_error(QCD_EINVAL, "lattice too large for 32-bit site indices");
    g->Vh = (int)(g->V / 2);
    return QCD_OK;
}
static bool same_dims(const Geom& g, const int dims[4])
{
    return dims && g.X == dims[0] && g.Y == dims[1] && g.Z == dims[2] && g.T == dims[3];
}
static bool aligned16(const void* p) { return p && (((uintptr_t)p) & 15u) == 0; }
static bool overlap(const void* a, const void* b, size_t bytes)
{
    const uintptr_t x = (uintptr_t)a, y = (uintptr_t)b;
    return x < y + bytes && y < x + bytes;
}

extern "C" {

const char* qcd_last_error(void) { return g_err; }
int qcd_version(void) { return 100; }

int qcd_init(int device, void* cuda_stream, qcd_ctx** out)
{
    if (!out) return qcd_set_error(QCD_EINVAL, "ctx is NULL");
    *out = nullptr;
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0)
        return qcd_set_error(QCD_ECUDA, "no CUDA device (%s); this library has no CPU fallback", cudaGetErrorString(e));
    if (device < 0 || device >= ndev) return qcd_set_error(QCD_EINVAL, "device %d out of range", device);
    QCD_CHECK_CUDA(cudaSetDevice(device));
    qcd_ctx* c = (qcd_ctx*)calloc(1, sizeof(qcd_ctx));
    if (!c) return qcd_set_error(QCD_EALLOC, "ctx alloc");
    c->device = device;
    c->stream = (cudaStream_t)cuda_stream;
    cudaDeviceProp prop;
    QCD_CHECK_CUDA(cudaGetDeviceProperties(&prop, device));
    c->num_sms = prop.multiProcessorCount;
    c->max_blocks = c->num_sms * 8; /* 8 resident 256-thread blocks per SM */
    e = cudaMalloc(&c->d_partial, sizeof(double) * (size_t)c->max_blocks);
    if (e == cudaSuccess) e = cudaMalloc(&c->d_ticket, sizeof(unsigned int) * 64);
    if (e == cudaSuccess) e = cudaMalloc(&c->d_scalar, sizeof(double) * SC_COUNT);
    if (e == cudaSuccess) e = cudaMallocHost(&c->h_scalar, sizeof(double) * SC_COUNT);
    if (e == cudaSuccess) e = cudaMalloc(&c->d_ctl, sizeof(CgCtl));
    if (e == cudaSuccess) e = cudaHostAlloc((void**)&c->h_status, 64, cudaHostAllocMapped);
    if (e == cudaSuccess) e = cudaHostGetDevicePointer((void**)&c->d_status, (void*)c->h_status, 0);
    if (e == cudaSuccess) e = cudaMemset(c->d_ticket, 0, sizeof(unsigned int) * 64);
    if (e == cudaSuccess) e = cudaMemset(c->d_scalar, 0, sizeof(double) * SC_COUNT);
    if (e == cudaSuccess) e = cudaMemset(c->d_ctl, 0, sizeof(CgCtl));
    if (e != cudaSuccess) {
        qcd_finalize(c);
        return qcd_set_error(QCD_EALLOC, "scratch allocation: %s", cudaGetErrorString(e));
    }
    *out = c;
    return QCD_OK;
}

int qcd_finalize(qcd_ctx* c)
{
    if (!c) return QCD_OK;
    solver_forget_ctx(c);
    cudaSetDevice(c->device);
    if (c->d_ctl) cudaFree(c->d_ctl);
    if (c->h_status) cudaFreeHost((void*)c->h_status);
    if (c->d_hop_partial) cudaFree(c->d_hop_partial);
    if (c->d_hop_ticket) cudaFree(c->d_hop_ticket);
    if (c->d_partial) cudaFree(c->d_partial);
    if (c->d_ticket) cudaFree(c->d_ticket);
    if (c->d_scalar) cudaFree(c->d_scalar);
    if (c->h_scalar) cudaFreeHost(c->h_scalar);
    if (c->pipe_ready) {
        cudaStreamDestroy(c->s_h2d);
        cudaStreamDestroy(c->s_d2h);
        cudaEventDestroy(c->ev_start);
        for (int b = 0; b < 2; b++) {
            cudaEventDestroy(c->ev_in[b]);
            cudaEventDestroy(c->ev_comp[b]);
            cudaEventDestroy(c->ev_out[b]);
        }
    }
    free(c);
    return QCD_OK;
}

long long qcd_launch_count(const qcd_ctx* c) { return c ? c->launches : 0; }

/* ---- gauge ------------------------------------------------------------------------ */
size_t qcd_gauge_bytes(const int dims[4], int precision, int reconstruct)
{
    Geom g;
    if (make_geom(dims, &g) != QCD_OK) return 0;
    if (precision == 2) return reconstruct == 12 ? 8 * gauge_block_bytes(g, 2, 12) : 0;
    if ((precision != 4 && precision != 8) || (reconstruct != 12 && reconstruct != 18)) return 0;
    return 8 * gauge_block_bytes(g, precision, reconstruct);
}

int qcd_gauge_load(qcd_ctx* ctx, qcd_gauge** out, const void* links, int precision_in, void* storage, const int dims[4],
                   int precision, int reconstruct, int t_boundary)
{
    QCD_REQUIRE(ctx && out, "gauge_load: NULL ctx/handle");
    *out = nullptr;
    Geom g;
    int rc = make_geom(dims, &g);
    if (rc) return rc;
    QCD_REQUIRE(precision == 2 || precision == 4 || precision == 8, "gauge_load: precision must be 2|4|8");
    QCD_REQUIRE(precision_in == 4 || precision_in == 8, "gauge_load: precision_in must be 4|8");
    QCD_REQUIRE(reconstruct == 12 || reconstruct == 18, "gauge_load: reconstruct must be 12|18");
    QCD_REQUIRE(precision != 2 || reconstruct == 12, "gauge_load: 16-bit links are stored with 12 reals");
    QCD_REQUIRE(t_boundary == 1 || t_boundary == -1, "gauge_load: t_boundary must be +1|-1");
    QCD_REQUIRE(aligned16(links) && aligned16(storage), "gauge_load: pointers must be non-NULL and 16-byte aligned");
    QCD_ON_DEVICE(ctx);
    qcd_gauge* h = (qcd_gauge*)calloc(1, sizeof(qcd_gauge));
    if (!h) return qcd_set_error(QCD_EALLOC, "gauge handle");
    h->ctx = ctx; h->geo = g; h->precision = precision; h->reconstruct = reconstruct; h->tb = t_boundary;
    h->data = storage;
    h->block_bytes = gauge_block_bytes(g, precision, reconstruct);
    rc = layout_gauge_load(ctx, h, links, precision_in);
    if (rc) { free(h); return rc; }
    *out = h;
    return QCD_OK;
}
int qcd_gauge_free(qcd_gauge* g) { free(g); return QCD_OK; }

/* ---- clover ------------------------------------------------------------------------- */
size_t qcd_clover_bytes(const int dims[4], int precision)
{
    Geom g;
    if (make_geom(dims, &g) != QCD_OK) return 0;
    if (precision == 2) return (size_t)4 * g.Vh * 148; /* 72 int16 codes + one fp32 norm per site */
    if (precision != 4 && precision != 8) return 0;
    return (size_t)4 * g.Vh * 72 * precision; /* A[2 parities] + Ainv[2 parities] */
}

int qcd_clover_build(qcd_ctx* ctx, qcd_clover** out, const qcd_gauge* g, void* storage, double kappa, double csw, int precision)
{
    QCD_REQUIRE(ctx && out && g, "clover_build: NULL argument");
    *out = nullptr;
    QCD_REQUIRE(precision == 2 || precision == 4 || precision == 8, "clover_build: precision must be 2|4|8");
    QCD_REQUIRE(g->precision != 2, "clover_build: build from an fp32 or fp64 gauge handle");
    QCD_REQUIRE(aligned16(storage), "clover_build: storage must be non-NULL and 16-byte aligned");
    QCD_REQUIRE(g->ctx == ctx, "clover_build: the gauge handle belongs to another ctx");
    QCD_ON_DEVICE(ctx);
    qcd_clover* c = (qcd_clover*)calloc(1, sizeof(qcd_clover));
    if (!c) return qcd_set_error(QCD_EALLOC, "clover handle");
    c->ctx = ctx; c->geo = g->geo; c->precision = precision; c->kappa = kappa; c->csw = csw;
    c->data = storage;
    c->block_bytes = precision == 2 ? (size_t)g->geo.Vh * 148 : (size_t)g->geo.Vh * 72 * precision;
    int rc = clover_build(ctx, g, c);
    if (rc) { free(c); return rc; }
    *out = c;
    return QCD_OK;
}
int qcd_clover_free(qcd_clover* c) { free(c); return QCD_OK; }

int qcd_clover_unpack(qcd_ctx* ctx, void* dense, const qcd_clover* c, int which)
{
    QCD_REQUIRE(ctx && c && aligned16(dense), "clover_unpack: bad argument");
    QCD_REQUIRE(which == 0 || which == 1, "clover_unpack: which must be 0|1");
    QCD_ON_DEVICE(ctx);
    return clover_unpack(ctx, dense, c, which);
}

/* ---- spinor layout ------------------------------------------------------------------ */
size_t qcd_spinor_bytes(const int dims[4], int precision)
{
    Geom g;
    if (make_geom(dims, &g) != QCD_OK) return 0;
    if (precision != 4 && precision != 8) return 0;
    return (size_t)g.V * 24 * precision;
}

static int pack_common(qcd_ctx* ctx, void* internal, const void* boundary, const int dims[4], int precision, int unpack)
{
    QCD_REQUIRE(ctx, "spinor pack: NULL ctx");
    Geom g;
    int rc = make_geom(dims, &g);
    if (rc) return rc;
    QCD_REQUIRE(precision == 4 || precision == 8, "spinor pack: precision must be 4|8");
    QCD_REQUIRE(aligned16(internal) && aligned16(boundary), "spinor pack: pointers must be non-NULL, 16-byte aligned");
    QCD_REQUIRE(!overlap(internal, boundary, (size_t)g.V * 24 * precision), "spinor pack: buffers alias");
    QCD_ON_DEVICE(ctx);
    return layout_spinor_pack(ctx, internal, boundary, g, precision, unpack);
}
int qcd_spinor_pack(qcd_ctx* ctx, void* internal, const void* boundary, const int dims[4], int precision)
{
    return pack_common(ctx, internal, boundary, dims, precision, 0);
}
int qcd_spinor_unpack(qcd_ctx* ctx, void* boundary, const void* internal, const int dims[4], int precision)
{
    return pack_common(ctx, const_cast<void*>(internal), boundary, dims, precision, 1);
}

int qcd_convert(qcd_ctx* ctx, void* dst, int pd, const void* src, int ps, const int dims[4], int nblocks)
{
    QCD_REQUIRE(ctx && aligned16(dst) && aligned16(src), "convert: bad pointer");
    QCD_REQUIRE((pd == 4 || pd == 8) && (ps == 4 || ps == 8), "convert: precision must be 4|8");
    QCD_REQUIRE(nblocks == 1 || nblocks == 2, "convert: nblocks must be 1 (one parity) or 2 (full field)");
    QCD_ON_DEVICE(ctx);
    Geom g;
    int rc = make_geom(dims, &g);
    if (rc) return rc;
    return blas_convert(ctx, dst, pd, src, ps, (size_t)nblocks * g.Vh * 24, (size_t)g.Vh);
}

/* ---- workspace ------------------------------------------------------------------------ */
size_t qcd_workspace_bytes(const int dims[4], int precision)
{
    Geom g;
    if (make_geom(dims, &g) != QCD_OK) return 0;
    if (precision != 4 && precision != 8) return 0;
    /* pure CG: r,p,q,t,tmp (5); mixed CG: 4 fp64 + 6 fp32 = 7 fp64-equivalents; Chebyshev: 2 */
    return (size_t)8 * g.V * 24 * precision;
}
int qcd_set_workspace(qcd_ctx* ctx, void* ws, size_t bytes)
{
    QCD_REQUIRE(ctx, "set_workspace: NULL ctx");
    QCD_REQUIRE(ws == nullptr || aligned16(ws), "set_workspace: misaligned");
    ctx->ws = ws;
    ctx->ws_bytes = ws ? bytes : 0;
    return QCD_OK;
}

/* ---- the stencil ------------------------------------------------------------------------ */
int qcd_hop_xpay(void* out, const void* in, const void* z, double a, double b, const qcd_gauge* g, int out_parity, int dagger)
{
    QCD_REQUIRE(g && g->ctx, "hop: NULL gauge");
    QCD_REQUIRE(g->precision != 2, "hop: 16-bit gauge handle: use qcd_dslash_half");
    const size_t bytes = (size_t)g->geo.Vh * 24 * g->precision;
    QCD_REQUIRE(aligned16(out) && aligned16(in), "hop: pointers must be non-NULL, 16-byte aligned");
    QCD_REQUIRE(!overlap(out, in, bytes), "hop: in and out alias");
    QCD_REQUIRE(out_parity == 0 || out_parity == 1, "hop: out_parity must be 0|1");
    QCD_ON_DEVICE(g->ctx);
    HopLaunch L;
    memset(&L, 0, sizeof(L));
    L.out = out; L.in = in; L.out_parity = out_parity; L.dagger = dagger ? 1 : 0;
    if (z) {
        QCD_REQUIRE(aligned16(z) && !overlap(z, in, bytes), "hop_xpay: z misaligned or aliases in");
        L.mode = HOP_XPAY; L.z = z; L.a = a; L.b = b;
    } else {
        L.mode = HOP_PLAIN;
    }
    return hop_launch(g->ctx, g, L);
}

int qcd_hop(void* out, const void* in, const qcd_gauge* g, int out_parity, int dagger, const int dims[4], int precision)
{
    QCD_REQUIRE(g, "hop: NULL gauge");
    QCD_REQUIRE(same_dims(g->geo, dims) && precision == g->precision, "hop: dims/precision do not match the gauge handle");
    return qcd_hop_xpay(out, in, nullptr, 0.0, 0.0, g, out_parity, dagger);
}

} /* extern "C" */

/* out_p = A_pp in_p - kappa H_{p,pb} in_pb for both parities (full lattice) */
static int apply_full(qcd_ctx* ctx, void* out, const void* in, const qcd_gauge* g, const qcd_clover* c, double kappa, int dagger,
                      const OpExtra* ex)
{
    const size_t blk = (size_t)g->geo.Vh * 24 * g->precision;
    for (int p = 0; p < 2; p++) {
        HopLaunch L;
        memset(&L, 0, sizeof(L));
        if (ex) {
            L.halt = ex->halt;
            if (ex->norm_out) { /* |out|^2 = even block (into norm_tmp) + odd block */
                L.norm_out = p == 0 ? ex->norm_tmp : ex->norm_out;
                L.norm_add = p == 0 ? nullptr : ex->norm_tmp;
            }
            if (ex->cg_r) { /* each launch updates its parity block of r; the second one decides */
                L.cg_r = (char*)ex->cg_r + p * blk;
                L.cg_num = ex->cg_num; L.cg_den = ex->cg_den;
                L.cg_ctl = p == 1 ? ex->cg_ctl : nullptr;
                L.cg_status = p == 1 ? ex->cg_status : nullptr;
            }
        }
        L.out = (char*)out + p * blk;
        L.in = (const char*)in + (1 - p) * blk;
        L.z = (const char*)in + p * blk;
        L.a = 1.0; L.b = -kappa;
        L.out_parity = p; L.dagger = dagger;
        if (c) { L.mode = HOP_CLOVER_Z; L.clover = (const char*)c->data + p * c->block_bytes; }
        else L.mode = HOP_XPAY;
        int rc = hop_launch(ctx, g, L);
        if (rc) return rc;
    }
    return QCD_OK;
}

/* even-odd Schur operator (reading O5):
 *   tmp_pb = Ainv_pb H_{pb,p} in_p ;  out_p = A_pp in_p - kappa^2 H_{p,pb} tmp_pb */
static int apply_eo(qcd_ctx* ctx, void* out, const void* in, void* tmp, const qcd_gauge* g, const qcd_clover* c, double kappa, int p,
                    int dagger, const OpExtra* ex)
{
    HopLaunch L;
    memset(&L, 0, sizeof(L));
    if (ex) L.halt = ex->halt;
    L.out = tmp; L.in = in; L.out_parity = 1 - p; L.dagger = dagger;
    if (c) { L.mode = HOP_CLOVER_OUT; L.clover = (const char*)c->data + (2 + (1 - p)) * c->block_bytes; }
    else L.mode = HOP_PLAIN;
    int rc = hop_launch(ctx, g, L);
    if (rc) return rc;
    memset(&L, 0, sizeof(L));
    if (ex) {
        L.halt = ex->halt; L.norm_out = ex->norm_out;
        L.cg_r = ex->cg_r; L.cg_num = ex->cg_num; L.cg_den = ex->cg_den; L.cg_ctl = ex->cg_ctl; L.cg_status = ex->cg_status;
    }
    L.out = out; L.in = tmp; L.z = in; L.a = 1.0; L.b = -kappa * kappa; L.out_parity = p; L.dagger = dagger;
    if (c) { L.mode = HOP_CLOVER_Z; L.clover = (const char*)c->data + p * c->block_bytes; }
    else L.mode = HOP_XPAY;
    return hop_launch(ctx, g, L);
}

int op_apply_M(qcd_ctx* ctx, void* out, const void* in, void* tmp, const qcd_gauge* g, const qcd_clover* c, double kappa, int parity,
               int dagger, const OpExtra* ex)
{
    if (parity == QCD_PARITY_FULL) return apply_full(ctx, out, in, g, c, kappa, dagger, ex);
    return apply_eo(ctx, out, in, tmp, g, c, kappa, parity, dagger, ex);
}

extern "C" {

int qcd_dslash_ex(void* out, const void* in, const qcd_gauge* g, const qcd_clover* c, double kappa, double csw, int parity, int flags,
                  void* tmp)
{
    QCD_REQUIRE(g && g->ctx, "dslash: NULL gauge");
    QCD_REQUIRE(g->precision != 2, "dslash: 16-bit gauge handle: use qcd_dslash_half");
    qcd_ctx* ctx = g->ctx;
    QCD_REQUIRE(parity == 0 || parity == 1 || parity == 2, "dslash: parity must be 0|1|2");
    QCD_ON_DEVICE(ctx);
    QCD_REQUIRE(aligned16(out) && aligned16(in), "dslash: pointers must be non-NULL, 16-byte aligned");
    const size_t blk = (size_t)g->geo.Vh * 24 * g->precision;
    const size_t bytes = parity == 2 ? 2 * blk : blk;
    QCD_REQUIRE(!overlap(out, in, bytes), "dslash: in and out alias");
    if (c) {
        QCD_REQUIRE(c->precision == g->precision && c->geo.V == g->geo.V, "dslash: clover does not match gauge");
        QCD_REQUIRE(c->kappa == kappa && c->csw == csw, "dslash: kappa/csw differ from the values the clover was built with");
    }
    if (parity != 2) {
        if (!tmp) {
            QCD_REQUIRE(ctx->ws && ctx->ws_bytes >= blk, "dslash: parity 0|1 needs a temporary (qcd_set_workspace or tmp)");
            tmp = ctx->ws;
        }
        QCD_REQUIRE(aligned16(tmp) && !overlap(tmp, in, blk) && !overlap(tmp, out, blk), "dslash: tmp misaligned or aliased");
    }
    return op_apply_M(ctx, out, in, tmp, g, c, kappa, parity, (flags & QCD_DAGGER) ? 1 : 0);
}

int qcd_dslash(void* out, const void* in, const qcd_gauge* g, const qcd_clover* c, double kappa, double csw, int parity,
               const int dims[4], int precision)
{
    QCD_REQUIRE(g, "dslash: NULL gauge");
    QCD_REQUIRE(same_dims(g->geo, dims) && precision == g->precision, "dslash: dims/precision do not match the gauge handle");
    return qcd_dslash_ex(out, in, g, c, kappa, csw, parity, 0, nullptr);
}

/* ---- 16-bit storage (reading H1) ---------------------------------------------- */
} /* extern "C" */

/* out = M in with every streamed field in 16 bits; in: 16-bit field; out: 16-bit or fp32 */
int op_apply_M_half(qcd_ctx* ctx, void* out, int out_f32, const void* in, void* tmp, const qcd_gauge* g, const qcd_clover* c,
                    double kappa, int parity, int dagger, const int* halt)
{
    const size_t hblk = (size_t)g->geo.Vh * 52, oblk = out_f32 ? (size_t)g->geo.Vh * 96 : hblk;
    HopLaunch L;
    if (parity == QCD_PARITY_FULL) {
        for (int p = 0; p < 2; p++) {
            memset(&L, 0, sizeof(L));
            L.halt = halt;
            L.out = (char*)out + p * oblk;
            L.in = (const char*)in + (1 - p) * hblk;
            L.z = (const char*)in + p * hblk;
            L.a = 1.0; L.b = -kappa; L.out_parity = p; L.dagger = dagger;
            if (c) { L.mode = HOP_CLOVER_Z; L.clover = (const char*)c->data + p * c->block_bytes; }
            else L.mode = HOP_XPAY;
            int rc = hop_half_launch(ctx, g, L, out_f32);
            if (rc) return rc;
        }
        return QCD_OK;
    }
    const int p = parity;
    memset(&L, 0, sizeof(L));
    L.halt = halt;
    L.out = tmp; L.in = in; L.out_parity = 1 - p; L.dagger = dagger;
    if (c) { L.mode = HOP_CLOVER_OUT; L.clover = (const char*)c->data + (2 + (1 - p)) * c->block_bytes; }
    else L.mode = HOP_PLAIN;
    int rc = hop_half_launch(ctx, g, L, 0);
    if (rc) return rc;
    memset(&L, 0, sizeof(L));
    L.halt = halt;
    L.out = out; L.in = tmp; L.z = in; L.a = 1.0; L.b = -kappa * kappa; L.out_parity = p; L.dagger = dagger;
    if (c) { L.mode = HOP_CLOVER_Z; L.clover = (const char*)c->data + p * c->block_bytes; }
    else L.mode = HOP_XPAY;
    return hop_half_launch(ctx, g, L, out_f32);
}

extern "C" {

size_t qcd_half_spinor_bytes(const int dims[4])
{
    Geom g;
    if (make_geom(dims, &g) != QCD_OK) return 0;
    return (size_t)g.V * 52;
}

int qcd_spinor_to_half(qcd_ctx* ctx, void* half, const void* f32, const int dims[4], int nblocks)
{
    QCD_REQUIRE(ctx && aligned16(half) && aligned16(f32), "spinor_to_half: bad pointer");
    QCD_REQUIRE(nblocks == 1 || nblocks == 2, "spinor_to_half: nblocks must be 1|2");
    QCD_ON_DEVICE(ctx);
    Geom g;
    int rc = make_geom(dims, &g);
    if (rc) return rc;
    return half_convert(ctx, half, const_cast<void*>(f32), (size_t)g.Vh, nblocks, 1);
}

int qcd_spinor_from_half(qcd_ctx* ctx, void* f32, const void* half, const int dims[4], int nblocks)
{
    QCD_REQUIRE(ctx && aligned16(half) && aligned16(f32), "spinor_from_half: bad pointer");
    QCD_REQUIRE(nblocks == 1 || nblocks == 2, "spinor_from_half: nblocks must be 1|2");
    QCD_ON_DEVICE(ctx);
    Geom g;
    int rc = make_geom(dims, &g);
    if (rc) return rc;
    return half_convert(ctx, const_cast<void*>(half), f32, (size_t)g.Vh, nblocks, 0);
}

int qcd_dslash_half(void* out, int out_precision, const void* in_half, const qcd_gauge* g, const qcd_clover* c, double kappa, double csw,
                    int parity, int flags, void* tmp_half)
{
    QCD_REQUIRE(g && g->ctx && g->precision == 2, "dslash_half: needs a 16-bit gauge handle");
    QCD_REQUIRE(out_precision == 2 || out_precision == 4, "dslash_half: out_precision must be 2|4");
    QCD_REQUIRE(parity == 0 || parity == 1 || parity == 2, "dslash_half: parity must be 0|1|2");
    QCD_ON_DEVICE(g->ctx);
    QCD_REQUIRE(aligned16(out) && aligned16(in_half) && out != in_half, "dslash_half: bad in/out pointer");
    if (c) {
        QCD_REQUIRE(c->precision == 2 && c->geo.V == g->geo.V, "dslash_half: needs a 16-bit clover handle of the same lattice");
        QCD_REQUIRE(c->kappa == kappa && c->csw == csw, "dslash_half: kappa/csw differ from the values the clover was built with");
    }
    if (parity != 2) QCD_REQUIRE(aligned16(tmp_half) && tmp_half != out && tmp_half != in_half, "dslash_half: parity 0|1 needs tmp_half");
    return op_apply_M_half(g->ctx, out, out_precision == 4, in_half, tmp_half, g, c, kappa, parity, (flags & QCD_DAGGER) ? 1 : 0);
}

/* ---- BLAS ------------------------------------------------------------------------------ */
static int blas_args(qcd_ctx* ctx, const void* x, const void* y, size_t nreal, int precision)
{
    QCD_REQUIRE(ctx, "blas: NULL ctx");
    QCD_REQUIRE(precision == 4 || precision == 8, "blas: precision must be 4|8");
    QCD_REQUIRE(nreal % 4 == 0, "blas: nreal must be a multiple of 4");
    QCD_REQUIRE(aligned16(x) && aligned16(y), "blas: pointers must be non-NULL, 16-byte aligned");
    QCD_ON_DEVICE(ctx);
    return QCD_OK;
}
static int fetch_scalar(qcd_ctx* ctx, int slot, double* result)
{
    QCD_CHECK_CUDA(cudaMemcpyAsync(ctx->h_scalar + slot, ctx->d_scalar + slot, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    QCD_CHECK_CUDA(cudaStreamSynchronize(ctx->stream));
    *result = ctx->h_scalar[slot];
    return QCD_OK;
}

int qcd_axpy(qcd_ctx* ctx, double a, const void* x, void* y, size_t nreal, int precision)
{
    int rc = blas_args(ctx, x, y, nreal, precision);
    if (rc) return rc;
    return blas_axpby(ctx, host_scalar(a), x, host_scalar(1.0), y, nreal, precision);
}
int qcd_xpay(qcd_ctx* ctx, const void* x, double a, void* y, size_t nreal, int precision)
{
    int rc = blas_args(ctx, x, y, nreal, precision);
    if (rc) return rc;
    return blas_axpby(ctx, host_scalar(1.0), x, host_scalar(a), y, nreal, precision);
}
int qcd_axpby(qcd_ctx* ctx, double a, const void* x, double b, void* y, size_t nreal, int precision)
{
    int rc = blas_args(ctx, x, y, nreal, precision);
    if (rc) return rc;
    return blas_axpby(ctx, host_scalar(a), x, host_scalar(b), y, nreal, precision);
}
int qcd_norm2(qcd_ctx* ctx, const void* x, size_t nreal, int precision, double* result)
{
    int rc = blas_args(ctx, x, x, nreal, precision);
    if (rc) return rc;
    rc = blas_norm2(ctx, x, nreal, precision, ctx->d_scalar + SC_TMP);
    if (rc || !result) return rc;
    return fetch_scalar(ctx, SC_TMP, result);
}
int qcd_redot(qcd_ctx* ctx, const void* x, const void* y, size_t nreal, int precision, double* result)
{
    int rc = blas_args(ctx, x, y, nreal, precision);
    if (rc) return rc;
    rc = blas_redot(ctx, x, y, nreal, precision, ctx->d_scalar + SC_TMP);
    if (rc || !result) return rc;
    return fetch_scalar(ctx, SC_TMP, result);
}
int qcd_cg_update(qcd_ctx* ctx, double a, const void* p, const void* q, void* x, void* r, size_t nreal, int precision, double* result)
{
    int rc = blas_args(ctx, p, q, nreal, precision);
    if (rc) return rc;
    rc = blas_args(ctx, x, r, nreal, precision);
    if (rc) return rc;
    rc = blas_cg_update(ctx, host_scalar(a), p, q, x, r, nreal, precision, ctx->d_scalar + SC_TMP);
    if (rc || !result) return rc;
    return fetch_scalar(ctx, SC_TMP, result);
}

/* ---- host-buffer end-to-end path ----------------------------------------------------------- */
int qcd_hop_host(qcd_ctx* ctx, void* out_host, const void* in_host, const qcd_gauge* g, int out_parity, int dagger)
{
    QCD_REQUIRE(ctx && g && out_host && in_host, "hop_host: NULL argument");
    QCD_ON_DEVICE(ctx);
    const size_t blk = (size_t)g->geo.Vh * 24 * g->precision;
    QCD_REQUIRE(ctx->ws && ctx->ws_bytes >= 2 * blk, "hop_host: workspace too small (qcd_set_workspace)");
    char* d_in = (char*)ctx->ws;
    char* d_out = d_in + blk;
    QCD_CHECK_CUDA(cudaMemcpyAsync(d_in, in_host, blk, cudaMemcpyHostToDevice, ctx->stream));
    int rc = qcd_hop_xpay(d_out, d_in, nullptr, 0.0, 0.0, g, out_parity, dagger);
    if (rc) return rc;
    QCD_CHECK_CUDA(cudaMemcpyAsync(out_host, d_out, blk, cudaMemcpyDeviceToHost, ctx->stream));
    QCD_CHECK_CUDA(cudaStreamSynchronize(ctx->stream));
    return QCD_OK;
}

int qcd_dslash_host(qcd_ctx* ctx, void* out_host, const void* in_host, const qcd_gauge* g, const qcd_clover* c, double kappa,
                    double csw, int parity, int flags)
{
    QCD_REQUIRE(ctx && g && out_host && in_host, "dslash_host: NULL argument");
    QCD_REQUIRE(parity == 0 || parity == 1 || parity == 2, "dslash_host: parity must be 0|1|2");
    QCD_ON_DEVICE(ctx);
    const size_t blk = (size_t)g->geo.Vh * 24 * g->precision;
    const size_t bytes = parity == 2 ? 2 * blk : blk;
    QCD_REQUIRE(ctx->ws && ctx->ws_bytes >= 2 * bytes + blk, "dslash_host: workspace too small (qcd_set_workspace)");
    char* d_in = (char*)ctx->ws;
    char* d_out = d_in + bytes;
    char* d_tmp = d_out + bytes;
    QCD_CHECK_CUDA(cudaMemcpyAsync(d_in, in_host, bytes, cudaMemcpyHostToDevice, ctx->stream));
    int rc = qcd_dslash_ex(d_out, d_in, g, c, kappa, csw, parity, flags, d_tmp);
    if (rc) return rc;
    QCD_CHECK_CUDA(cudaMemcpyAsync(out_host, d_out, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    QCD_CHECK_CUDA(cudaStreamSynchronize(ctx->stream));
    return QCD_OK;
}

/* nvec host vectors through the operator as a three-stage pipeline: H2D of vector i+1, the
 * operator on vector i and D2H of vector i-1 run concurrently (PCIe is full duplex), on two
 * copy streams of the ctx and the ctx stream, with double-buffered device input / output. */
int qcd_dslash_host_batch(qcd_ctx* ctx, void* out_host, const void* in_host, int nvec, size_t out_stride, size_t in_stride,
                          const qcd_gauge* g, const qcd_clover* c, double kappa, double csw, int parity, int flags)
{
    QCD_REQUIRE(ctx && g && out_host && in_host && nvec >= 0, "dslash_host_batch: NULL argument or nvec < 0");
    QCD_REQUIRE(parity == 0 || parity == 1 || parity == 2, "dslash_host_batch: parity must be 0|1|2");
    QCD_ON_DEVICE(ctx);
    const size_t blk = (size_t)g->geo.Vh * 24 * g->precision;
    const size_t bytes = parity == 2 ? 2 * blk : blk;
    QCD_REQUIRE(out_stride == 0 || out_stride >= bytes, "dslash_host_batch: out_stride smaller than a vector");
    QCD_REQUIRE(in_stride == 0 || in_stride >= bytes, "dslash_host_batch: in_stride smaller than a vector");
    QCD_REQUIRE(ctx->ws && ctx->ws_bytes >= 4 * bytes + blk, "dslash_host_batch: workspace too small (need 4 fields + one parity block)");
    if (!ctx->pipe_ready) {
        QCD_CHECK_CUDA(cudaStreamCreateWithFlags(&ctx->s_h2d, cudaStreamNonBlocking));
        QCD_CHECK_CUDA(cudaStreamCreateWithFlags(&ctx->s_d2h, cudaStreamNonBlocking));
        QCD_CHECK_CUDA(cudaEventCreateWithFlags(&ctx->ev_start, cudaEventDisableTiming));
        for (int b = 0; b < 2; b++) {
            QCD_CHECK_CUDA(cudaEventCreateWithFlags(&ctx->ev_in[b], cudaEventDisableTiming));
            QCD_CHECK_CUDA(cudaEventCreateWithFlags(&ctx->ev_comp[b], cudaEventDisableTiming));
            QCD_CHECK_CUDA(cudaEventCreateWithFlags(&ctx->ev_out[b], cudaEventDisableTiming));
        }
        ctx->pipe_ready = 1;
    }
    char* w = (char*)ctx->ws;
    char* d_in[2] = {w, w + bytes};
    char* d_out[2] = {w + 2 * bytes, w + 3 * bytes};
    char* d_tmp = w + 4 * bytes;
    /* the copy streams start after whatever the ctx stream was doing with the workspace */
    QCD_CHECK_CUDA(cudaEventRecord(ctx->ev_start, ctx->stream));
    QCD_CHECK_CUDA(cudaStreamWaitEvent(ctx->s_h2d, ctx->ev_start, 0));
    QCD_CHECK_CUDA(cudaStreamWaitEvent(ctx->s_d2h, ctx->ev_start, 0));
    for (int i = 0; i < nvec; i++) {
        const int b = i & 1;
        /* H2D: the input buffer is free once the operator on vector i-2 has run */
        if (i >= 2) QCD_CHECK_CUDA(cudaStreamWaitEvent(ctx->s_h2d, ctx->ev_comp[b], 0));
        QCD_CHECK_CUDA(cudaMemcpyAsync(d_in[b], (const char*)in_host + (size_t)i * in_stride, bytes, cudaMemcpyHostToDevice, ctx->s_h2d));
        QCD_CHECK_CUDA(cudaEventRecord(ctx->ev_in[b], ctx->s_h2d));
        /* operator: needs the input, and the output buffer drained by the D2H of vector i-2 */
        QCD_CHECK_CUDA(cudaStreamWaitEvent(ctx->stream, ctx->ev_in[b], 0));
        if (i >= 2) QCD_CHECK_CUDA(cudaStreamWaitEvent(ctx->stream, ctx->ev_out[b], 0));
        int rc = qcd_dslash_ex(d_out[b], d_in[b], g, c, kappa, csw, parity, flags, d_tmp);
        if (rc) return rc;
        QCD_CHECK_CUDA(cudaEventRecord(ctx->ev_comp[b], ctx->stream));
        /* D2H */
        QCD_CHECK_CUDA(cudaStreamWaitEvent(ctx->s_d2h, ctx->ev_comp[b], 0));
        QCD_CHECK_CUDA(cudaMemcpyAsync((char*)out_host + (size_t)i * out_stride, d_out[b], bytes, cudaMemcpyDeviceToHost, ctx->s_d2h));
        QCD_CHECK_CUDA(cudaEventRecord(ctx->ev_out[b], ctx->s_d2h));
    }
    QCD_CHECK_CUDA(cudaStreamSynchronize(ctx->s_d2h));
    QCD_CHECK_CUDA(cudaStreamSynchronize(ctx->stream));
    return QCD_OK;
}

} /* extern "C" */
