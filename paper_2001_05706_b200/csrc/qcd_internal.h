/*
 * qcd_internal.h -- host-side structures shared by the translation units of
 * libqcd_b200.so (CUDA path only; nothing here is used by oracle/).
 *
 * Field layouts in HBM (include/qcd.h "Conventions"):
 *   spinor, one parity : [chunk][cb]            chunk = one 128-bit word
 *                        fp32: 6 x float4 (2 complex each), fp64: 12 x double2
 *   gauge              : [mu][parity][chunk][cb]
 *                        12-real: 3 float4 / 6 double2 (rows 0,1)
 *                        18-real: fp32 4 float4 + 1 float2 plane, fp64 9 double2
 *   clover (A, A^-1)   : [which][parity][chunk][cb], 72 reals = 18 float4 / 36 double2
 *                        per site: chirality block b=0,1 -> 6 real diagonal then the
 *                        15 complex strictly-lower entries, column by column.
 */
#ifndef QCD_INTERNAL_H
#define QCD_INTERNAL_H

#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/qcd.h"

struct Geom {
    int X, Y, Z, T;   /* full dims                       */
    int X2;           /* X/2                             */
    int Vh;           /* sites per parity                */
    long long V;
};

/* Solver control block, device resident: the CG update kernel takes the
 * stopping / reliable-update decision on the device and every kernel of the iteration returns at
 * once while `halt` is set, so the host can enqueue iterations ahead without a synchronisation
 * per iteration. */
struct CgCtl {
    double thresh;  /* tol * |b|                                                  */
    double delta;   /* reliable-update threshold (reading O7); 0 = pure CG        */
    double rmax;    /* max |r| since the last reliable update                     */
    double rnorm;   /* |r| after the last executed update                         */
    int halt;       /* 0 running, 1 converged, 2 reliable update due, 3 breakdown */
    int iter;       /* iterations executed                                        */
    int pad[2];
};
enum { CG_RUN = 0, CG_CONVERGED = 1, CG_UPDATE_DUE = 2, CG_BREAKDOWN = 3 };

struct qcd_ctx {
    int device;
    cudaStream_t stream;
    void* ws;
    size_t ws_bytes;
    double* d_partial;      /* block partial sums (device)                 */
    unsigned int* d_ticket; /* last-block tickets, one per reduction slot  */
    double* d_scalar;       /* device-resident CG scalars                  */
    double* h_scalar;       /* pinned host mirror                          */
    CgCtl* d_ctl;           /* solver control block (device)               */
    volatile int* h_status; /* mapped pinned host words written by the CG update kernel: [0] = iterations
                               executed, [1] = halt code; the host polls them instead of synchronising */
    int* d_status;          /* device address of h_status                  */
    double* d_hop_partial;  /* norm fused into the hop epilogue: per-block partials, then one per group of
                               HOP_NORM_GROUP blocks (grown on demand, hop_norm_scratch)               */
    unsigned int* d_hop_ticket; /* one ticket per group + one for the groups, zero between launches   */
    size_t hop_partial_cap;     /* blocks the scratch is sized for                                    */
    int max_blocks;
    int num_sms;
    long long launches;
    /* operator selected by qcd_set_operator */
    const qcd_gauge *g_hi, *g_lo;
    const qcd_clover *c_hi, *c_lo;
    double kappa, csw, delta;
    int op_parity;
    int op_set;
    /* qcd_dslash_host_batch: copy streams and events, created on first use */
    cudaStream_t s_h2d, s_d2h;
    cudaEvent_t ev_start, ev_in[2], ev_comp[2], ev_out[2];
    int pipe_ready;
};

struct qcd_gauge {
    qcd_ctx* ctx;
    Geom geo;
    int precision;    /* 4 | 8   */
    int reconstruct;  /* 12 | 18 */
    int tb;           /* +1 | -1 */
    void* data;
    size_t block_bytes; /* bytes of one (mu, parity) block */
};

struct qcd_clover {
    qcd_ctx* ctx;
    Geom geo;
    int precision;
    double kappa, csw;
    void* data;          /* A[parity 0], A[parity 1], Ainv[parity 0], Ainv[parity 1] */
    size_t block_bytes;  /* bytes of one parity block = Vh * 72 * precision          */
};

/* device scalar slots (doubles) used by the solvers */
enum { SC_RHO = 0, SC_PQ = 1, SC_RHO_NEW = 2, SC_BETA = 3, SC_TMP = 4, SC_COUNT = 16 };

int qcd_set_error(int code, const char* fmt, ...);
#define QCD_CHECK_CUDA(expr)                                                          \
    do {                                                                              \
        cudaError_t e__ = (expr);                                                     \
        if (e__ != cudaSuccess)                                                       \
            return qcd_set_error(QCD_ECUDA, "%s: %s (%s:%d)", #expr,                  \
                                 cudaGetErrorString(e__), __FILE__, __LINE__);        \
    } while (0)
/* every public entry point runs on its ctx's device whatever device the caller left current */
#define QCD_ON_DEVICE(ctx) QCD_CHECK_CUDA(cudaSetDevice((ctx)->device))
#define QCD_REQUIRE(cond, ...)                                                        \
    do {                                                                              \
        if (!(cond)) return qcd_set_error(QCD_EINVAL, __VA_ARGS__);                   \
    } while (0)

/* ---- hop launch description (hop.cu) ------------------------------------------- */
enum HopMode {
    HOP_PLAIN = 0,       /* out = H in                                            */
    HOP_XPAY = 1,        /* out = a z + b H in                                    */
    HOP_CLOVER_Z = 2,    /* out = a (A z) + b H in                                */
    HOP_CLOVER_OUT = 3,  /* out = Ainv (H in)                                     */
    HOP_CHEB = 4         /* out_j = c1 g5 (z_j + b H in_j) + c2 tm_j + c3 v_j, j < nvec */
};

struct HopLaunch {
    void* out;            /* one-parity block                                     */
    const int* halt;      /* device flag: the launch does nothing while *halt != 0 (NULL = always run) */
    double* norm_out;     /* device: receives |out|^2 (+ *norm_add), accumulated in fp64 in the epilogue (modes 1,2) */
    const double* norm_add;
    /* CG residual update fused into the epilogue (modes 1,2): with q the value this launch computes for a site,
     *   r -= (cg_num / cg_den) q ;  norm_out = |r|^2 (+ *norm_add) ;  q itself is not stored.
     * A denominator that is not > 0 makes the launch flag a breakdown and write nothing.  With cg_ctl the
     * last block counts the iteration and takes the stop / reliable-update decision (cg_decide). */
    void* cg_r;           /* one-parity block of the residual, same precision as out */
    const double* cg_num;
    const double* cg_den;
    CgCtl* cg_ctl;
    int* cg_status;
    const void* in;       /* other-parity block                                   */
    const void* z;        /* own-parity block (modes 1,2,4)                       */
    const void* tm;       /* cheb: b_{k+2}, own parity (may alias out)            */
    const void* v;        /* cheb: source vector, own parity                      */
    const void* clover;   /* A or A^-1 block of the output parity (modes 2,3)     */
    double a, b, c1, c2, c3;
    double s5;            /* cheb: factor on spin rows 2,3 of the bracket (-1 = gamma5, +1 = none; 0 reads as -1) */
    size_t vstride;       /* cheb: reals between consecutive right-hand sides     */
    int nvec;             /* cheb: number of right-hand sides                     */
    int out_parity, dagger, mode;
};

int hop_launch(qcd_ctx* ctx, const qcd_gauge* g, const HopLaunch& L);
int clover_site_apply(qcd_ctx* ctx, void* out, const void* in, const qcd_clover* c, int block); /* hop.cu: block 0,1 = A, 2,3 = A^-1 */
enum { HOP_NORM_GROUP = 64 }; /* blocks per first-level group of the fused norm's reduction */
int hop_norm_scratch(qcd_ctx* ctx, size_t nblocks); /* hop.cu: make the scratch of the fused norm hold nblocks blocks */
void solver_forget_ctx(const qcd_ctx* ctx); /* solver.cu: qcd_finalize clears the "last ctx" of qcd_cg_solve */

/* out = M in (or M^dag in): parity 2 = (A - kappa H) on the full lattice (two launches);
 * parity 0|1 = even-odd Schur operator on that parity (two launches, tmp = one parity block). */
struct OpExtra {
    const int* halt;   /* gate (see HopLaunch)                                                  */
    double* norm_out;  /* device: |out|^2 of the whole result, fused into the launch(es) writing it */
    double* norm_tmp;  /* device scratch double (full-lattice form: partial result of the first launch) */
    /* residual update fused into the launch(es) that would write `out` (see HopLaunch::cg_r): r is a field
     * shaped like out; norm_out then receives |r|^2 and out is not written */
    void* cg_r;
    const double* cg_num;
    const double* cg_den;
    CgCtl* cg_ctl;
    int* cg_status;
};
int op_apply_M(qcd_ctx* ctx, void* out, const void* in, void* tmp, const qcd_gauge* g, const qcd_clover* c,
               double kappa, int parity, int dagger, const OpExtra* ex = nullptr);

/* ---- 16-bit storage path (hop_half.cu, api.cu) ---------------------------- */
int hop_half_launch(qcd_ctx* ctx, const qcd_gauge* g, const HopLaunch& L, int out_f32);
int half_convert(qcd_ctx* ctx, void* half, void* f32, size_t Vh, int nblocks, int to_half);
/* p = a r + b p (fp32) ; ph = 16-bit copy of p */
int op_apply_M_half(qcd_ctx* ctx, void* out, int out_f32, const void* in, void* tmp, const qcd_gauge* g, const qcd_clover* c,
                    double kappa, int parity, int dagger, const int* halt = nullptr);

/* ---- blas.cu --------------------------------------------------------------------- */
/* A scalar that is either a host value or the quotient of two device doubles. */
struct DevScalar {
    double val;
    const double* num;
    const double* den;
    double sign;
};
static inline DevScalar host_scalar(double v) { DevScalar s = {v, nullptr, nullptr, 1.0}; return s; }
static inline DevScalar dev_ratio(const double* n, const double* d, double sign = 1.0)
{
    DevScalar s = {0.0, n, d, sign};
    return s;
}

/* `halt` (device, may be NULL) gates a launch: it does nothing while *halt != 0 */
int blas_axpby(qcd_ctx*, DevScalar a, const void* x, DevScalar b, void* y, size_t nreal, int prec, const int* halt = nullptr);
int blas_norm2(qcd_ctx*, const void* x, size_t nreal, int prec, double* d_out);
int blas_redot(qcd_ctx*, const void* x, const void* y, size_t nreal, int prec, double* d_out, const int* halt = nullptr);
/* x += a p; r -= a q; *d_out = |r|^2.  With ctl: skipped while ctl->halt != 0; a breakdown (the
 * denominator of `a` not > 0) sets halt = CG_BREAKDOWN and leaves x, r untouched; after the update
 * the last block counts the iteration and takes the stopping / reliable-update decision
 * (CgCtl) and mirrors (iter, halt) to the mapped host words `status`. */
int blas_cg_update(qcd_ctx*, DevScalar a, const void* p, const void* q, void* x, void* r,
                   size_t nreal, int prec, double* d_out, CgCtl* ctl = nullptr, int* status = nullptr);
/* x += a p; and, unless the solver halted in iteration `iter`, p = r + b p (see blas.cu) */
int blas_cg_xp(qcd_ctx*, DevScalar a, DevScalar b, const void* r, void* x, void* p, size_t nreal, int prec, const CgCtl* ctl, int iter);
/* y(hi) += x(lo); x = 0 */
int blas_accumulate_hi(qcd_ctx*, void* y_hi, void* x_lo, size_t nreal, size_t Vh);
/* r_hi = b - t (fp64); r_lo = (float) r_hi; *d_out = |r_hi|^2; with ctl: rmax = |r_hi|,
 * halt = CG_CONVERGED if |r_hi| <= thresh else CG_RUN */
int blas_residual_hi(qcd_ctx*, void* r_hi, void* r_lo, const void* b, const void* t, size_t nreal,
                     size_t Vh, double* d_out, CgCtl* ctl = nullptr);
/* p = a r + b p (fp32) ; ph = 16-bit copy of p (hop_half.cu) */
int half_xpay_store(qcd_ctx* ctx, DevScalar a, const void* r, DevScalar b, int p_is_zero, void* p, void* ph, size_t Vh, int nblocks,
                    const int* halt = nullptr);
/* internal-layout spinor blocks of Vh sites each (nreal = nblocks*24*Vh), layout-aware */
int blas_convert(qcd_ctx*, void* dst, int pdst, const void* src, int psrc, size_t nreal, size_t Vh);
/* multi-shift CG: ns consecutive fields of nreal reals in x and p */
enum { QCD_MAX_SHIFTS = 16 };
struct MultiShiftCoef {
    int ns;
    double alpha;
    double c[QCD_MAX_SHIFTS];
};
/* r -= alpha q ; *d_out = |r|^2 ; x_j += c[j] p_j */
int blas_multishift_xp(qcd_ctx*, const MultiShiftCoef& cx, const MultiShiftCoef& zeta, const MultiShiftCoef& beta, void* x, void* p, const void* r,
                       size_t nreal, int prec);
int blas_multishift_x(qcd_ctx*, const MultiShiftCoef& cf, void* x, const void* p, const void* q, void* r, size_t nreal,
                      int prec, double* d_out);
/* p_j = zeta.c[j] r + beta.c[j] p_j */
int blas_multishift_p(qcd_ctx*, const MultiShiftCoef& zeta, const MultiShiftCoef& beta, void* p, const void* r, size_t nreal,
                      int prec);
int blas_zero(qcd_ctx*, void* x, size_t bytes);
int blas_copy(qcd_ctx*, void* dst, const void* src, size_t bytes);

int layout_spinor_pack(qcd_ctx*, void* internal, const void* boundary, const Geom&, int prec, int unpack);
int layout_gauge_load(qcd_ctx*, const qcd_gauge* g, const void* links, int prec_in);

/* ---- clover.cu -------------------------------------------------------------------- */
int clover_build(qcd_ctx*, const qcd_gauge* g, const qcd_clover* c);
int clover_unpack(qcd_ctx*, void* dense, const qcd_clover* c, int which);

static inline size_t gauge_block_bytes(const Geom& g, int precision, int reconstruct)
{
    return (size_t)g.Vh * (size_t)reconstruct * (size_t)precision; /* precision 2: 12 int16 codes = 24 B */
}

#endif
