/*
 * qcd.h -- C ABI of libqcd_b200.so: Wilson / Wilson-clover Dslash, fused BLAS-1,
 * CG on M^dag M, reliable-update mixed CG and a Chebyshev driver, as hand-written
 * sm_100a CUDA kernels.
 *
 * Source of the operations.  The paper (arXiv 2001.05706, /root/reference/PAPER.md)
 * prints no equation; it names the hot path "the D-slash" (Table 2
 * caption, sec. 4), run in single precision with SU(3) links
 * "suppressed to 12 real numbers to save the memory bandwidth",
 * vector operations / reductions as separate kernels (sec. 3) and the
 * mixed-precision Krylov solvers of its ref. [1].  The formula is the
 * one in BASELINE.json north_star,
 *   D psi(x) = psi(x) - kappa sum_mu [ (1-gamma_mu) U_mu(x) psi(x+mu)
 *                                    + (1+gamma_mu) U_mu(x-mu)^dag psi(x-mu) ],
 * with the readings listed in DESIGN.md ("Readings", S1..S23 / O1..O8).
 *
 * Conventions
 *  - Every field pointer is a DEVICE pointer owned by the caller, 16-byte aligned.
 *    The library never allocates field-sized memory; handles are small host structs.
 *    (qcd_*_host entry points take HOST pointers and say so.)
 *  - dims = {X,Y,Z,T}, all even and >= 2.  precision = bytes per real: 4 or 8 (2 = the
 *    16-bit storage of the low-precision operator, where a function says so).
 *  - Boundary (user) layouts, real type = precision:
 *      gauge  [t][z][y][x][mu=0..3 (x,y,z,t)][row][col][re,im]
 *      spinor [t][z][y][x][spin 0..3][colour 0..2][re,im]
 *  - Internal spinor layout (what qcd_hop / qcd_dslash / qcd_cg_solve take):
 *      full field = even-parity block then odd-parity block; one parity block =
 *      [chunk][cb], chunk = one 128-bit word (fp32: 2 complex, 6 chunks; fp64: 1
 *      complex, 12 chunks), complex index = spin*3+colour, cb = checkerboard index
 *      (lexicographic site index >> 1), parity = (x+y+z+t)&1.
 *  - All work is enqueued on the stream given to qcd_init.  Calls that return host
 *    scalars (reductions, solvers) synchronise that stream; the others do not.
 *  - Return: 0 = QCD_OK; < 0 error; > 0 soft status.  No exceptions, no aborts, no
 *    printing.  qcd_last_error() returns text for the last error of this thread.
 *  - There is no CPU fallback anywhere: without a CUDA device every compute call
 *    returns QCD_ECUDA.
 *  - Every entry point runs on the device of its ctx (it calls cudaSetDevice).
 *  - Environment (read at call time, for experiments; none changes a result beyond rounding order):
 *      QCD_CG_RUNAHEAD=n  iterations the CG drivers may enqueue ahead of the device (default 0; any n gives
 *                         bit-identical solves, the kernels enqueued past the stopping iteration skip themselves)
 *      QCD_MRHS_TILE=1    multi-right-hand-side hop: opt into the shared-memory tile kernel (slower on B200,
 *                         DESIGN.md section 6); QCD_MRHS_VARIANT=40|41|31|32 picks its staging variant
 *      QCD_PDL=0          launch every kernel fully serialised; default: programmatic stream serialisation
 *                         (the next launch places its blocks while the previous one drains, and waits on the
 *                         device for its completion before it reads anything); same results
 *      QCD_TRACE=1        the mixed solver prints its reliable updates to stderr
 */
#ifndef QCD_B200_H
#define QCD_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    QCD_OK = 0,
    QCD_NOCONV = 1,      /* maxiter reached; x still holds the last iterate          */
    QCD_EINVAL = -1,     /* bad argument (null / misaligned / aliased / odd dims ...) */
    QCD_EALLOC = -2,     /* small host or device scratch allocation failed           */
    QCD_ECUDA = -3,      /* CUDA runtime error (text in qcd_last_error)              */
    QCD_EBREAKDOWN = -4  /* CG breakdown: <p,Np> <= 0 or NaN; x holds the last iterate
                            before the failing update (nothing is written by it)          */
};

enum { QCD_DAGGER = 1 };                       /* flags for qcd_dslash_ex */
enum { QCD_PARITY_EVEN = 0, QCD_PARITY_ODD = 1, QCD_PARITY_FULL = 2 };

typedef struct qcd_ctx qcd_ctx;
typedef struct qcd_gauge qcd_gauge;
typedef struct qcd_clover qcd_clover;

typedef struct {
    int iters;             /* number of (low-precision) N = M^dag M applies          */
    int reliable_updates;  /* mixed CG only                                          */
    int converged;         /* 1 if |r| <= tol |b| was reached                        */
    int breakdown;
    double r_iter;         /* iterated (mixed: last fp64-recomputed) residual / |b|  */
    double r_true;         /* |b - N x| / |b| in the high precision.  Pure CG: recomputed from
                              scratch after the loop.  Mixed CG: the fp64 residual b - N_hi y of
                              the reliable update that declared convergence (it IS the residual
                              of the returned y, computed from scratch by that update); recomputed
                              only on the other exits (maxiter, breakdown)                   */
    double seconds;        /* device time of the solve loop (CUDA events)            */
    double flops;          /* nominal: 1320/site hop, +504 clover; BLAS uncounted    */
    double bytes;          /* compulsory bytes moved by hop + BLAS kernels           */
} qcd_stats;

const char* qcd_last_error(void);
int qcd_version(void);

/* device: CUDA ordinal.  cuda_stream: a cudaStream_t (NULL = default stream). */
int qcd_init(int device, void* cuda_stream, qcd_ctx** ctx);
int qcd_finalize(qcd_ctx* ctx);

/* ---- gauge field (PAPER.md:143 12-real storage) -----------------
 * qcd_gauge_load reorders `links` (DEVICE, boundary layout, real = precision_in)
 * into the checkerboarded SoA layout inside `storage` (DEVICE, caller-owned,
 * qcd_gauge_bytes(dims, precision, reconstruct) bytes), converting precision if
 * precision_in != precision.  reconstruct = 18 keeps all 9 complex; 12 keeps rows
 * 0,1 and the kernels rebuild row 2 = conj(row0 x row1).  t_boundary = -1
 * antiperiodic / +1 periodic in t: it is recorded in the handle and applied to the
 * spinor hop, never folded into the stored links (reading S4).
 * The handle keeps pointers into `storage`; qcd_gauge_free frees only the handle. */
size_t qcd_gauge_bytes(const int dims[4], int precision, int reconstruct);
int qcd_gauge_load(qcd_ctx* ctx, qcd_gauge** g, const void* links, int precision_in,
                   void* storage, const int dims[4], int precision, int reconstruct,
                   int t_boundary);
int qcd_gauge_free(qcd_gauge* g);

/* ---- clover term (readings O3, S9, S10) ----------------------
 * Builds, from the links of `g`, Fhat_munu = (Q - Q^dag)/8 over the 4 plaquette
 * leaves, A(x) = 1 + kappa*csw*sum_{mu<nu} i sigma_munu (x) Fhat_munu(x) as two
 * Hermitian 6x6 chiral blocks (2 x (6 real diag + 15 complex) = 72 reals/site) and
 * A^-1; arithmetic in fp64, stored in `precision`.  storage: DEVICE,
 * qcd_clover_bytes(dims, precision) bytes (A then A^-1).  A^-1 is taken block by block
 * through A = L D L^dag without pivoting (A is positive definite for physical kappa*csw);
 * QCD_EBREAKDOWN if a block has a vanishing or non-finite pivot (the fields are then
 * not to be used). */
size_t qcd_clover_bytes(const int dims[4], int precision);
int qcd_clover_build(qcd_ctx* ctx, qcd_clover** c, const qcd_gauge* g, void* storage,
                     double kappa, double csw, int precision);
int qcd_clover_free(qcd_clover* c);
/* Debug / parity: expand A (which=0) or A^-1 (which=1) to boundary-order dense
 * [t][z][y][x][12][12][re,im] fp64 (DEVICE, V*288 doubles). */
int qcd_clover_unpack(qcd_ctx* ctx, void* dense, const qcd_clover* c, int which);
/* out = A in (inverse = 0) or A^-1 in (inverse = 1) on the sites of one parity (SURVEY 8(a) a7 as a
 * stand-alone, site-local step): in/out one-parity blocks in the handle's precision (4|8), out == in allowed. */
int qcd_clover_apply(qcd_ctx* ctx, void* out, const void* in, const qcd_clover* c, int inverse, int parity);

/* ---- spinor layout conversion (boundary <-> internal, both DEVICE) ---------------- */
size_t qcd_spinor_bytes(const int dims[4], int precision);   /* full lattice */
int qcd_spinor_pack(qcd_ctx* ctx, void* internal, const void* boundary, const int dims[4],
                    int precision);
int qcd_spinor_unpack(qcd_ctx* ctx, void* boundary, const void* internal, const int dims[4],
                      int precision);
/* precision conversion of internal-layout spinor blocks: nblocks = 1 (one parity) or 2
 * (full field).  Layout-aware: a 128-bit chunk holds 2 complex in fp32 and 1 in fp64, so
 * fp32 chunk c of site cb maps to the fp64 chunks 2c, 2c+1 of that site. */
int qcd_convert(qcd_ctx* ctx, void* dst, int precision_dst, const void* src, int precision_src,
                const int dims[4], int nblocks);

/* ---- the stencil (north_star formula) --------------------------
 * qcd_hop: raw single-parity hopping term, the kernel the 1320 flop/site figure is
 * for:  out_p = H_{p,1-p} in_{1-p}   (dagger: H^dag, projector signs swapped).
 * `out`, `in`: ONE-parity internal blocks (Vh*24 reals), must not alias.
 * qcd_hop_xpay: out_p = a * z_p + b * H_{p,1-p} in_{1-p}  (z may alias out). */
int qcd_hop(void* out, const void* in, const qcd_gauge* g, int out_parity, int dagger,
            const int dims[4], int precision);
int qcd_hop_xpay(void* out, const void* in, const void* z, double a, double b,
                 const qcd_gauge* g, int out_parity, int dagger);

/* qcd_dslash (north_star signature):
 *   parity = 2: full lattice, out = (A - kappa H) in; in/out = full internal fields
 *               (A = 1 when clover == NULL);
 *   parity = 0|1: even-odd preconditioned operator on that parity (reading O5),
 *               out_p = A_pp in_p - kappa^2 H_{p,pb} A^-1_{pb,pb} H_{pb,p} in_p,
 *               in/out = one-parity blocks.  Needs a Vh*24-real temporary: use
 *               qcd_dslash_ex with tmp, or qcd_dslash allocates nothing and returns
 *               QCD_EINVAL if the ctx has no workspace set (qcd_set_workspace).
 * kappa/csw must equal the values the clover handle was built with (S10).
 * dims/precision must match the gauge handle.  in and out must not alias. */
int qcd_dslash(void* out, const void* in, const qcd_gauge* gauge, const qcd_clover* clover,
               double kappa, double csw, int parity, const int dims[4], int precision);
int qcd_dslash_ex(void* out, const void* in, const qcd_gauge* gauge, const qcd_clover* clover,
                  double kappa, double csw, int parity, int flags, void* tmp);

/* ---- 16-bit storage of the low-precision operator (PAPER.md:163 ref. [1]) --------
 * precision = 2 in qcd_gauge_load (12-real only) and qcd_clover_build selects 16-bit
 * fixed-point storage (reading H1 in DESIGN.md): int16 codes, a per-site fp32 norm for
 * spinors and clover blocks, scale 32767 for links; arithmetic stays fp32.
 * A 16-bit spinor field is nblocks parity blocks of [3 x int4][Vh] codes + [Vh] fp32 norms
 * (52 bytes per site).  qcd_spinor_to_half / _from_half convert an fp32 internal field.
 * qcd_dslash_half: out = M in (or M^dag) as qcd_dslash_ex, with the 16-bit gauge / clover
 * handles, `in_half` a 16-bit field, the even-odd intermediate stored in 16 bits in
 * `tmp_half` (one parity block; parity 0|1 only) and `out` a 16-bit (out_precision = 2) or
 * fp32 (4) field.  Passing 16-bit handles as g_lo / c_lo to qcd_set_operator makes
 * qcd_cg_solve run the reliable-update CG with this operator inside (inner vectors fp32). */
size_t qcd_half_spinor_bytes(const int dims[4]);   /* full lattice */
int qcd_spinor_to_half(qcd_ctx* ctx, void* half, const void* f32, const int dims[4], int nblocks);
int qcd_spinor_from_half(qcd_ctx* ctx, void* f32, const void* half, const int dims[4], int nblocks);
int qcd_dslash_half(void* out, int out_precision, const void* in_half, const qcd_gauge* gauge,
                    const qcd_clover* clover, double kappa, double csw, int parity, int flags,
                    void* tmp_half);

/* ---- workspace ----------------------------------------------------------------------
 * Caller-provided DEVICE scratch used by qcd_dslash (parity 0|1), the solvers and the
 * Chebyshev driver.  qcd_workspace_bytes gives the size that covers every call for
 * this lattice (precision = the highest precision used). */
size_t qcd_workspace_bytes(const int dims[4], int precision);
int qcd_set_workspace(qcd_ctx* ctx, void* ws, size_t bytes);

/* ---- fused BLAS-1 ("vector operations", reductions) --
 * Arrays of `nreal` reals (multiple of 4) in `precision`.  Reductions multiply and
 * accumulate in fp64 (warp shuffle -> block -> last-block final pass, fixed order,
 * deterministic) and return the scalar to the HOST pointer `result` (synchronises);
 * with result == NULL the scalar stays in the ctx's device slot and the call does not
 * synchronise (used for back-to-back timing).                                       */
int qcd_axpy(qcd_ctx*, double a, const void* x, void* y, size_t nreal, int precision);   /* y += a x   */
int qcd_xpay(qcd_ctx*, const void* x, double a, void* y, size_t nreal, int precision);   /* y = x + a y */
int qcd_axpby(qcd_ctx*, double a, const void* x, double b, void* y, size_t nreal, int precision); /* y = a x + b y */
int qcd_norm2(qcd_ctx*, const void* x, size_t nreal, int precision, double* result);
int qcd_redot(qcd_ctx*, const void* x, const void* y, size_t nreal, int precision, double* result); /* Re<x,y> */
/* x += a p; r -= a q; *result = |r|^2  (the CG update, one pass) */
int qcd_cg_update(qcd_ctx*, double a, const void* p, const void* q, void* x, void* r,
                  size_t nreal, int precision, double* result);

/* ---- reduction without any allocation (variant of qcd_norm2) ----
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops): needs no qcd_ctx
 * (qcd_init allocates) and calls no cudaMalloc / cudaFree / allocating routine.  Its scratch, one fp64 partial per
 * block of 16 KiB of x and a ticket, is a static 512 KiB + 256 B device array inside the library, which every GPU
 * that loads the library holds until the process exits.
 *   qcd_noalloc_setup(device)   once per device, outside any capture: takes the device address of that array
 *                               (cudaGetSymbolAddress with `device` current).  QCD_ECUDA / QCD_EINVAL on failure.
 *   qcd_norm2_noalloc(...)      *result_dev = sum_i x_i^2, products and sums in fp64, deterministic (the value
 *                               depends on nreal only).  x: DEVICE, 16-byte aligned, nreal reals of `precision`
 *                               4|8, nreal a multiple of 16/precision; result_dev: DEVICE double, written on
 *                               cuda_stream (nothing is synchronised or copied to the host).
 * Limit: x of at most qcd_noalloc_max_bytes() = 1 GiB (2^28 fp32 or 2^27 fp64 reals); a larger nreal is rejected
 * with QCD_EINVAL before anything is enqueued (use qcd_norm2).  All calls on a device share the array: calls that
 * overlap on the GPU (two streams, concurrent graph replays) race on it and must be serialised by the caller;
 * calls on one stream are safe, the ticket is cleared on the stream before each launch. */
size_t qcd_noalloc_max_bytes(void);
int qcd_noalloc_setup(int device);
int qcd_norm2_noalloc(int device, void* cuda_stream, const void* x, size_t nreal, int precision, double* result_dev);

/* ---- solvers (readings O6, O7, S13, S15) ----------------------
 * qcd_set_operator selects M for the solvers of this ctx:
 *   parity 2: M = A - kappa H on the full lattice; 0|1: even-odd Schur operator.
 *   g_lo/c_lo != NULL selects the reliable-update mixed solver (fp32 inner iteration
 *   with g_lo/c_lo, fp64 true residual with g_hi/c_hi, threshold delta).
 * qcd_cg_solve solves (M^dag M) x = b, x0 = 0 (input x ignored), x and b in the
 * precision of g_hi, internal layout (full field for parity 2, one block else).
 * Stops when the iterated residual |r| <= tol |b| (tested after the update).
 * Returns QCD_OK, QCD_NOCONV, QCD_EBREAKDOWN or an error.  Uses the ctx that last
 * called qcd_set_operator (qcd_cg_solve_ex names it). */
int qcd_set_operator(qcd_ctx* ctx, const qcd_gauge* g_hi, const qcd_gauge* g_lo,
                     const qcd_clover* c_hi, const qcd_clover* c_lo, double kappa, double csw,
                     int parity, double delta);
int qcd_cg_solve(void* x, const void* b, double tol, int maxiter);
int qcd_cg_solve_ex(qcd_ctx* ctx, void* x, const void* b, double tol, int maxiter,
                    qcd_stats* stats);
/* Multi-shift CG (PAPER.md:169 ref. [5]): solves (M^dag M + shifts[i]) x_i = b
 * for nshift <= 16 strictly ascending shifts >= 0 with ONE application of M^dag M per
 * iteration (B. Jegerlehner, hep-lat/9612014).  x: nshift consecutive fields (out), b: one
 * field, both in the precision of the (pure-precision) operator of qcd_set_operator.
 * shifts, r_true: HOST arrays; r_true (may be NULL) receives |b - (N + s_i) x_i| / |b|.
 * Stops when the base (smallest-shift) residual meets tol; a shifted system whose own residual
 * |zeta_i| |r| has met tol earlier is frozen from then on (reading M1), which also keeps
 * zeta_i from underflowing on long solves.  Workspace: (4 + nshift) fields. */
int qcd_cg_multishift(qcd_ctx* ctx, void* x, const void* b, const double* shifts, int nshift,
                      double tol, int maxiter, qcd_stats* stats, double* r_true);
/* out = M in (flags & QCD_DAGGER: M^dag in) for the operator of qcd_set_operator, in
 * the high precision. */
int qcd_apply_operator(qcd_ctx* ctx, void* out, const void* in, int flags);
/* Even-odd source preparation and solution reconstruction (SURVEY.md 8(c) reading O5; the even-odd
 * preconditioning is north_star's, PAPER.md names only the "inverter" that uses it) for the
 * operator of qcd_set_operator with parity p = 0|1, pb = 1 - p, in its high precision:
 *   qcd_eo_prepare:      bhat_p = b_p + kappa H_{p,pb} A^-1_{pb} b_pb
 *   qcd_eo_reconstruct:  x_pb   = A^-1_{pb} (b_pb + kappa H_{pb,p} x_p)
 * so that Mhat x_p = bhat_p (e.g. x_p from qcd_cg_solve on Mhat^dag bhat_p) followed by the reconstruction
 * solves the full system (A - kappa H) x = b.  b: full field (even block, then odd block), read only;
 * bhat: one-parity block, must not overlap b; x: full field whose parity-p block is read and whose
 * parity-pb block is written, must not overlap b.  With a clover term qcd_eo_prepare uses one parity
 * block of the workspace (qcd_set_workspace) as scratch.  QCD_EINVAL if no even-odd operator is set. */
int qcd_eo_prepare(qcd_ctx* ctx, void* bhat, const void* b);
int qcd_eo_reconstruct(qcd_ctx* ctx, void* x, const void* b);

/* ---- Chebyshev driver (reading O8/S16) ----
 * y = sum_{k=0}^{degree} coeff[k] T_k(H_W/scale) v,  H_W = gamma5 (1 - kappa H), full
 * lattice.  Evaluated by the Clenshaw recurrence b_k = c_k v + 2 X b_{k+1} - b_{k+2},
 * y = c_0 v + X b_1 - b_2 (the same polynomial as the forward three-term recurrence of
 * reading O8, one operator apply per degree; gamma5, the recurrence and the coefficient
 * term are fused into the hop kernel's epilogue: 2 launches per degree).
 * v, y: full internal fields in the gauge's precision; coeff: HOST array of degree+1
 * doubles.  Uses the ctx workspace (2 full fields per vector).
 * qcd_cheb_apply_multi: nvec right-hand sides stored as nvec consecutive full fields in
 * v and y; each link is read from HBM once per thread block and reused for all vectors
 * (PAPER.md:68,109 multi-blas batching; PAPER.md:155 many-vector overlap workload). */
int qcd_cheb_apply(qcd_ctx* ctx, void* y, const void* v, const qcd_gauge* g, double kappa,
                   const double* coeff, int degree, double scale);
int qcd_cheb_apply_multi(qcd_ctx* ctx, void* y, const void* v, int nvec, const qcd_gauge* g,
                         double kappa, const double* coeff, int degree, double scale);

/* Multi-right-hand-side Wilson operator: out_j = (1 - kappa H) in_j, or
 * gamma5 (1 - kappa H) in_j when gamma5 != 0, for nvec full-lattice vectors stored one after the
 * other (internal layout, precision of the gauge handle: 4 | 8; no clover).  Two launches; for
 * nvec > 1 every link is fetched from HBM once per block of 128 sites and reused from shared
 * memory for all vectors.  out and in must not overlap. */
int qcd_wilson_multi(qcd_ctx* ctx, void* out, const void* in, int nvec, const qcd_gauge* g,
                     double kappa, int gamma5);

/* ---- host-buffer convenience (end-to-end path: copies inside the call) -------------
 * out_host = H_{p,1-p} in_host for one-parity blocks held in HOST memory, internal
 * layout: copies in -> device scratch (ctx workspace), runs qcd_hop, copies out. */
int qcd_hop_host(qcd_ctx* ctx, void* out_host, const void* in_host, const qcd_gauge* g,
                 int out_parity, int dagger);

/* out_host = M in_host (or M^dag, flags & QCD_DAGGER) with M as in qcd_dslash: HOST buffers in
 * the internal layout (full field for parity 2, one parity block else); gauge / clover stay
 * resident on the device.  H2D copy, the operator, D2H copy, then a stream synchronise.
 * Needs a workspace of 2 * field + one parity block. */
int qcd_dslash_host(qcd_ctx* ctx, void* out_host, const void* in_host, const qcd_gauge* g,
                    const qcd_clover* c, double kappa, double csw, int parity, int flags);

/* The same for nvec HOST vectors (vector i at in_host + i * in_stride, result at out_host +
 * i * out_stride, strides in bytes, 0 = the same buffer every time), as a three-stage pipeline:
 * the H2D copy of vector i+1, the operator on vector i and the D2H copy of vector i-1 overlap
 * (two copy streams owned by the ctx; PCIe is full duplex).  Host buffers should be pinned, else
 * the copies serialise.  Needs a workspace of 4 * field + one parity block.  Returns after the
 * last result has landed in host memory.  The kernels are qcd_dslash's: per-vector results are
 * bit-identical to qcd_dslash_host. */
int qcd_dslash_host_batch(qcd_ctx* ctx, void* out_host, const void* in_host, int nvec,
                          size_t out_stride, size_t in_stride, const qcd_gauge* g, const qcd_clover* c,
                          double kappa, double csw, int parity, int flags);

/* number of kernels this library has launched on this ctx since qcd_init */
long long qcd_launch_count(const qcd_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* QCD_B200_H */
