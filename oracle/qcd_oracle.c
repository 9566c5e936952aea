/*
 * qcd_oracle.c -- plain, slow, obviously-correct CPU oracle for the Wilson /
 * Wilson-clover operator and the CG solvers built on it.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load this.  It shares no code with
 * the CUDA path (paper_2001_05706_b200/csrc) and neither includes the other.
 *
 * The paper (/root/reference/PAPER.md, arXiv 2001.05706) prints no equation;
 * it names the hot path ("the D-slash", Table 2 caption,
 * PAPER.md:151 section 4), its precision and 12-real link storage
 * (PAPER.md:143), that vector operations and reductions are separate kernels
 * (section 3) and that the solvers are the mixed-precision Krylov
 * solvers of ref. [1].  The mathematics is BASELINE.json
 * north_star's formula and the readings listed in DESIGN.md ("Readings");
 * each function below names the reading it follows.
 *
 * Arithmetic: fp64 throughout (C99 double complex); the *_f32 instantiation
 * exists only for the fp32 inner iteration of reading O7.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): Clifford algebra, free-field
 * plane waves in closed form, gamma5-hermiticity, gauge covariance, constant
 * abelian field (clover normalisation), dense 2^4 matrix + LU solve, Schur
 * identities, Chebyshev vs Clenshaw / scalar polynomial.  Parity unpinned by the
 * paper (conventions of this build): RNG draw order, Chebyshev
 * coefficient choice, asymmetric even-odd form, "solve N x = b" reading.
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---- DeGrand-Rossi gamma matrices (reading S2/O2) --
 * orc_gamma[mu], mu = 0..3 = x,y,z,t; orc_gamma[4] = gamma5 = gx gy gz gt,
 * computed as the product (test P1 checks it is diag(1,1,-1,-1)).
 * orc_sigma[plane] = (i/2)[gamma_mu, gamma_nu], planes (01,02,03,12,13,23). */
static double complex orc_gamma[5][4][4];
static double complex orc_sigma[6][4][4];
static int orc_gamma_ready = 0;
static const int orc_plane_mu[6] = {0, 0, 0, 1, 1, 2};
static const int orc_plane_nu[6] = {1, 2, 3, 2, 3, 3};

static void mat4mul(double complex c[4][4], double complex a[4][4], double complex b[4][4])
{
    double complex t[4][4];
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++) {
            double complex s = 0;
            for (int k = 0; k < 4; k++) s += a[i][k] * b[k][j];
            t[i][j] = s;
        }
    memcpy(c, t, sizeof t);
}

static void orc_init_gamma(void)
{
    if (orc_gamma_ready) return;
#pragma omp critical(orc_gamma_init)
    {
        if (!orc_gamma_ready) {
            memset(orc_gamma, 0, sizeof orc_gamma);
            /* gamma_x */
            orc_gamma[0][0][3] = I;  orc_gamma[0][1][2] = I;
            orc_gamma[0][2][1] = -I; orc_gamma[0][3][0] = -I;
            /* gamma_y */
            orc_gamma[1][0][3] = -1; orc_gamma[1][1][2] = 1;
            orc_gamma[1][2][1] = 1;  orc_gamma[1][3][0] = -1;
            /* gamma_z */
            orc_gamma[2][0][2] = I;  orc_gamma[2][1][3] = -I;
            orc_gamma[2][2][0] = -I; orc_gamma[2][3][1] = I;
            /* gamma_t */
            orc_gamma[3][0][2] = 1;  orc_gamma[3][1][3] = 1;
            orc_gamma[3][2][0] = 1;  orc_gamma[3][3][1] = 1;
            /* gamma_5 = gx gy gz gt */
            double complex g5[4][4];
            mat4mul(g5, orc_gamma[0], orc_gamma[1]);
            mat4mul(g5, g5, orc_gamma[2]);
            mat4mul(g5, g5, orc_gamma[3]);
            memcpy(orc_gamma[4], g5, sizeof g5);
            for (int pl = 0; pl < 6; pl++) {
                double complex ab[4][4], ba[4][4];
                mat4mul(ab, orc_gamma[orc_plane_mu[pl]], orc_gamma[orc_plane_nu[pl]]);
                mat4mul(ba, orc_gamma[orc_plane_nu[pl]], orc_gamma[orc_plane_mu[pl]]);
                for (int i = 0; i < 4; i++)
                    for (int j = 0; j < 4; j++) orc_sigma[pl][i][j] = 0.5 * I * (ab[i][j] - ba[i][j]);
            }
            orc_gamma_ready = 1;
        }
    }
}

/* out: 5 matrices of 4x4 complex (interleaved re,im) */
void orc_get_gamma(double *out)
{
    orc_init_gamma();
    memcpy(out, orc_gamma, sizeof orc_gamma);
}
void orc_get_sigma(double *out)
{
    orc_init_gamma();
    memcpy(out, orc_sigma, sizeof orc_sigma);
}
int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- precision-generic part, instantiated twice -------------------------- */
#define REAL double
#define FN(name) name##_f64
#include "qcd_oracle_impl.h"
#undef REAL
#undef FN
#undef CPLX

#define REAL float
#define FN(name) name##_f32
#include "qcd_oracle_impl.h"
#undef REAL
#undef FN
#undef CPLX

typedef double complex zc;
typedef float complex fc;

/* ---- clover field strength (reading O3 / S9) ------
 * Q_mn(x) = U_m(x)     U_n(x+m)      U_m(x+n)^+    U_n(x)^+
 *         + U_n(x)     U_m(x-m+n)^+  U_n(x-m)^+    U_m(x-m)
 *         + U_m(x-m)^+ U_n(x-m-n)^+  U_m(x-m-n)    U_n(x-n)
 *         + U_n(x-n)^+ U_m(x-n)      U_n(x+m-n)    U_m(x)^+
 * Fhat_mn = (Q_mn - Q_mn^+)/8, no trace subtraction; all shifts periodic (the
 * antiperiodic sign cancels in closed loops).
 */
static long site_shift(const int *dims, const int *c, int m, int dm, int n, int dn)
{
    int d[4] = {c[0], c[1], c[2], c[3]};
    d[m] = (d[m] + dm + 2 * dims[m]) % dims[m];
    d[n] = (d[n] + dn + 2 * dims[n]) % dims[n];
    return d[0] + (long)dims[0] * (d[1] + (long)dims[1] * (d[2] + (long)dims[2] * d[3]));
}

static void field_strength_site(zc *Fo, const zc *U, const int *dims, long s)
{
#define LINK(site, mu) (U + (((site) * 4 + (mu)) * 9))
    int c[4];
    long r = s;
    c[0] = (int)(r % dims[0]); r /= dims[0];
    c[1] = (int)(r % dims[1]); r /= dims[1];
    c[2] = (int)(r % dims[2]); r /= dims[2];
    c[3] = (int)r;
    for (int pl = 0; pl < 6; pl++) {
        const int m = orc_plane_mu[pl], n = orc_plane_nu[pl];
        const long x = s;
        const long xpm = site_shift(dims, c, m, +1, n, 0);
        const long xpn = site_shift(dims, c, m, 0, n, +1);
        const long xmm = site_shift(dims, c, m, -1, n, 0);
        const long xmn = site_shift(dims, c, m, 0, n, -1);
        const long xmmpn = site_shift(dims, c, m, -1, n, +1);
        const long xmmmn = site_shift(dims, c, m, -1, n, -1);
        const long xpmmn = site_shift(dims, c, m, +1, n, -1);
        zc Q[9], L[9];
        leaf_f64(Q, LINK(x, m), 0, LINK(xpm, n), 0, LINK(xpn, m), 1, LINK(x, n), 1);
        leaf_f64(L, LINK(x, n), 0, LINK(xmmpn, m), 1, LINK(xmm, n), 1, LINK(xmm, m), 0);
        for (int i = 0; i < 9; i++) Q[i] += L[i];
        leaf_f64(L, LINK(xmm, m), 1, LINK(xmmmn, n), 1, LINK(xmmmn, m), 0, LINK(xmn, n), 0);
        for (int i = 0; i < 9; i++) Q[i] += L[i];
        leaf_f64(L, LINK(xmn, n), 1, LINK(xmn, m), 0, LINK(xpmmn, n), 0, LINK(x, m), 1);
        for (int i = 0; i < 9; i++) Q[i] += L[i];
        for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) Fo[pl * 9 + i * 3 + j] = (Q[i * 3 + j] - conj(Q[j * 3 + i])) / 8.0;
    }
#undef LINK
}

/* F for every site: F[((s*6 + plane)*3 + row)*3 + col] */
void orc_field_strength(double *F_, const double *U_, const int *dims)
{
    const long V = (long)dims[0] * dims[1] * dims[2] * dims[3];
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; s++) field_strength_site((zc *)F_ + s * 54, (const zc *)U_, dims, s);
}
/* F at listed sites only: F[((i*6 + plane)*3 + row)*3 + col] for sites[i] */
void orc_field_strength_sites(double *F_, const double *U_, const int *dims, const long *sites,
                              long nsites)
{
    for (long i = 0; i < nsites; i++) field_strength_site((zc *)F_ + i * 54, (const zc *)U_, dims, sites[i]);
}

/* A(x) = 1 + coeff * sum_{mu<nu} i sigma_munu (x) Fhat_munu(x), coeff = kappa*csw;
 * coeff = 1 with unit = 0 gives the bare C(x).  12x12, index = spin*3 + colour. */
void orc_clover_matrix(double *A_, const double *F_, const int *dims, double coeff, int add_unit)
{
    zc *A = (zc *)A_;
    const zc *F = (const zc *)F_;
    const long V = (long)dims[0] * dims[1] * dims[2] * dims[3];
    orc_init_gamma();
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; s++) {
        zc *Ao = A + s * 144;
        for (int i = 0; i < 144; i++) Ao[i] = 0;
        if (add_unit)
            for (int i = 0; i < 12; i++) Ao[i * 12 + i] = 1.0;
        for (int pl = 0; pl < 6; pl++) {
            const zc *Fp = F + ((s * 6 + pl) * 9);
            for (int sp = 0; sp < 4; sp++)
                for (int sq = 0; sq < 4; sq++) {
                    const zc w = coeff * I * orc_sigma[pl][sp][sq];
                    if (w == 0) continue;
                    for (int a = 0; a < 3; a++)
                        for (int b = 0; b < 3; b++) Ao[(sp * 3 + a) * 12 + (sq * 3 + b)] += w * Fp[a * 3 + b];
                }
        }
    }
}

/* Ainv(x) = A(x)^{-1}: Gauss-Jordan with partial pivoting on each 12x12 block.
 * Returns the number of singular blocks (0 = fine). */
int orc_invert_12(double *Ainv_, const double *A_, long nsites)
{
    zc *Ainv = (zc *)Ainv_;
    const zc *A = (const zc *)A_;
    int bad = 0;
#pragma omp parallel for schedule(static) reduction(+ : bad)
    for (long s = 0; s < nsites; s++) {
        zc m[12][24];
        for (int i = 0; i < 12; i++)
            for (int j = 0; j < 12; j++) {
                m[i][j] = A[s * 144 + i * 12 + j];
                m[i][12 + j] = (i == j) ? 1.0 : 0.0;
            }
        int ok = 1;
        for (int col = 0; col < 12; col++) {
            int piv = col;
            double best = cabs(m[col][col]);
            for (int r = col + 1; r < 12; r++)
                if (cabs(m[r][col]) > best) { best = cabs(m[r][col]); piv = r; }
            if (best == 0.0) { ok = 0; break; }
            if (piv != col)
                for (int j = 0; j < 24; j++) { zc t = m[col][j]; m[col][j] = m[piv][j]; m[piv][j] = t; }
            const zc inv = 1.0 / m[col][col];
            for (int j = 0; j < 24; j++) m[col][j] *= inv;
            for (int r = 0; r < 12; r++) {
                if (r == col) continue;
                const zc f = m[r][col];
                if (f == 0) continue;
                for (int j = 0; j < 24; j++) m[r][j] -= f * m[col][j];
            }
        }
        if (!ok) bad += 1;
        for (int i = 0; i < 12; i++)
            for (int j = 0; j < 12; j++) Ainv[s * 144 + i * 12 + j] = ok ? m[i][12 + j] : 0.0;
    }
    return bad;
}

/* ---- exported wrappers (flat double/float arrays, interleaved re,im) ------ */
void orc_hop(double *out, const double *in, const double *U, const int *dims, int tb, int dagger,
             int parity_mask)
{
    orc_hop_f64((zc *)out, (const zc *)in, (const zc *)U, dims, tb, dagger, parity_mask);
}
void orc_site_matrix_apply(double *out, const double *M, const double *in, const int *dims,
                           int parity_mask)
{
    orc_site_matrix_apply_f64((zc *)out, (const zc *)M, (const zc *)in, dims, parity_mask);
}

static void fill_op64(orc_op_f64 *op, const double *U, const double *A, const double *Ainv,
                      const int *dims, double kappa, int tb, int mode)
{
    op->U = (const zc *)U; op->A = (const zc *)A; op->Ainv = (const zc *)Ainv;
    memcpy(op->dims, dims, 4 * sizeof(int));
    op->kappa = kappa; op->tb = tb; op->mode = mode;
}
static void fill_op32(orc_op_f32 *op, const float *U, const float *A, const float *Ainv,
                      const int *dims, double kappa, int tb, int mode)
{
    op->U = (const fc *)U; op->A = (const fc *)A; op->Ainv = (const fc *)Ainv;
    memcpy(op->dims, dims, 4 * sizeof(int));
    op->kappa = kappa; op->tb = tb; op->mode = mode;
}

/* out = M in or M^dag in; mode 2 = full lattice, 0/1 = even-odd on that parity. */
int orc_apply_M(double *out, const double *in, const double *U, const double *A, const double *Ainv,
                const int *dims, double kappa, int tb, int mode, int dagger)
{
    const long n = (long)dims[0] * dims[1] * dims[2] * dims[3] * 12;
    orc_op_f64 op;
    fill_op64(&op, U, A, Ainv, dims, kappa, tb, mode);
    zc *t1 = malloc(n * sizeof(zc)), *t2 = malloc(n * sizeof(zc));
    if (!t1 || !t2) { free(t1); free(t2); return -1; }
    orc_apply_M_f64((zc *)out, (const zc *)in, &op, dagger, t1, t2);
    free(t1); free(t2);
    return 0;
}

/* ---- CG on N = M^dag M, reading O6 / S13 -----------------------------------
 *   x=0; r=b; p=r; rho=<r,r>
 *   for k=1..maxiter: q=Np; alpha=rho/Re<p,q>; x+=alpha p; r-=alpha q; rho'=<r,r>
 *       if sqrt(rho') <= tol*|b|: stop (iters=k); beta=rho'/rho; p=r+beta p; rho=rho'
 *   r_true = |b - N x|/|b| recomputed from scratch.
 * stats[0]=iters, [1]=iterated residual/|b|, [2]=true residual/|b|, [3]=converged(1/0),
 * stats[4]=breakdown flag.  Returns 0, or -1 on allocation failure.
 */
int orc_cg(double *x_, const double *b_, const double *U, const double *A, const double *Ainv,
           const int *dims, double kappa, int tb, int mode, double tol, int maxiter, double *stats)
{
    const long n = (long)dims[0] * dims[1] * dims[2] * dims[3] * 12;
    orc_op_f64 op;
    fill_op64(&op, U, A, Ainv, dims, kappa, tb, mode);
    zc *x = (zc *)x_;
    const zc *b = (const zc *)b_;
    zc *r = malloc(n * sizeof(zc)), *p = malloc(n * sizeof(zc)), *q = malloc(n * sizeof(zc));
    zc *tmp = malloc(n * sizeof(zc)), *t1 = malloc(n * sizeof(zc)), *t2 = malloc(n * sizeof(zc));
    if (!r || !p || !q || !tmp || !t1 || !t2) {
        free(r); free(p); free(q); free(tmp); free(t1); free(t2);
        return -1;
    }
    for (long i = 0; i < n; i++) { x[i] = 0; r[i] = b[i]; p[i] = b[i]; }
    const double bnorm = sqrt(norm2_f64(b, n));
    double rho = norm2_f64(r, n);
    int k = 0, conv = 0, brk = 0;
    double rnorm = sqrt(rho);
    if (bnorm == 0.0) conv = 1;
    while (!conv && k < maxiter) {
        k++;
        apply_N_f64(q, p, &op, tmp, t1, t2);
        const double pq = redot_f64(p, q, n);
        if (!(pq > 0.0)) { brk = 1; break; }
        const double alpha = rho / pq;
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) { x[i] += alpha * p[i]; r[i] -= alpha * q[i]; }
        const double rho2 = norm2_f64(r, n);
        rnorm = sqrt(rho2);
        if (rnorm <= tol * bnorm) { conv = 1; break; }
        const double beta = rho2 / rho;
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) p[i] = r[i] + beta * p[i];
        rho = rho2;
    }
    apply_N_f64(q, x, &op, tmp, t1, t2);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; i++) q[i] = b[i] - q[i];
    stats[0] = k;
    stats[1] = bnorm > 0 ? rnorm / bnorm : 0.0;
    stats[2] = bnorm > 0 ? sqrt(norm2_f64(q, n)) / bnorm : 0.0;
    stats[3] = conv;
    stats[4] = brk;
    free(r); free(p); free(q); free(tmp); free(t1); free(t2);
    return 0;
}

static void apply_N_q16(fc *q, const fc *p, const orc_op_f32 *op, fc *tmp, fc *t1, fc *t2, fc *ph);

/* ---- reliable-update mixed-precision CG, reading O7 / S15 (PAPER.md:163 ref [1])
 * Inner vectors x,r,p,q and N in fp32 (Ulo/Alo/Ainvlo = the fp64 fields rounded to
 * fp32 by the caller); y, r_hi and N_hi in fp64; delta = 0.1 by default.
 *   y=0; r_hi=b; x=0; r=(f32)b; p=r; rho=|r|^2; rmax=|r|
 *   each iteration: q=N_lo p; alpha=rho/Re<p,q>; x+=alpha p; r-=alpha q; rho'=|r|^2
 *     rmax=max(rmax,|r|);  if |r| < delta*rmax or |r| <= tol|b|:
 *         y+=x; r_hi=b-N_hi y; x=0; r=(f32)r_hi; rmax=|r_hi|; rho'=|r_hi|^2;
 *         stop iff |r_hi| <= tol|b|
 *     beta=rho'/rho; p=r+beta p (p is kept); rho=rho'
 * stats[0]=iters (fp32 N applies), [1]=last |r_hi|/|b|, [2]=true residual, [3]=converged,
 * [4]=breakdown, [5]=reliable updates.  update_at (may be NULL): the iteration index k of each of
 * the first max_updates reliable updates, reporting only (pinned against an independent
 * dense-matrix run in tests/test_oracle_pins.py).
 */
int orc_cg_mixed(double *y_, const double *b_, const double *Uhi, const double *Ahi,
                 const double *Ainvhi, const float *Ulo, const float *Alo, const float *Ainvlo,
                 const int *dims, double kappa, int tb, int mode, double tol, int maxiter,
                 double delta, int half, double *stats, int *update_at, int max_updates)
{
    const long n = (long)dims[0] * dims[1] * dims[2] * dims[3] * 12;
    orc_op_f64 ohi;
    orc_op_f32 olo;
    fill_op64(&ohi, Uhi, Ahi, Ainvhi, dims, kappa, tb, mode);
    fill_op32(&olo, Ulo, Alo, Ainvlo, dims, kappa, tb, mode);
    zc *y = (zc *)y_;
    const zc *b = (const zc *)b_;
    zc *rh = malloc(n * sizeof(zc)), *th = malloc(n * sizeof(zc)), *h1 = malloc(n * sizeof(zc)),
       *h2 = malloc(n * sizeof(zc));
    fc *x = malloc(n * sizeof(fc)), *r = malloc(n * sizeof(fc)), *p = malloc(n * sizeof(fc)),
       *q = malloc(n * sizeof(fc)), *tl = malloc(n * sizeof(fc)), *l1 = malloc(n * sizeof(fc)),
       *l2 = malloc(n * sizeof(fc)), *ph = malloc(n * sizeof(fc));
    if (!rh || !th || !h1 || !h2 || !x || !r || !p || !q || !tl || !l1 || !l2 || !ph) {
        free(rh); free(th); free(h1); free(h2); free(x); free(r); free(p); free(q); free(tl);
        free(l1); free(l2); free(ph);
        return -1;
    }
    for (long i = 0; i < n; i++) {
        y[i] = 0; rh[i] = b[i]; x[i] = 0; r[i] = (fc)b[i]; p[i] = r[i];
    }
    const double bnorm = sqrt(norm2_f64(b, n));
    double rho = norm2_f32(r, n);
    double rmax = sqrt(rho), rhnorm = bnorm;
    int k = 0, conv = 0, brk = 0, nup = 0;
    if (bnorm == 0.0) conv = 1;
    while (!conv && k < maxiter) {
        k++;
        /* half != 0: the inner operator streams 16-bit fields (reading H1); x, r, p, q stay fp32 */
        if (half) apply_N_q16(q, p, &olo, tl, l1, l2, ph);
        else apply_N_f32(q, p, &olo, tl, l1, l2);
        const double pq = redot_f32(p, q, n);
        if (!(pq > 0.0)) { brk = 1; break; }
        const float alpha = (float)(rho / pq);
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) { x[i] += alpha * p[i]; r[i] -= alpha * q[i]; }
        double rho2 = norm2_f32(r, n);
        const double rnorm = sqrt(rho2);
        if (rnorm > rmax) rmax = rnorm;
        if (rnorm < delta * rmax || rnorm <= tol * bnorm) {
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; i++) y[i] += (zc)x[i];
            apply_N_f64(th, y, &ohi, rh, h1, h2);
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; i++) { rh[i] = b[i] - th[i]; x[i] = 0; r[i] = (fc)rh[i]; }
            rho2 = norm2_f64(rh, n);
            rhnorm = sqrt(rho2);
            rmax = rhnorm;
            if (update_at && nup < max_updates) update_at[nup] = k;
            nup++;
            if (rhnorm <= tol * bnorm) { conv = 1; break; }
        }
        const float beta = (float)(rho2 / rho);
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) p[i] = r[i] + beta * p[i];
        rho = rho2;
    }
    if (!conv) {
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) y[i] += (zc)x[i];
    }
    apply_N_f64(th, y, &ohi, rh, h1, h2);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; i++) th[i] = b[i] - th[i];
    stats[0] = k;
    stats[1] = bnorm > 0 ? rhnorm / bnorm : 0.0;
    stats[2] = bnorm > 0 ? sqrt(norm2_f64(th, n)) / bnorm : 0.0;
    stats[3] = conv;
    stats[4] = brk;
    stats[5] = nup;
    free(rh); free(th); free(h1); free(h2); free(x); free(r); free(p); free(q); free(tl);
    free(l1); free(l2); free(ph);
    return 0;
}

/* ---- 16-bit fixed-point storage for the low-precision operator (
 * PAPER.md:163 ref. [1], mixed-precision solvers with a 16-bit "half" format) -------------
 * Reading H1: the paper gives no format; this build's is
 *   spinor site (24 reals v_k): n = max_k |v_k| (fp32); code_k = rintf(v_k * (32767.0f / n)),
 *       an int16 (all codes 0 when n = 0); value read back = (float)code_k * (n / 32767.0f).
 *   link: the 12 reals of rows 0,1 (|u| <= 1): code = rintf(u * 32767.0f) clamped to
 *       +-32767, read back = (float)code * (1.0f/32767.0f); row 2 = conj(row0 x row1) of the
 *       values read back (fp32).
 *   clover site (A or A^-1, Hermitian, 2 chiral 6x6 blocks): n = max |Re|,|Im| over the
 *       diagonal and lower triangle; codes and read-back as for a spinor site; upper
 *       triangle = conjugate of the lower one, diagonal real, off-chirality blocks zero.
 * All fp32, round-to-nearest-even.  The functions below apply "store then read back" in
 * place, so that the rest of the oracle can keep working on plain float arrays.
 */
static inline float q16_code(float v, float scale)
{
    float c = rintf(v * scale);
    if (c > 32767.0f) c = 32767.0f;
    if (c < -32767.0f) c = -32767.0f;
    return c;
}
void orc_q16_codes(const float *v, short *codes, float *norms, long nsites)
{
    for (long s = 0; s < nsites; s++) {
        float n = 0.0f;
        for (int k = 0; k < 24; k++) n = fmaxf(n, fabsf(v[s * 24 + k]));
        norms[s] = n;
        const float scale = n > 0.0f ? 32767.0f / n : 0.0f;
        for (int k = 0; k < 24; k++) codes[s * 24 + k] = (short)q16_code(v[s * 24 + k], scale);
    }
}
void orc_q16_spinor(float *v, long nsites)
{
#pragma omp parallel for schedule(static)
    for (long s = 0; s < nsites; s++) {
        float n = 0.0f;
        for (int k = 0; k < 24; k++) n = fmaxf(n, fabsf(v[s * 24 + k]));
        const float scale = n > 0.0f ? 32767.0f / n : 0.0f;
        const float d = n / 32767.0f;
        for (int k = 0; k < 24; k++) v[s * 24 + k] = q16_code(v[s * 24 + k], scale) * d;
    }
}
void orc_q16_links(float *U, long nlinks)
{
    const float d = 1.0f / 32767.0f;
#pragma omp parallel for schedule(static)
    for (long l = 0; l < nlinks; l++) {
        float *u = U + l * 18;
        for (int k = 0; k < 12; k++) u[k] = q16_code(u[k], 32767.0f) * d;
        /* row 2 = conj(row0 x row1), written out component by component */
        const float complex a0 = u[0] + I * u[1], a1 = u[2] + I * u[3], a2 = u[4] + I * u[5];
        const float complex b0 = u[6] + I * u[7], b1 = u[8] + I * u[9], b2 = u[10] + I * u[11];
        const float complex c0 = conjf(a1 * b2 - a2 * b1), c1 = conjf(a2 * b0 - a0 * b2), c2 = conjf(a0 * b1 - a1 * b0);
        u[12] = crealf(c0); u[13] = cimagf(c0);
        u[14] = crealf(c1); u[15] = cimagf(c1);
        u[16] = crealf(c2); u[17] = cimagf(c2);
    }
}
void orc_q16_clover(float *A_, long nsites)
{
#pragma omp parallel for schedule(static)
    for (long s = 0; s < nsites; s++) {
        fc *A = (fc *)A_ + s * 144;
        float n = 0.0f;
        for (int b = 0; b < 2; b++)
            for (int i = 0; i < 6; i++)
                for (int j = 0; j <= i; j++) {
                    const fc a = A[(6 * b + i) * 12 + 6 * b + j];
                    n = fmaxf(n, fabsf(crealf(a)));
                    if (j < i) n = fmaxf(n, fabsf(cimagf(a)));
                }
        const float scale = n > 0.0f ? 32767.0f / n : 0.0f, d = n / 32767.0f;
        fc Q[144];
        for (int k = 0; k < 144; k++) Q[k] = 0;
        for (int b = 0; b < 2; b++)
            for (int i = 0; i < 6; i++)
                for (int j = 0; j <= i; j++) {
                    const int r = 6 * b + i, c = 6 * b + j;
                    const fc a = A[r * 12 + c];
                    const float re = q16_code(crealf(a), scale) * d;
                    const float im = (j < i) ? q16_code(cimagf(a), scale) * d : 0.0f;
                    Q[r * 12 + c] = re + I * im;
                    if (j < i) Q[c * 12 + r] = re - I * im;
                }
        for (int k = 0; k < 144; k++) A[k] = Q[k];
    }
}

/* out = M in (or M^dag in) with 16-bit storage of every field the operator streams: `in` must
 * already be a stored-and-read-back field, op holds stored-and-read-back links / clover; the
 * intermediate of the even-odd form is stored in 16 bits, and so is the result when
 * store_out != 0 (it is the input of the next operator).  Arithmetic fp32. */
static void apply_M_q16(fc *out, const fc *in, const orc_op_f32 *op, int dagger, int store_out, fc *t1, fc *t2)
{
    const long V = (long)op->dims[0] * op->dims[1] * op->dims[2] * op->dims[3];
    const long n = V * 12;
    if (op->mode == 2) {
        orc_apply_M_f32(out, in, op, dagger, t1, t2);
    } else {
        const int p = op->mode, pb = 1 - op->mode;
        orc_hop_f32(t1, in, op->U, op->dims, op->tb, dagger, pb);
        orc_site_matrix_apply_f32(t2, op->Ainv, t1, op->dims, pb);
        orc_q16_spinor((float *)t2, V);
        orc_hop_f32(t1, t2, op->U, op->dims, op->tb, dagger, p);
        orc_site_matrix_apply_f32(t2, op->A, in, op->dims, p);
        const float k2 = (float)(op->kappa * op->kappa);
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) out[i] = t2[i] - k2 * t1[i];
    }
    if (store_out) orc_q16_spinor((float *)out, V);
}
/* q = N_16 p :  ph = store(p);  t = store(M ph);  q = M^dag t  (q left in fp32) */
static void apply_N_q16(fc *q, const fc *p, const orc_op_f32 *op, fc *tmp, fc *t1, fc *t2, fc *ph)
{
    const long V = (long)op->dims[0] * op->dims[1] * op->dims[2] * op->dims[3];
    memcpy(ph, p, (size_t)V * 12 * sizeof(fc));
    orc_q16_spinor((float *)ph, V);
    apply_M_q16(tmp, ph, op, 0, 1, t1, t2);
    apply_M_q16(q, tmp, op, 1, 0, t1, t2);
}
int orc_apply_N_q16(float *q, const float *p, const float *U, const float *A, const float *Ainv, const int *dims,
                    double kappa, int tb, int mode)
{
    const long n = (long)dims[0] * dims[1] * dims[2] * dims[3] * 12;
    orc_op_f32 op;
    fill_op32(&op, U, A, Ainv, dims, kappa, tb, mode);
    fc *tmp = malloc(n * sizeof(fc)), *t1 = malloc(n * sizeof(fc)), *t2 = malloc(n * sizeof(fc)), *ph = malloc(n * sizeof(fc));
    if (!tmp || !t1 || !t2 || !ph) { free(tmp); free(t1); free(t2); free(ph); return -1; }
    orc_init_gamma();
    apply_N_q16((fc *)q, (const fc *)p, &op, tmp, t1, t2, ph);
    free(tmp); free(t1); free(t2); free(ph);
    return 0;
}
int orc_apply_M_q16(float *out, const float *in, const float *U, const float *A, const float *Ainv, const int *dims,
                    double kappa, int tb, int mode, int dagger, int store_out)
{
    const long n = (long)dims[0] * dims[1] * dims[2] * dims[3] * 12;
    orc_op_f32 op;
    fill_op32(&op, U, A, Ainv, dims, kappa, tb, mode);
    fc *t1 = malloc(n * sizeof(fc)), *t2 = malloc(n * sizeof(fc));
    if (!t1 || !t2) { free(t1); free(t2); return -1; }
    orc_init_gamma();
    apply_M_q16((fc *)out, (const fc *)in, &op, dagger, store_out, t1, t2);
    free(t1); free(t2);
    return 0;
}

/* ---- multi-shift CG (PAPER.md:169 ref. [5], the GWU-code solver family) ---
 * Solves (N + sigma_i) x_i = b, i = 0..ns-1, N = M^dag M, shifts ascending, sigma_i >= 0,
 * with ONE application of N per iteration.  Base system: CG on N + sigma_0 exactly as orc_cg
 * (reading O6); the shifted systems ride on the collinearity of the residuals,
 * r_i^n = zeta_i^n r^n (B. Jegerlehner, hep-lat/9612014, in the alpha/beta notation of O6):
 *   s_i = sigma_i - sigma_0,  zeta_i^{-1} = zeta_i^0 = 1,  alpha_{-1} = 1,  beta_{-1} = 0
 *   q = (N + sigma_0) p_0 ; alpha_n = rho_n / Re<p_0, q>
 *   zeta_i^{n+1} = zeta_i^n zeta_i^{n-1} alpha_{n-1}
 *                  / ( alpha_n beta_{n-1} (zeta_i^{n-1} - zeta_i^n) + zeta_i^{n-1} alpha_{n-1} (1 + s_i alpha_n) )
 *   x_i += alpha_n (zeta_i^{n+1}/zeta_i^n) p_i ;  r -= alpha_n q ; rho_{n+1} = |r|^2
 *   stop when |r| <= tol |b|  (the smallest shift converges last: |zeta_i| <= 1)
 *   beta_n = rho_{n+1}/rho_n ;  p_i = zeta_i^{n+1} r + beta_n (zeta_i^{n+1}/zeta_i^n)^2 p_i
 * A shifted system whose own residual |r_i| = |zeta_i^{n+1}| |r| has reached tol |b| is frozen: x_i,
 * p_i and zeta_i are no longer updated (reading M1 in DESIGN.md).  Without this zeta_i of a large
 * shift underflows to 0 on a long solve and the recurrence above turns 0/0 into NaN in x_i.  The
 * shifts ascend, so the active systems are always the first `nact`.
 * x: ns consecutive fields.  stats[0]=iters, [1]=iterated |r|/|b|, [3]=converged, [4]=breakdown;
 * rtrue[i] = |b - (N + sigma_i) x_i| / |b| recomputed from scratch.
 */
int orc_cg_multishift(double *x_, const double *b_, const double *U, const double *A, const double *Ainv,
                      const int *dims, double kappa, int tb, int mode, const double *sigma, int ns,
                      double tol, int maxiter, double *stats, double *rtrue)
{
    const long n = (long)dims[0] * dims[1] * dims[2] * dims[3] * 12;
    orc_op_f64 op;
    fill_op64(&op, U, A, Ainv, dims, kappa, tb, mode);
    zc *x = (zc *)x_;
    const zc *b = (const zc *)b_;
    zc *r = malloc(n * sizeof(zc)), *q = malloc(n * sizeof(zc)), *tmp = malloc(n * sizeof(zc));
    zc *t1 = malloc(n * sizeof(zc)), *t2 = malloc(n * sizeof(zc)), *p = malloc((size_t)ns * n * sizeof(zc));
    double *zm = malloc(ns * sizeof(double)), *z0 = malloc(ns * sizeof(double)), *zp = malloc(ns * sizeof(double));
    if (!r || !q || !tmp || !t1 || !t2 || !p || !zm || !z0 || !zp) {
        free(r); free(q); free(tmp); free(t1); free(t2); free(p); free(zm); free(z0); free(zp);
        return -1;
    }
    for (long i = 0; i < n; i++) r[i] = b[i];
    for (int s = 0; s < ns; s++) {
        zm[s] = z0[s] = 1.0;
        for (long i = 0; i < n; i++) { x[s * n + i] = 0; p[s * n + i] = b[i]; }
    }
    const double bnorm = sqrt(norm2_f64(b, n));
    double rho = bnorm * bnorm, alpha_old = 1.0, beta_old = 0.0, rnorm = bnorm;
    int k = 0, conv = (bnorm == 0.0), brk = 0, nact = ns;
    while (!conv && k < maxiter) {
        k++;
        apply_N_f64(q, p, &op, tmp, t1, t2);
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) q[i] += sigma[0] * p[i];
        const double pq = redot_f64(p, q, n);
        if (!(pq > 0.0)) { brk = 1; break; }
        const double alpha = rho / pq;
        for (int s = 0; s < nact; s++) {
            const double sh = sigma[s] - sigma[0];
            zp[s] = z0[s] * zm[s] * alpha_old /
                    (alpha * beta_old * (zm[s] - z0[s]) + zm[s] * alpha_old * (1.0 + sh * alpha));
            const double as = alpha * zp[s] / z0[s];
            zc *xs = x + (long)s * n, *ps = p + (long)s * n;
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; i++) xs[i] += as * ps[i];
        }
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) r[i] -= alpha * q[i];
        const double rho2 = norm2_f64(r, n);
        rnorm = sqrt(rho2);
        if (rnorm <= tol * bnorm) { conv = 1; break; }
        while (nact > 1 && fabs(zp[nact - 1]) * rnorm <= tol * bnorm) nact--;
        const double beta = rho2 / rho;
        for (int s = 0; s < nact; s++) {
            const double ratio = zp[s] / z0[s], bs = beta * ratio * ratio, zs = zp[s];
            zc *ps = p + (long)s * n;
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; i++) ps[i] = zs * r[i] + bs * ps[i];
            zm[s] = z0[s];
            z0[s] = zp[s];
        }
        rho = rho2; alpha_old = alpha; beta_old = beta;
    }
    for (int s = 0; s < ns; s++) {
        const zc *xs = x + (long)s * n;
        apply_N_f64(q, xs, &op, tmp, t1, t2);
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) q[i] = b[i] - q[i] - sigma[s] * xs[i];
        rtrue[s] = bnorm > 0 ? sqrt(norm2_f64(q, n)) / bnorm : 0.0;
    }
    stats[0] = k;
    stats[1] = bnorm > 0 ? rnorm / bnorm : 0.0;
    stats[2] = rtrue[0];
    stats[3] = conv;
    stats[4] = brk;
    free(r); free(q); free(tmp); free(t1); free(t2); free(p); free(zm); free(z0); free(zp);
    return 0;
}

/* ---- Chebyshev polynomial of H_W = gamma5 D_W, reading O8 / S16 -------------
 *   X = H_W/scale;  T_0 v = v, T_1 v = X v, T_{k+1} v = 2 X T_k v - T_{k-1} v
 *   y = sum_{k=0}^{degree} coeff[k] T_k v        (forward three-term recurrence)
 * D_W = full-lattice Wilson operator 1 - kappa H (no clover).
 */
static void apply_HW(zc *out, const zc *in, const zc *U, const int *dims, double kappa, int tb, zc *t1)
{
    const long V = (long)dims[0] * dims[1] * dims[2] * dims[3];
    orc_hop_f64(t1, in, U, dims, tb, 0, 2);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; s++)
        for (int sp = 0; sp < 4; sp++)
            for (int a = 0; a < 3; a++) {
                /* gamma5 is diagonal in this basis (P1); apply it as the matrix anyway */
                zc v = 0;
                for (int sq = 0; sq < 4; sq++) {
                    const long j = (s * 4 + sq) * 3 + a;
                    v += orc_gamma[4][sp][sq] * (in[j] - kappa * t1[j]);
                }
                out[(s * 4 + sp) * 3 + a] = v;
            }
}

void orc_apply_HW(double *out, const double *in, const double *U, const int *dims, double kappa, int tb)
{
    const long n = (long)dims[0] * dims[1] * dims[2] * dims[3] * 12;
    zc *t1 = malloc(n * sizeof(zc));
    orc_init_gamma();
    apply_HW((zc *)out, (const zc *)in, (const zc *)U, dims, kappa, tb, t1);
    free(t1);
}

int orc_cheb(double *y_, const double *v_, const double *U_, const int *dims, double kappa, int tb,
             const double *coeff, int degree, double scale)
{
    const long n = (long)dims[0] * dims[1] * dims[2] * dims[3] * 12;
    const zc *U = (const zc *)U_, *v = (const zc *)v_;
    zc *y = (zc *)y_;
    zc *tm = malloc(n * sizeof(zc)), *tc = malloc(n * sizeof(zc)), *tn = malloc(n * sizeof(zc)),
       *t1 = malloc(n * sizeof(zc));
    if (!tm || !tc || !tn || !t1) { free(tm); free(tc); free(tn); free(t1); return -1; }
    orc_init_gamma();
    for (long i = 0; i < n; i++) { tm[i] = v[i]; y[i] = coeff[0] * v[i]; }
    if (degree >= 1) {
        apply_HW(tc, tm, U, dims, kappa, tb, t1);
        for (long i = 0; i < n; i++) { tc[i] /= scale; y[i] += coeff[1] * tc[i]; }
    }
    for (int k = 1; k < degree; k++) {
        apply_HW(tn, tc, U, dims, kappa, tb, t1);
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) {
            tn[i] = 2.0 * (tn[i] / scale) - tm[i];
            y[i] += coeff[k + 1] * tn[i];
        }
        zc *sw = tm; tm = tc; tc = tn; tn = sw;
    }
    free(tm); free(tc); free(tn); free(t1);
    return 0;
}

/* ---- sampled evaluation for full-size parity checks -------------------------
 * (H psi)(x) (or H^dag) at a list of sites only; `in`/`U` are full boundary-layout
 * fields; out[i] = 12 complex for site sites[i].  Same arithmetic as orc_hop. */
void orc_hop_sites(double *out_, const double *in_, const double *U_, const int *dims, int tb,
                   int dagger, const long *sites, long nsites)
{
    zc *out = (zc *)out_;
    orc_init_gamma();
    for (long i = 0; i < nsites; i++) {
        zc acc[4][3];
        hop_site_f64(acc, (const zc *)in_, (const zc *)U_, dims, tb, dagger, sites[i]);
        for (int sp = 0; sp < 4; sp++)
            for (int a = 0; a < 3; a++) out[i * 12 + sp * 3 + a] = acc[sp][a];
    }
}
