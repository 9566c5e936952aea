/*
 * qcd_oracle_impl.h -- precision-generic body of the CPU oracle.
 *
 * TEST INFRASTRUCTURE ONLY (see oracle/README.md): included twice by
 * qcd_oracle.c, once with REAL=double (suffix _f64) and once with REAL=float
 * (suffix _f32, needed only for the fp32 inner iteration of the reliable-update
 * CG, reading O7).  Shares no code with paper_2001_05706_b200/csrc.
 *
 * Everything here is the DEFINITION written out: full 4x4 gamma matrices, full
 * 3x3 links, lexicographic site order, no spin projection, no link
 * reconstruction, no checkerboarded storage.
 *
 * Layouts (the paper, PAPER.md, fixes none):
 *   site   s = x + X*(y + Y*(z + Z*t)),  dims = {X,Y,Z,T}
 *   spinor psi[(s*4 + spin)*3 + colour]                     (complex)
 *   gauge  U  [((s*4 + mu)*3 + row)*3 + col],  mu=0..3=x,y,z,t (complex)
 *   F      F  [((s*6 + plane)*3 + row)*3 + col], planes (01,02,03,12,13,23)
 *   A      A  [(s*12 + i)*12 + j],  i = spin*3 + colour       (complex)
 */

#define CPLX REAL complex

/* ---- small 3x3 helpers -------------------------------------------------- */
static inline void FN(mul33)(CPLX *c, const CPLX *a, const CPLX *b)
{
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            CPLX s = 0;
            for (int k = 0; k < 3; k++) s += a[i * 3 + k] * b[k * 3 + j];
            c[i * 3 + j] = s;
        }
}
static inline void FN(dag33)(CPLX *c, const CPLX *a)
{
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) c[i * 3 + j] = conj(a[j * 3 + i]);
}
/* product of four matrices, each optionally daggered: r = op(a) op(b) op(c) op(d) */
static inline void FN(leaf)(CPLX *r, const CPLX *a, int da, const CPLX *b, int db,
                            const CPLX *c, int dc, const CPLX *d, int dd)
{
    CPLX ta[9], tb[9], tc[9], td[9], t1[9], t2[9];
    if (da) FN(dag33)(ta, a); else memcpy(ta, a, sizeof ta);
    if (db) FN(dag33)(tb, b); else memcpy(tb, b, sizeof tb);
    if (dc) FN(dag33)(tc, c); else memcpy(tc, c, sizeof tc);
    if (dd) FN(dag33)(td, d); else memcpy(td, d, sizeof td);
    FN(mul33)(t1, ta, tb);
    FN(mul33)(t2, t1, tc);
    FN(mul33)(r, t2, td);
}

/* ---- Wilson hopping term --------------------------------------------------
 * BASELINE.json north_star formula (the paper prints no equation; reading S1/O1):
 *   (H psi)(x) = sum_mu [ (1 - gamma_mu) U_mu(x) psi(x+mu)
 *                       + (1 + gamma_mu) U_mu(x-mu)^dagger psi(x-mu) ]
 * dagger != 0 gives the explicit adjoint (reading O4)
 *   (H^dag psi)(x) = sum_mu [ (1 + gamma_mu) U_mu(x) psi(x+mu)
 *                           + (1 - gamma_mu) U_mu(x-mu)^dagger psi(x-mu) ]
 * Periodic in x,y,z; a hop across the t = T-1 <-> 0 seam multiplies psi by
 * tb (= -1 antiperiodic, +1 periodic), reading S4.
 * parity_mask: 2 = all sites; 0/1 = compute only sites with (x+y+z+t)&1 == mask
 * and write zero to the others (even-odd bookkeeping without any checkerboarded
 * storage, reading O5).
 */
static inline void FN(hop_site)(CPLX acc[4][3], const CPLX *in, const CPLX *U, const int *dims,
                                int tb, int dagger, long s)
{
    const int X = dims[0], Y = dims[1], Z = dims[2], T = dims[3];
    const double sg = dagger ? -1.0 : 1.0;
    int c[4];
    long r = s;
    c[0] = (int)(r % X); r /= X;
    c[1] = (int)(r % Y); r /= Y;
    c[2] = (int)(r % Z); r /= Z;
    c[3] = (int)r;
    for (int sp = 0; sp < 4; sp++)
        for (int a = 0; a < 3; a++) acc[sp][a] = 0;
    for (int mu = 0; mu < 4; mu++) {
        const int L = dims[mu];
        int cp[4] = {c[0], c[1], c[2], c[3]}, cm[4] = {c[0], c[1], c[2], c[3]};
        cp[mu] = (c[mu] + 1) % L;
        cm[mu] = (c[mu] + L - 1) % L;
        const long sp_ = cp[0] + (long)X * (cp[1] + (long)Y * (cp[2] + (long)Z * cp[3]));
        const long sm_ = cm[0] + (long)X * (cm[1] + (long)Y * (cm[2] + (long)Z * cm[3]));
        const double sf = (mu == 3 && c[3] == T - 1) ? (double)tb : 1.0;
        const double sb = (mu == 3 && c[3] == 0) ? (double)tb : 1.0;
        const CPLX *Uf = U + ((s * 4 + mu) * 9);
        const CPLX *Ub = U + ((sm_ * 4 + mu) * 9);
        CPLX chi[4][3];
        /* forward: chi = U_mu(x) psi(x+mu); acc += sf (1 -/+ gamma_mu) chi */
        for (int sp = 0; sp < 4; sp++)
            for (int a = 0; a < 3; a++) {
                CPLX v = 0;
                for (int b = 0; b < 3; b++) v += Uf[a * 3 + b] * in[(sp_ * 4 + sp) * 3 + b];
                chi[sp][a] = v;
            }
        for (int sp = 0; sp < 4; sp++)
            for (int a = 0; a < 3; a++) {
                CPLX g = 0;
                for (int sq = 0; sq < 4; sq++) g += (CPLX)orc_gamma[mu][sp][sq] * chi[sq][a];
                acc[sp][a] += (REAL)sf * (chi[sp][a] - (REAL)sg * g);
            }
        /* backward: chi = U_mu(x-mu)^dag psi(x-mu); acc += sb (1 +/- gamma_mu) chi */
        for (int sp = 0; sp < 4; sp++)
            for (int a = 0; a < 3; a++) {
                CPLX v = 0;
                for (int b = 0; b < 3; b++) v += conj(Ub[b * 3 + a]) * in[(sm_ * 4 + sp) * 3 + b];
                chi[sp][a] = v;
            }
        for (int sp = 0; sp < 4; sp++)
            for (int a = 0; a < 3; a++) {
                CPLX g = 0;
                for (int sq = 0; sq < 4; sq++) g += (CPLX)orc_gamma[mu][sp][sq] * chi[sq][a];
                acc[sp][a] += (REAL)sb * (chi[sp][a] + (REAL)sg * g);
            }
    }
}

void FN(orc_hop)(CPLX *out, const CPLX *in, const CPLX *U, const int *dims,
                 int tb, int dagger, int parity_mask)
{
    const int X = dims[0], Y = dims[1], Z = dims[2], T = dims[3];
    const long V = (long)X * Y * Z * T;
    orc_init_gamma();
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; s++) {
        long r = s;
        const int x = (int)(r % X); r /= X;
        const int y = (int)(r % Y); r /= Y;
        const int z = (int)(r % Z); r /= Z;
        const int t = (int)r;
        CPLX acc[4][3];
        if (parity_mask == 2 || ((x + y + z + t) & 1) == parity_mask)
            FN(hop_site)(acc, in, U, dims, tb, dagger, s);
        else
            memset(acc, 0, sizeof acc);
        for (int sp = 0; sp < 4; sp++)
            for (int a = 0; a < 3; a++) out[(s * 4 + sp) * 3 + a] = acc[sp][a];
    }
}

/* out(x) = M(x) in(x) with M a 12x12 complex matrix per site (M == NULL: copy).
 * parity_mask as in orc_hop (other sites get zero). */
void FN(orc_site_matrix_apply)(CPLX *out, const CPLX *M, const CPLX *in, const int *dims,
                               int parity_mask)
{
    const int X = dims[0], Y = dims[1], Z = dims[2], T = dims[3];
    const long V = (long)X * Y * Z * T;
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; s++) {
        long r = s;
        int x = (int)(r % X); r /= X;
        int y = (int)(r % Y); r /= Y;
        int z = (int)(r % Z); r /= Z;
        int t = (int)r;
        CPLX o[12];
        if (parity_mask != 2 && ((x + y + z + t) & 1) != parity_mask) {
            for (int i = 0; i < 12; i++) o[i] = 0;
        } else if (!M) {
            for (int i = 0; i < 12; i++) o[i] = in[s * 12 + i];
        } else {
            for (int i = 0; i < 12; i++) {
                CPLX v = 0;
                for (int j = 0; j < 12; j++) v += M[(s * 12 + i) * 12 + j] * in[s * 12 + j];
                o[i] = v;
            }
        }
        for (int i = 0; i < 12; i++) out[s * 12 + i] = o[i];
    }
}

/* ---- the operator M and its adjoint --------------------------------------
 * mode 2 (full lattice, reading S11):  M psi = A psi - kappa H psi   (A = 1 if NULL)
 * mode p in {0,1} (even-odd Schur complement on parity p, reading O5/S12):
 *   Mhat psi_p = A_pp psi_p - kappa^2 H_{p,pbar} A^{-1}_{pbar,pbar} H_{pbar,p} psi_p
 * psi_p is a full-lattice array that is zero on parity pbar.
 * dagger: H -> H^dag (A and A^{-1} are Hermitian), reading O4.
 * t1, t2: caller-provided scratch spinors.
 */
typedef struct {
    const CPLX *U, *A, *Ainv;
    int dims[4];
    double kappa;
    int tb, mode;
} FN(orc_op);

void FN(orc_apply_M)(CPLX *out, const CPLX *in, const FN(orc_op) *op, int dagger,
                     CPLX *t1, CPLX *t2)
{
    const long n = (long)op->dims[0] * op->dims[1] * op->dims[2] * op->dims[3] * 12;
    if (op->mode == 2) {
        FN(orc_hop)(t1, in, op->U, op->dims, op->tb, dagger, 2);
        FN(orc_site_matrix_apply)(t2, op->A, in, op->dims, 2);
        const REAL k = (REAL)op->kappa;
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) out[i] = t2[i] - k * t1[i];
    } else {
        const int p = op->mode, pb = 1 - op->mode;
        FN(orc_hop)(t1, in, op->U, op->dims, op->tb, dagger, pb);     /* H_{pb,p} in      */
        FN(orc_site_matrix_apply)(t2, op->Ainv, t1, op->dims, pb);   /* A^-1_{pb,pb} ... */
        FN(orc_hop)(t1, t2, op->U, op->dims, op->tb, dagger, p);      /* H_{p,pb} ...     */
        FN(orc_site_matrix_apply)(t2, op->A, in, op->dims, p);       /* A_pp in          */
        const REAL k2 = (REAL)(op->kappa * op->kappa);
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) out[i] = t2[i] - k2 * t1[i];
    }
}

/* N = M^dag M */
static void FN(apply_N)(CPLX *out, const CPLX *in, const FN(orc_op) *op, CPLX *tmp, CPLX *t1, CPLX *t2)
{
    FN(orc_apply_M)(tmp, in, op, 0, t1, t2);
    FN(orc_apply_M)(out, tmp, op, 1, t1, t2);
}

/* inner products: products and sums in fp64 whatever REAL is (reading O6) */
static double FN(norm2)(const CPLX *a, long n)
{
    double s = 0;
#pragma omp parallel for schedule(static) reduction(+ : s)
    for (long i = 0; i < n; i++) {
        double re = (double)creal(a[i]), im = (double)cimag(a[i]);
        s += re * re + im * im;
    }
    return s;
}
static double FN(redot)(const CPLX *a, const CPLX *b, long n)
{
    double s = 0;
#pragma omp parallel for schedule(static) reduction(+ : s)
    for (long i = 0; i < n; i++)
        s += (double)creal(a[i]) * (double)creal(b[i]) + (double)cimag(a[i]) * (double)cimag(b[i]);
    return s;
}
