/*
 * packed_math.cuh -- the site arithmetic of the hopping term on sm_100a packed fp32 pairs
 * (add / sub / mul / fma.rn.f32x2 -> FADD2 / FMUL2 / FFMA2: one issue slot for two lanes).
 *
 * A lane is a lattice site: a thread works on two sites at once and every quantity of
 * hop_kernel.cuh (spinor s[24], link u[18], half spinor h[12], accumulator acc[24]) becomes an
 * array of f2 = (site A value, site B value).  The formulas are those of hop_kernel.cuh
 * (DeGrand-Rossi projectors); they are written without a negated
 * multiplicand because fma.f32x2 has no operand negation in PTX: where the scalar code has
 * c - a*b, the negated operand is formed once (f2_neg) and reused.
 * Used by the 16-bit kernel (hop_half.cu), which is bound by instruction issue, not by HBM.
 */
#ifndef QCD_PACKED_MATH_CUH
#define QCD_PACKED_MATH_CUH

struct f2 {
    unsigned long long v;
};

__device__ __forceinline__ f2 f2_make(float lo, float hi)
{
    f2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ f2 f2_bits(unsigned lo, unsigned hi)
{
    f2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "r"(lo), "r"(hi));
    return r;
}
__device__ __forceinline__ void f2_get(f2 a, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a.v)); }
__device__ __forceinline__ void f2_get_bits(f2 a, unsigned& lo, unsigned& hi) { asm("mov.b64 {%0, %1}, %2;" : "=r"(lo), "=r"(hi) : "l"(a.v)); }
__device__ __forceinline__ f2 f2_set1(float x) { return f2_make(x, x); }
__device__ __forceinline__ f2 operator+(f2 a, f2 b)
{
    f2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}
__device__ __forceinline__ f2 operator-(f2 a, f2 b)
{
    f2 r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}
__device__ __forceinline__ f2 operator*(f2 a, f2 b)
{
    f2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}
/* a * b + c */
__device__ __forceinline__ f2 f2_fma(f2 a, f2 b, f2 c)
{
    f2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(a.v), "l"(b.v), "l"(c.v));
    return r;
}
__device__ __forceinline__ f2 f2_neg(f2 a)
{
    f2 z;
    z.v = 0ull;
    return z - a;
}
/* a + b (SG > 0) or a - b (SG < 0), SG a compile-time sign */
template <int SG> __device__ __forceinline__ f2 f2_pm(f2 a, f2 b) { return SG > 0 ? a + b : a - b; }

/* ---- spin projection: h = rows 0,1 of (1 + S g_mu) psi (hop_kernel.cuh project) ------------- */
template <int MU, int S> __device__ __forceinline__ void project2(f2 (&h)[12], const f2 (&s)[24])
{
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const int r0 = 2 * c, r1 = 2 * (3 + c), r2 = 2 * (6 + c), r3 = 2 * (9 + c);
        if (MU == 0) {
            h[r0] = f2_pm<-S>(s[r0], s[r3 + 1]);
            h[r0 + 1] = f2_pm<S>(s[r0 + 1], s[r3]);
            h[r1] = f2_pm<-S>(s[r1], s[r2 + 1]);
            h[r1 + 1] = f2_pm<S>(s[r1 + 1], s[r2]);
        } else if (MU == 1) {
            h[r0] = f2_pm<-S>(s[r0], s[r3]);
            h[r0 + 1] = f2_pm<-S>(s[r0 + 1], s[r3 + 1]);
            h[r1] = f2_pm<S>(s[r1], s[r2]);
            h[r1 + 1] = f2_pm<S>(s[r1 + 1], s[r2 + 1]);
        } else if (MU == 2) {
            h[r0] = f2_pm<-S>(s[r0], s[r2 + 1]);
            h[r0 + 1] = f2_pm<S>(s[r0 + 1], s[r2]);
            h[r1] = f2_pm<S>(s[r1], s[r3 + 1]);
            h[r1 + 1] = f2_pm<-S>(s[r1 + 1], s[r3]);
        } else {
            h[r0] = f2_pm<S>(s[r0], s[r2]);
            h[r0 + 1] = f2_pm<S>(s[r0 + 1], s[r2 + 1]);
            h[r1] = f2_pm<S>(s[r1], s[r3]);
            h[r1 + 1] = f2_pm<S>(s[r1 + 1], s[r3 + 1]);
        }
    }
}

/* The same projection taken straight from the UNDECODED 16-bit codes (hop_half.cu).  A code c sits in
 * the low mantissa bits of a float as pos = M + c (M = 2^23 + 2^15) or, from the word negated in the
 * integer domain, as neg = M - c.  Every h component is (upper code) +- (lower code), and both
 *     pos(a) - pos(b) = c_a - c_b      and      pos(a) - neg(b) = c_a + c_b
 * are exact in fp32: one packed subtraction per component replaces two decoding subtractions and the
 * projection's own add (12 instead of 36 FMA-pipe instructions per direction). */
template <int SG, typename Src> __device__ __forceinline__ f2 f2_pm_codes(const Src& src, int ia, int ib)
{
    return SG > 0 ? src.pos(ia) - src.neg(ib) : src.pos(ia) - src.pos(ib);
}
template <int MU, int S, typename Src> __device__ __forceinline__ void project2_codes(f2 (&h)[12], const Src& src)
{
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const int r0 = 2 * c, r1 = 2 * (3 + c), r2 = 2 * (6 + c), r3 = 2 * (9 + c);
        if (MU == 0) {
            h[r0] = f2_pm_codes<-S>(src, r0, r3 + 1);
            h[r0 + 1] = f2_pm_codes<S>(src, r0 + 1, r3);
            h[r1] = f2_pm_codes<-S>(src, r1, r2 + 1);
            h[r1 + 1] = f2_pm_codes<S>(src, r1 + 1, r2);
        } else if (MU == 1) {
            h[r0] = f2_pm_codes<-S>(src, r0, r3);
            h[r0 + 1] = f2_pm_codes<-S>(src, r0 + 1, r3 + 1);
            h[r1] = f2_pm_codes<S>(src, r1, r2);
            h[r1 + 1] = f2_pm_codes<S>(src, r1 + 1, r2 + 1);
        } else if (MU == 2) {
            h[r0] = f2_pm_codes<-S>(src, r0, r2 + 1);
            h[r0 + 1] = f2_pm_codes<S>(src, r0 + 1, r2);
            h[r1] = f2_pm_codes<S>(src, r1, r3 + 1);
            h[r1 + 1] = f2_pm_codes<-S>(src, r1 + 1, r3);
        } else {
            h[r0] = f2_pm_codes<S>(src, r0, r2);
            h[r0 + 1] = f2_pm_codes<S>(src, r0 + 1, r2 + 1);
            h[r1] = f2_pm_codes<S>(src, r1, r3);
            h[r1 + 1] = f2_pm_codes<S>(src, r1 + 1, r3 + 1);
        }
    }
}

/* ---- acc += rows 0..3 of (1 + S g_mu) chi from its upper half w (reconstruct_add) ----------- */
template <int MU, int S> __device__ __forceinline__ void reconstruct_add2(f2 (&acc)[24], const f2 (&w)[12])
{
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const int j0 = 2 * c, j1 = 2 * (3 + c);
        const int r2 = 2 * (6 + c), r3 = 2 * (9 + c);
        acc[j0] = acc[j0] + w[j0];
        acc[j0 + 1] = acc[j0 + 1] + w[j0 + 1];
        acc[j1] = acc[j1] + w[j1];
        acc[j1 + 1] = acc[j1 + 1] + w[j1 + 1];
        if (MU == 0) {
            acc[r2] = f2_pm<S>(acc[r2], w[j1 + 1]);
            acc[r2 + 1] = f2_pm<-S>(acc[r2 + 1], w[j1]);
            acc[r3] = f2_pm<S>(acc[r3], w[j0 + 1]);
            acc[r3 + 1] = f2_pm<-S>(acc[r3 + 1], w[j0]);
        } else if (MU == 1) {
            acc[r2] = f2_pm<S>(acc[r2], w[j1]);
            acc[r2 + 1] = f2_pm<S>(acc[r2 + 1], w[j1 + 1]);
            acc[r3] = f2_pm<-S>(acc[r3], w[j0]);
            acc[r3 + 1] = f2_pm<-S>(acc[r3 + 1], w[j0 + 1]);
        } else if (MU == 2) {
            acc[r2] = f2_pm<S>(acc[r2], w[j0 + 1]);
            acc[r2 + 1] = f2_pm<-S>(acc[r2 + 1], w[j0]);
            acc[r3] = f2_pm<-S>(acc[r3], w[j1 + 1]);
            acc[r3 + 1] = f2_pm<S>(acc[r3 + 1], w[j1]);
        } else {
            acc[r2] = f2_pm<S>(acc[r2], w[j0]);
            acc[r2 + 1] = f2_pm<S>(acc[r2 + 1], w[j0 + 1]);
            acc[r3] = f2_pm<S>(acc[r3], w[j1]);
            acc[r3 + 1] = f2_pm<S>(acc[r3 + 1], w[j1 + 1]);
        }
    }
}

/* acc += sc * (rows 0..3 of (1 + S g_mu) chi) with the scale folded into the accumulation: one fused
 * multiply-add per term instead of a multiplication of w and an addition.  sc[c] / nsc[c] = the factor
 * of colour component c and its negation (fma.f32x2 has no operand negation). */
template <int MU, int S> __device__ __forceinline__ void reconstruct_add2_scaled(f2 (&acc)[24], const f2 (&w)[12], const f2 (&sc)[3], const f2 (&nsc)[3])
{
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const int j0 = 2 * c, j1 = 2 * (3 + c);
        const int r2 = 2 * (6 + c), r3 = 2 * (9 + c);
        const f2 p = S > 0 ? sc[c] : nsc[c], m = S > 0 ? nsc[c] : sc[c]; /* +S and -S times the scale */
        acc[j0] = f2_fma(sc[c], w[j0], acc[j0]);
        acc[j0 + 1] = f2_fma(sc[c], w[j0 + 1], acc[j0 + 1]);
        acc[j1] = f2_fma(sc[c], w[j1], acc[j1]);
        acc[j1 + 1] = f2_fma(sc[c], w[j1 + 1], acc[j1 + 1]);
        if (MU == 0) {
            acc[r2] = f2_fma(p, w[j1 + 1], acc[r2]);
            acc[r2 + 1] = f2_fma(m, w[j1], acc[r2 + 1]);
            acc[r3] = f2_fma(p, w[j0 + 1], acc[r3]);
            acc[r3 + 1] = f2_fma(m, w[j0], acc[r3 + 1]);
        } else if (MU == 1) {
            acc[r2] = f2_fma(p, w[j1], acc[r2]);
            acc[r2 + 1] = f2_fma(p, w[j1 + 1], acc[r2 + 1]);
            acc[r3] = f2_fma(m, w[j0], acc[r3]);
            acc[r3 + 1] = f2_fma(m, w[j0 + 1], acc[r3 + 1]);
        } else if (MU == 2) {
            acc[r2] = f2_fma(p, w[j0 + 1], acc[r2]);
            acc[r2 + 1] = f2_fma(m, w[j0], acc[r2 + 1]);
            acc[r3] = f2_fma(m, w[j1 + 1], acc[r3]);
            acc[r3 + 1] = f2_fma(p, w[j1], acc[r3 + 1]);
        } else {
            acc[r2] = f2_fma(p, w[j0], acc[r2]);
            acc[r2 + 1] = f2_fma(p, w[j0 + 1], acc[r2 + 1]);
            acc[r3] = f2_fma(p, w[j1], acc[r3]);
            acc[r3 + 1] = f2_fma(p, w[j1 + 1], acc[r3 + 1]);
        }
    }
}

/* ---- w_j = scale * U h_j (ADJ = 0) or scale * U^dag h_j (ADJ = 1), j = 0,1 (colour_mul) -----
 * re += ur hr - ui hi, im += ur hi + ui hr; U^dag takes conj(U_ba).  The subtraction runs on a
 * negated copy of the half spinor's imaginary (ADJ: real) parts: 6 negations per direction. */
template <int ADJ, bool SCALE = true> __device__ __forceinline__ void colour_mul2(f2 (&w)[12], const f2 (&u)[18], const f2 (&h)[12], f2 scale)
{
    f2 n[6]; /* ADJ = 0: -Im h_{j,b} ; ADJ = 1: -Re h_{j,b} */
#pragma unroll
    for (int k = 0; k < 6; k++) n[k] = f2_neg(h[2 * k + (ADJ ? 0 : 1)]);
#pragma unroll
    for (int j = 0; j < 2; j++)
#pragma unroll
        for (int a = 0; a < 3; a++) {
            f2 re, im;
#pragma unroll
            for (int b = 0; b < 3; b++) {
                const int k = ADJ ? 2 * (3 * b + a) : 2 * (3 * a + b);
                const f2 ur = u[k], ui = u[k + 1]; /* the stored imaginary part */
                const f2 hr = h[2 * (3 * j + b)], hi = h[2 * (3 * j + b) + 1], nn = n[3 * j + b];
                if (!ADJ) { /* re += ur hr + ui (-hi) ; im += ur hi + ui hr */
                    re = b == 0 ? ur * hr : f2_fma(ur, hr, re);
                    re = f2_fma(ui, nn, re);
                    im = b == 0 ? ur * hi : f2_fma(ur, hi, im);
                    im = f2_fma(ui, hr, im);
                } else { /* conj: re += ur hr + ui hi ; im += ur hi + ui (-hr) */
                    re = b == 0 ? ur * hr : f2_fma(ur, hr, re);
                    re = f2_fma(ui, hi, re);
                    im = b == 0 ? ur * hi : f2_fma(ur, hi, im);
                    im = f2_fma(ui, nn, im);
                }
            }
            w[2 * (3 * j + a)] = SCALE ? scale * re : re;
            w[2 * (3 * j + a) + 1] = SCALE ? scale * im : im;
        }
}

/* ---- row2 = d * conj(row0 x row1) (reconstruct_row2; reading S7), d a common factor --------- */
template <bool SCALE = true> __device__ __forceinline__ void reconstruct_row2_2(f2 (&u)[18], f2 d)
{
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
        const f2 ar = u[2 * c1], ai = u[2 * c1 + 1], br = u[6 + 2 * c2], bi = u[6 + 2 * c2 + 1];
        const f2 cr = u[2 * c2], ci = u[2 * c2 + 1], dr = u[6 + 2 * c1], di = u[6 + 2 * c1 + 1];
        /* re = ar br - ai bi - cr dr + ci di ; im = ar bi + ai br - cr di - ci dr ; row2 = (re, -im) */
        const f2 p = f2_fma(ci, di, ar * br), q = f2_fma(cr, dr, ai * bi);
        const f2 r = f2_fma(ai, br, ar * bi), t = f2_fma(ci, dr, cr * di);
        u[12 + 2 * c] = SCALE ? d * (p - q) : p - q;
        u[12 + 2 * c + 1] = SCALE ? d * (t - r) : t - r;
    }
}

/* ---- packed Hermitian 6x6 block times 6-vector (clover_block_apply) ---------
 * c = 36 reals of one block: 6 real diagonal, then the 15 complex lower-triangle entries. */
__device__ __forceinline__ void clover_block_apply2(f2* o, const f2* c, const f2* v)
{
    f2 nv[12];
#pragma unroll
    for (int k = 0; k < 12; k++) nv[k] = f2_neg(v[k]);
#pragma unroll
    for (int i = 0; i < 6; i++) {
        f2 re = c[i] * v[2 * i], im = c[i] * v[2 * i + 1];
#pragma unroll
        for (int j = 0; j < 6; j++) {
            if (j == i) continue;
            const int hi = i > j ? i : j, lo = i > j ? j : i;
            const int k = 6 + 2 * (5 * lo - (lo * (lo - 1)) / 2 + (hi - lo - 1));
            const f2 lr = c[k], li = c[k + 1];
            re = f2_fma(lr, v[2 * j], re);
            im = f2_fma(lr, v[2 * j + 1], im);
            if (i > j) { /* entry L_ij: re -= li vi ; im += li vr */
                re = f2_fma(li, nv[2 * j + 1], re);
                im = f2_fma(li, v[2 * j], im);
            } else { /* entry conj(L_ji): re += li vi ; im -= li vr */
                re = f2_fma(li, v[2 * j + 1], re);
                im = f2_fma(li, nv[2 * j], im);
            }
        }
        o[2 * i] = re;
        o[2 * i + 1] = im;
    }
}

#endif
