/*
 * hop_half.cu -- the hopping-term kernel with 16-bit storage of everything it streams
 * (reading H1): links, clover, the input spinor, the operand z and
 * (unless OUT_F32) the output are int16 codes + per-site norms, arithmetic is fp32 and
 * is the same code as the fp32 kernel (hop_site / clover_block_apply of hop_kernel.cuh).
 * Algorithmic bytes per site: 52 in + 8 x 24 links + 52 (or 96) out = 296 (340) for the
 * plain hop against 576 in fp32; +148 per clover block pair, +52 for z.
 */
#include "half_device.cuh"
#include "hop_kernel.cuh"
#include "packed_math.cuh"

namespace {

struct HalfHopArgs {
    unsigned char* out;
    const unsigned char* in;
    const unsigned char* z;
    const unsigned char* gauge;
    const unsigned char* clover;
    size_t gblock;
    DevGeom geo;
    int parity;
    float tb, a, b;
    const int* halt; /* the launch does nothing while *halt != 0 (NULL: always run) */
};

__device__ __forceinline__ void half_clover_apply(float (&o)[24], const unsigned char* clov, size_t Vh, size_t cb, const float (&v)[24])
{
#pragma unroll
    for (int b = 0; b < 2; b++) {
        float c[36];
        half_load_clover_block(c, clov, Vh, cb, b);
        clover_block_apply<float>(&o[12 * b], c, &v[12 * b]);
    }
}

#ifndef HOP_MINBLOCKS_HALF
#define HOP_MINBLOCKS_HALF 8 /* blocks of 64 threads = 128 sites; swept with the depth on B200 (Wilson Mhat, 2 launches):
                              (depth 1, 8 blocks) 213 us, (1,6) 223, (2,6) 223, (2,5) 223, (3,4) 231, (2,4) 248 */
#endif
#ifndef HOP_HALF_DEPTH
#define HOP_HALF_DEPTH 1 /* directions whose loads are in flight ahead of the arithmetic */
#endif
/* Round 2, tried and dropped (profiles/hop_half_r2.md): a loop over mu with a 4-way switch around the projection and
 * the spin reconstruction, two raw buffers in ping-pong (to bring the 50 KB body under the 32 KB instruction-cache
 * level: ncu shows 0.66 - 0.9 warps per issue waiting for instructions).  ptxas then keeps part of the accumulator in
 * local memory (600 - 830 B of spills, 164 LDL + 109 STL in the body) and the Wilson Mhat takes 359 us against 199 us. */

/* The undecoded words of one direction: neighbour spinor (3 x int4 + norm) and link (int4 + int2),
 * 19 registers.  The 16-bit kernel moves half the bytes of the fp32 one per load instruction, so
 * it needs more loads in flight to cover the same DRAM latency: the loads of HOP_HALF_DEPTH
 * directions are issued before the first one is decoded, and each slot is refilled as soon
 * as it has been consumed (ncu before this: 45 % of the stall samples were long-scoreboard
 * waits at the first use of each direction's data). */
struct HalfRaw {
    int4 q0, q1, q2, la;
    int2 lb;
    float n;
};

template <int MU, int DIR>
__device__ __forceinline__ void half_load_raw(HalfRaw& r, const HalfHopArgs& A, size_t Vh, int cb, int nb_cb)
{
    const int4* q = reinterpret_cast<const int4*>(A.in) + nb_cb;
    r.q0 = __ldg(q);
    r.q1 = __ldg(q + Vh);
    r.q2 = __ldg(q + 2 * Vh);
    r.n = __ldg(reinterpret_cast<const float*>(A.in + Vh * 48) + nb_cb);
    const unsigned char* blk = A.gauge + (size_t)(2 * MU + (DIR > 0 ? A.parity : 1 - A.parity)) * A.gblock;
    const size_t i = (size_t)(DIR > 0 ? cb : nb_cb);
    r.la = __ldg(reinterpret_cast<const int4*>(blk) + i);
    r.lb = __ldg(reinterpret_cast<const int2*>(blk + Vh * 16) + i);
}

/* ---- two sites per thread on packed fp32 pairs (packed_math.cuh) ------------------------------
 * lane A = site cbA, lane B = site cbB.  A decoded code needs one PRMT whichever register it
 * lands in, so pairing the two sites' values costs nothing; every arithmetic instruction then
 * serves both sites. */
__device__ __forceinline__ void half_int2x2(int wa, int wb, f2& lo, f2& hi)
{
    const unsigned xa = (unsigned)wa ^ 0x80008000u, xb = (unsigned)wb ^ 0x80008000u;
    const f2 m = f2_set1(8421376.0f);
    lo = f2_bits(__byte_perm(xa, 0x4B00u, 0x5410), __byte_perm(xb, 0x4B00u, 0x5410)) - m;
    hi = f2_bits(__byte_perm(xa, 0x4B00u, 0x5432), __byte_perm(xb, 0x4B00u, 0x5432)) - m;
}
__device__ __forceinline__ void half_int8x2(const int4& a, const int4& b, f2* o)
{
    half_int2x2(a.x, b.x, o[0], o[1]);
    half_int2x2(a.y, b.y, o[2], o[3]);
    half_int2x2(a.z, b.z, o[4], o[5]);
    half_int2x2(a.w, b.w, o[6], o[7]);
}

/* The 24 codes of the two sites' neighbour spinors as undecoded floats (packed_math.cuh,
 * project2_codes): real index i = code i of the site = half (i & 1) of word i / 2.  The words are
 * turned to offset binary (x = w ^ 0x80008000) and, for the lower spin components, also negated per
 * 16-bit half in the integer domain (0x10000 - x: no half is 0, codes are clamped to +-32767, so no
 * borrow crosses the halves); one PRMT drops a half into the mantissa of 2^23. */
struct HalfCodes2 {
    unsigned xa[12], xb[12], na[6], nb[6];
    __device__ __forceinline__ HalfCodes2(const HalfRaw& ra, const HalfRaw& rb)
    {
        const int wa[12] = {ra.q0.x, ra.q0.y, ra.q0.z, ra.q0.w, ra.q1.x, ra.q1.y, ra.q1.z, ra.q1.w, ra.q2.x, ra.q2.y, ra.q2.z, ra.q2.w};
        const int wb[12] = {rb.q0.x, rb.q0.y, rb.q0.z, rb.q0.w, rb.q1.x, rb.q1.y, rb.q1.z, rb.q1.w, rb.q2.x, rb.q2.y, rb.q2.z, rb.q2.w};
#pragma unroll
        for (int k = 0; k < 12; k++) {
            xa[k] = (unsigned)wa[k] ^ 0x80008000u;
            xb[k] = (unsigned)wb[k] ^ 0x80008000u;
        }
#pragma unroll
        for (int k = 0; k < 6; k++) {
            na[k] = 0x10000u - xa[6 + k];
            nb[k] = 0x10000u - xb[6 + k];
        }
    }
    static __device__ __forceinline__ unsigned half_of(unsigned w, int hi) { return __byte_perm(w, 0x4B00u, hi ? 0x5432 : 0x5410); }
    /* M + code i */
    __device__ __forceinline__ f2 pos(int i) const { return f2_bits(half_of(xa[i >> 1], i & 1), half_of(xb[i >> 1], i & 1)); }
    /* M - code i (i >= 12: only the lower spin components are ever wanted negated) */
    __device__ __forceinline__ f2 neg(int i) const { return f2_bits(half_of(na[(i >> 1) - 6], i & 1), half_of(nb[(i >> 1) - 6], i & 1)); }
};

template <int MU, int DIR, int SG>
__device__ __forceinline__ void half_compute_raw2(f2 (&acc)[24], const HalfRaw& ra, const HalfRaw& rb, f2 sign)
{
    f2 u[18], h[12], w[12];
    half_int8x2(ra.la, rb.la, &u[0]);
    half_int2x2(ra.lb.x, rb.lb.x, u[8], u[9]);
    half_int2x2(ra.lb.y, rb.lb.y, u[10], u[11]);
    /* rows 0,1 stay codes (value x 32767), row 2 = conj(row0 x row1) of the codes (value x 32767^2) */
    reconstruct_row2_2<false>(u, f2_set1(1.f));
    const HalfCodes2 codes(ra, rb);
    project2_codes<MU, SG>(h, codes);
    const f2 d = f2_set1(1.0f / 32767.0f);
    if (DIR < 0) {
        /* U^dag mixes row 2 into every output: bring the colour-2 inputs to the scale of the others instead */
        h[4] = h[4] * d; h[5] = h[5] * d; h[10] = h[10] * d; h[11] = h[11] * d;
    }
    colour_mul2<(DIR < 0), false>(w, u, h, d);
    /* codes -> values once, folded into the accumulation: norm / 32767 / 32767 (the division is a
     * multiplication by the rounded reciprocal: one ulp, inside the arithmetic's own rounding; the format's
     * exact n / 32767 is kept where stored values are read back as such).  U h: colour 2 of the result
     * comes from row 2 and carries one more factor 32767. */
    const f2 s01 = sign * f2_make(ra.n, rb.n) * f2_set1((1.0f / 32767.0f) * (1.0f / 32767.0f));
    const f2 s2 = DIR < 0 ? s01 : s01 * d;
    const f2 sc[3] = {s01, s01, s2};
    const f2 n01 = f2_neg(s01), n2 = DIR < 0 ? n01 : f2_neg(s2);
    const f2 nsc[3] = {n01, n01, n2};
    reconstruct_add2_scaled<MU, SG>(acc, w, sc, nsc);
}

/* the stored values code * (norm / 32767) of the two sites' spinors */
__device__ __forceinline__ void half_load_values2(f2 (&v)[24], const unsigned char* block, size_t Vh, int ia, int ib)
{
    const int4* q = reinterpret_cast<const int4*>(block);
    const float* nrm = reinterpret_cast<const float*>(block + Vh * 48);
    const f2 d = f2_make(__fdiv_rn(__ldg(nrm + ia), 32767.0f), __fdiv_rn(__ldg(nrm + ib), 32767.0f));
#pragma unroll
    for (int c = 0; c < 3; c++) half_int8x2(__ldg(q + (size_t)c * Vh + ia), __ldg(q + (size_t)c * Vh + ib), &v[8 * c]);
#pragma unroll
    for (int k = 0; k < 24; k++) v[k] = v[k] * d;
}

__device__ __forceinline__ void half_clover_apply2(f2 (&o)[24], const unsigned char* clov, size_t Vh, int ia, int ib, const f2 (&v)[24])
{
    const int4* q = reinterpret_cast<const int4*>(clov);
    const float* nrm = reinterpret_cast<const float*>(clov + Vh * 144);
    const f2 d = f2_make(__fdiv_rn(__ldg(nrm + ia), 32767.0f), __fdiv_rn(__ldg(nrm + ib), 32767.0f));
#pragma unroll
    for (int b = 0; b < 2; b++) {
        f2 t[40];
#pragma unroll
        for (int k = 0; k < 5; k++)
            half_int8x2(__ldg(q + (size_t)(4 * b + k) * Vh + ia), __ldg(q + (size_t)(4 * b + k) * Vh + ib), &t[8 * k]);
        /* block 1 starts at code 36 = chunk 4, offset 4; the site's scale multiplies the 12 results */
        clover_block_apply2(&o[12 * b], &t[4 * b], &v[12 * b]);
#pragma unroll
        for (int k = 0; k < 12; k++) o[12 * b + k] = o[12 * b + k] * d;
    }
}

/* 16-bit store of one lane (site idx); codes by the rule of half_store_spinor, computed packed */
__device__ __forceinline__ void half_store2(unsigned char* block, size_t Vh, int ia, int ib, bool store_b, const f2 (&v)[24])
{
    float na = 0.f, nb = 0.f;
#pragma unroll
    for (int k = 0; k < 24; k++) {
        float x, y;
        f2_get(v[k], x, y);
        na = fmaxf(na, fabsf(x));
        nb = fmaxf(nb, fabsf(y));
    }
    const f2 scale = f2_make(na > 0.f ? __fdiv_rn(32767.0f, na) : 0.f, nb > 0.f ? __fdiv_rn(32767.0f, nb) : 0.f);
    const f2 magic = f2_set1(12582912.0f);
    unsigned ca[24], cb[24];
#pragma unroll
    for (int k = 0; k < 24; k++) f2_get_bits(v[k] * scale + magic, ca[k], cb[k]);
    int4* q = reinterpret_cast<int4*>(block);
    float* nrm = reinterpret_cast<float*>(block + Vh * 48);
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const int k = 8 * c;
        q[(size_t)c * Vh + ia] = make_int4((int)__byte_perm(ca[k], ca[k + 1], 0x5410), (int)__byte_perm(ca[k + 2], ca[k + 3], 0x5410),
                                           (int)__byte_perm(ca[k + 4], ca[k + 5], 0x5410), (int)__byte_perm(ca[k + 6], ca[k + 7], 0x5410));
        if (store_b)
            q[(size_t)c * Vh + ib] = make_int4((int)__byte_perm(cb[k], cb[k + 1], 0x5410), (int)__byte_perm(cb[k + 2], cb[k + 3], 0x5410),
                                               (int)__byte_perm(cb[k + 4], cb[k + 5], 0x5410), (int)__byte_perm(cb[k + 6], cb[k + 7], 0x5410));
    }
    nrm[ia] = na;
    if (store_b) nrm[ib] = nb;
}

#define HALF_LOAD(k, MU, DIR, NB)                                          \
    do {                                                                   \
        half_load_raw<MU, DIR>(rawa[(k) % D], A, Vh, cba, na.NB);          \
        half_load_raw<MU, DIR>(rawb[(k) % D], A, Vh, cbb, nbb.NB);         \
    } while (0)
#define HALF_COMP(k, MU, DIR, SG, SIGN) half_compute_raw2<MU, DIR, SG>(acc, rawa[(k) % D], rawb[(k) % D], SIGN)

template <int DAG, int MODE, int OUT_F32>
__global__ void __launch_bounds__(64, HOP_MINBLOCKS_HALF) hop_half_kernel(const HalfHopArgs A)
{
    pdl_launch_dependents(); /* launched with launch_pdl (qcd_device.cuh) */
    pdl_wait();
    if (A.halt && *reinterpret_cast<const volatile int*>(A.halt) != 0) return;
    /* a block of 64 threads works on 128 consecutive sites: thread t on base + t and base + 64 + t */
    const int cba = blockIdx.x * 128 + threadIdx.x;
    if (cba >= A.geo.Vh) return;
    const bool has_b = cba + 64 < A.geo.Vh;
    const int cbb = has_b ? cba + 64 : cba; /* ragged tail: lane B repeats lane A and is not stored */
    const size_t Vh = (size_t)A.geo.Vh;
    const Neighbours<float> na(A.geo, cba, A.parity, A.tb), nbb(A.geo, cbb, A.parity, A.tb);
    constexpr int SF = DAG ? +1 : -1; /* forward hop carries (1 - g_mu), the adjoint swaps (O4) */
    constexpr int SB = DAG ? -1 : +1;
    constexpr int D = HOP_HALF_DEPTH;
    const f2 one = f2_set1(1.f);
    f2 acc[24];
#pragma unroll
    for (int i = 0; i < 24; i++) acc[i].v = 0ull;
    HalfRaw rawa[D], rawb[D];
    /* direction k: 0 x+, 1 x-, 2 y+, 3 y-, 4 z+, 5 z-, 6 t+, 7 t-; load k + D follows compute k */
    if (0 < D) HALF_LOAD(0, 0, +1, xp);
    if (1 < D) HALF_LOAD(1, 0, -1, xm);
    if (2 < D) HALF_LOAD(2, 1, +1, yp);
    if (3 < D) HALF_LOAD(3, 1, -1, ym);
    HALF_COMP(0, 0, +1, SF, one);
    if (D == 1) HALF_LOAD(1, 0, -1, xm);
    if (D == 2) HALF_LOAD(2, 1, +1, yp);
    if (D == 3) HALF_LOAD(3, 1, -1, ym);
    if (D == 4) HALF_LOAD(4, 2, +1, zp);
    HALF_COMP(1, 0, -1, SB, one);
    if (D == 1) HALF_LOAD(2, 1, +1, yp);
    if (D == 2) HALF_LOAD(3, 1, -1, ym);
    if (D == 3) HALF_LOAD(4, 2, +1, zp);
    if (D == 4) HALF_LOAD(5, 2, -1, zm);
    HALF_COMP(2, 1, +1, SF, one);
    if (D == 1) HALF_LOAD(3, 1, -1, ym);
    if (D == 2) HALF_LOAD(4, 2, +1, zp);
    if (D == 3) HALF_LOAD(5, 2, -1, zm);
    if (D == 4) HALF_LOAD(6, 3, +1, tp);
    HALF_COMP(3, 1, -1, SB, one);
    if (D == 1) HALF_LOAD(4, 2, +1, zp);
    if (D == 2) HALF_LOAD(5, 2, -1, zm);
    if (D == 3) HALF_LOAD(6, 3, +1, tp);
    if (D == 4) HALF_LOAD(7, 3, -1, tm);
    HALF_COMP(4, 2, +1, SF, one);
    if (D == 1) HALF_LOAD(5, 2, -1, zm);
    if (D == 2) HALF_LOAD(6, 3, +1, tp);
    if (D == 3) HALF_LOAD(7, 3, -1, tm);
    HALF_COMP(5, 2, -1, SB, one);
    if (D == 1) HALF_LOAD(6, 3, +1, tp);
    if (D == 2) HALF_LOAD(7, 3, -1, tm);
    HALF_COMP(6, 3, +1, SF, f2_make(na.sgn_tp, nbb.sgn_tp));
    if (D == 1) HALF_LOAD(7, 3, -1, tm);
    HALF_COMP(7, 3, -1, SB, f2_make(na.sgn_tm, nbb.sgn_tm));

    if (MODE == HOP_XPAY || MODE == HOP_CLOVER_Z) {
        f2 zz[24];
        half_load_values2(zz, A.z, Vh, cba, cbb);
        const f2 ca = f2_set1(A.a), cb = f2_set1(A.b);
        if (MODE == HOP_CLOVER_Z) {
            f2 az[24];
            half_clover_apply2(az, A.clover, Vh, cba, cbb, zz);
#pragma unroll
            for (int i = 0; i < 24; i++) acc[i] = f2_fma(ca, az[i], cb * acc[i]);
        } else {
#pragma unroll
            for (int i = 0; i < 24; i++) acc[i] = f2_fma(ca, zz[i], cb * acc[i]);
        }
    } else if (MODE == HOP_CLOVER_OUT) {
        f2 o[24];
        half_clover_apply2(o, A.clover, Vh, cba, cbb, acc);
#pragma unroll
        for (int i = 0; i < 24; i++) acc[i] = o[i];
    }
    if (OUT_F32) {
        float va[24], vb[24];
#pragma unroll
        for (int i = 0; i < 24; i++) f2_get(acc[i], va[i], vb[i]);
        store_planes<float, 24>(reinterpret_cast<float*>(A.out), Vh, (size_t)cba, va);
        if (has_b) store_planes<float, 24>(reinterpret_cast<float*>(A.out), Vh, (size_t)cbb, vb);
    } else {
        half_store2(A.out, Vh, cba, cbb, has_b, acc);
    }
}

template <int DAG, int MODE> cudaError_t launch_mode(const HalfHopArgs& A, int out_f32, cudaStream_t st)
{
    const int threads = 64, blocks = (A.geo.Vh + 127) / 128;
    if (out_f32) launch_pdl(hop_half_kernel<DAG, MODE, 1>, blocks, threads, st, A);
    else launch_pdl(hop_half_kernel<DAG, MODE, 0>, blocks, threads, st, A);
    return cudaGetLastError();
}
template <int DAG> cudaError_t launch_dag(const HalfHopArgs& A, int mode, int out_f32, cudaStream_t st)
{
    switch (mode) {
    case HOP_PLAIN: return launch_mode<DAG, HOP_PLAIN>(A, out_f32, st);
    case HOP_XPAY: return launch_mode<DAG, HOP_XPAY>(A, out_f32, st);
    case HOP_CLOVER_Z: return launch_mode<DAG, HOP_CLOVER_Z>(A, out_f32, st);
    case HOP_CLOVER_OUT: return launch_mode<DAG, HOP_CLOVER_OUT>(A, out_f32, st);
    default: return cudaErrorInvalidValue;
    }
}

/* fp32 internal blocks <-> 16-bit blocks; one thread per (block, cb) */
template <int TO_HALF> __global__ void half_convert_kernel(unsigned char* half, float* f32, size_t Vh, int nblocks)
{
    pdl_launch_dependents();
    pdl_wait();
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= Vh * (size_t)nblocks) return;
    const size_t blk = i / Vh, cb = i - blk * Vh;
    float v[24];
    if (TO_HALF) {
        load_planes_rw<float, 24>(v, f32 + blk * 24 * Vh, Vh, cb);
        half_store_spinor(half + blk * HALF_SPINOR_BYTES * Vh, Vh, cb, v);
    } else {
        const HalfSpinor s = {half + blk * HALF_SPINOR_BYTES * Vh, Vh};
        s.load_values(v, (int)cb);
        store_planes<float, 24>(f32 + blk * 24 * Vh, Vh, cb, v);
    }
}

/* p = a r + b p (fp32; p_is_zero: p not read) ; ph = store16(p).  a, b: host values or quotients of
 * device doubles, rounded to fp32 (reading O7: beta = (float)(rho'/rho)) */
__global__ void xpay_q16_kernel(DevScalar as, const float* r, DevScalar bs, int p_is_zero, float* p, unsigned char* ph, size_t Vh, int nblocks,
                                const int* halt)
{
    pdl_launch_dependents();
    pdl_wait();
    if (halt && *reinterpret_cast<const volatile int*>(halt) != 0) return;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= Vh * (size_t)nblocks) return;
    const float a = (float)(as.num ? as.sign * (*as.num / *as.den) : as.val);
    const float b = p_is_zero ? 0.f : (float)(bs.num ? bs.sign * (*bs.num / *bs.den) : bs.val);
    const size_t blk = i / Vh, cb = i - blk * Vh;
    float rv[24], pv[24];
    load_planes_rw<float, 24>(rv, r + blk * 24 * Vh, Vh, cb);
    if (!p_is_zero) {
        load_planes_rw<float, 24>(pv, p + blk * 24 * Vh, Vh, cb);
#pragma unroll
        for (int k = 0; k < 24; k++) pv[k] = a * rv[k] + b * pv[k];
    } else {
#pragma unroll
        for (int k = 0; k < 24; k++) pv[k] = a * rv[k];
    }
    store_planes<float, 24>(p + blk * 24 * Vh, Vh, cb, pv);
    half_store_spinor(ph + blk * HALF_SPINOR_BYTES * Vh, Vh, cb, pv);
}

} // namespace

int hop_half_launch(qcd_ctx* ctx, const qcd_gauge* g, const HopLaunch& L, int out_f32)
{
    HalfHopArgs A;
    A.out = (unsigned char*)L.out;
    A.in = (const unsigned char*)L.in;
    A.z = (const unsigned char*)L.z;
    A.gauge = (const unsigned char*)g->data;
    A.clover = (const unsigned char*)L.clover;
    A.gblock = g->block_bytes;
    A.geo = dev_geom(g->geo);
    A.parity = L.out_parity;
    A.tb = (float)g->tb;
    A.a = (float)L.a;
    A.b = (float)L.b;
    A.halt = L.halt;
    cudaError_t e = L.dagger ? launch_dag<1>(A, L.mode, out_f32, ctx->stream) : launch_dag<0>(A, L.mode, out_f32, ctx->stream);
    if (e != cudaSuccess) return qcd_set_error(QCD_ECUDA, "half hop launch: %s", cudaGetErrorString(e));
    ctx->launches++;
    return QCD_OK;
}

int half_convert(qcd_ctx* ctx, void* half, void* f32, size_t Vh, int nblocks, int to_half)
{
    const size_t n = Vh * (size_t)nblocks;
    const int threads = 128, blocks = (int)((n + threads - 1) / threads);
    if (to_half) launch_pdl(half_convert_kernel<1>, blocks, threads, ctx->stream, (unsigned char*)half, (float*)f32, Vh, nblocks);
    else launch_pdl(half_convert_kernel<0>, blocks, threads, ctx->stream, (unsigned char*)half, (float*)f32, Vh, nblocks);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return qcd_set_error(QCD_ECUDA, "half convert: %s", cudaGetErrorString(e));
    ctx->launches++;
    return QCD_OK;
}

int half_xpay_store(qcd_ctx* ctx, DevScalar a, const void* r, DevScalar b, int p_is_zero, void* p, void* ph, size_t Vh, int nblocks,
                    const int* halt)
{
    const size_t n = Vh * (size_t)nblocks;
    const int threads = 128, blocks = (int)((n + threads - 1) / threads);
    launch_pdl(xpay_q16_kernel, blocks, threads, ctx->stream, a, (const float*)r, b, p_is_zero, (float*)p, (unsigned char*)ph, Vh, nblocks, halt);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return qcd_set_error(QCD_ECUDA, "half xpay: %s", cudaGetErrorString(e));
    ctx->launches++;
    return QCD_OK;
}
