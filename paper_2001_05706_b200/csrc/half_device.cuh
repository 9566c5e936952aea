/*
 * half_device.cuh -- the 16-bit fixed-point storage format of the low-precision operator
 * (PAPER.md:163 ref. [1]; reading H1 in DESIGN.md).
 *
 *   spinor, one parity block : int4 q[3][Vh] (24 int16 codes per site, code k of chunk k/8)
 *                              then float norm[Vh]                      -> 52 B / site
 *                              value = (float)code * (norm / 32767.0f), code = rintf(v * (32767.0f / norm))
 *   gauge (mu, parity) block : int4 a[Vh] (reals 0..7 of rows 0,1) then int2 b[Vh] (reals 8..11)
 *                              value = (float)code * (1.0f/32767.0f)    -> 24 B / link
 *   clover (which, parity)   : int4 c[9][Vh] (72 codes, packed order of qcd_internal.h) then
 *                              float norm[Vh]                           -> 148 B / site
 * Arithmetic is fp32; only storage is 16-bit.
 */
#ifndef QCD_HALF_DEVICE_CUH
#define QCD_HALF_DEVICE_CUH

#include "qcd_device.cuh"

constexpr size_t HALF_SPINOR_BYTES = 52;  /* per site */
constexpr size_t HALF_LINK_BYTES = 24;
constexpr size_t HALF_CLOVER_BYTES = 148;

/* (float)code without I2F (an XU instruction, 16 lanes/clk/SM): code + 32768 in the low
 * mantissa bits of 2^23 is the float 2^23 + 32768 + code; the subtraction is exact. */
__device__ __forceinline__ void half_int2(int w, float& lo, float& hi)
{
    const unsigned x = (unsigned)w ^ 0x80008000u;
#ifdef QCD_HALF_NO_F32X2
    lo = __uint_as_float(__byte_perm(x, 0x4B00u, 0x5410)) - 8421376.0f;
    hi = __uint_as_float(__byte_perm(x, 0x4B00u, 0x5432)) - 8421376.0f;
#else
    /* both halves in one packed add (sm_100 add.f32x2: one issue slot for two lanes) */
    unsigned long long p, m, r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(p) : "r"(__byte_perm(x, 0x4B00u, 0x5410)), "r"(__byte_perm(x, 0x4B00u, 0x5432)));
    asm("mov.b64 %0, {%1, %1};" : "=l"(m) : "f"(-8421376.0f));
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(p), "l"(m));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(r));
#endif
}
__device__ __forceinline__ void half_int8(const int4& w, float* o)
{
    half_int2(w.x, o[0], o[1]);
    half_int2(w.y, o[2], o[3]);
    half_int2(w.z, o[4], o[5]);
    half_int2(w.w, o[6], o[7]);
}
__device__ __forceinline__ void half_unpack2(int w, float d, float& lo, float& hi)
{
    half_int2(w, lo, hi);
    lo *= d;
    hi *= d;
}
__device__ __forceinline__ void half_unpack8(const int4& w, float d, float* o)
{
    half_unpack2(w.x, d, o[0], o[1]);
    half_unpack2(w.y, d, o[2], o[3]);
    half_unpack2(w.z, d, o[4], o[5]);
    half_unpack2(w.w, d, o[6], o[7]);
}
/* rintf(v * scale) for |v * scale| < 2^22 without F2I: adding 1.5 * 2^23 rounds to the nearest
 * (even) integer and leaves its two's complement in the low mantissa bits.  The product is
 * rounded to fp32 first (no fma), as the format's definition has it.  No clamp: callers
 * guarantee |v| * scale <= 32767 (scale = 32767 / max|v|). */
__device__ __forceinline__ int half_pack2_fast(float lo, float hi, float scale)
{
    const unsigned a = __float_as_uint(__fadd_rn(__fmul_rn(lo, scale), 12582912.0f));
    const unsigned b = __float_as_uint(__fadd_rn(__fmul_rn(hi, scale), 12582912.0f));
    return (int)__byte_perm(a, b, 0x5410);
}
__device__ __forceinline__ int4 half_pack8_fast(const float* v, float scale)
{
    return make_int4(half_pack2_fast(v[0], v[1], scale), half_pack2_fast(v[2], v[3], scale),
                     half_pack2_fast(v[4], v[5], scale), half_pack2_fast(v[6], v[7], scale));
}
__device__ __forceinline__ int half_code(float v, float scale)
{
    int c = __float2int_rn(v * scale);
    return max(-32767, min(32767, c));
}
__device__ __forceinline__ int half_pack2(float lo, float hi, float scale)
{
    return (half_code(lo, scale) & 0xffff) | (half_code(hi, scale) << 16);
}
__device__ __forceinline__ int4 half_pack8(const float* v, float scale)
{
    return make_int4(half_pack2(v[0], v[1], scale), half_pack2(v[2], v[3], scale), half_pack2(v[4], v[5], scale),
                     half_pack2(v[6], v[7], scale));
}

struct HalfSpinor {
    const unsigned char* block;
    size_t Vh;
    /* the stored values, bit for bit: code * (norm / 32767) */
    __device__ __forceinline__ void load_values(float (&s)[24], int idx) const
    {
        const int4* q = reinterpret_cast<const int4*>(block) + idx;
        const float n = __ldg(reinterpret_cast<const float*>(block + Vh * 48) + idx);
        const float d = __fdiv_rn(n, 32767.0f);
#pragma unroll
        for (int c = 0; c < 3; c++) half_unpack8(__ldg(q + (size_t)c * Vh), d, &s[8 * c]);
    }
    /* the codes as floats; returns the factor norm / 32767 still to be applied (the hop applies
     * it once to the colour-multiplied half spinor: 12 multiplications instead of 24) */
    __device__ __forceinline__ float load(float (&s)[24], int idx) const
    {
        const int4* q = reinterpret_cast<const int4*>(block) + idx;
        const float n = __ldg(reinterpret_cast<const float*>(block + Vh * 48) + idx);
#pragma unroll
        for (int c = 0; c < 3; c++) half_int8(__ldg(q + (size_t)c * Vh), &s[8 * c]);
        return __fdiv_rn(n, 32767.0f);
    }
};

__device__ __forceinline__ void half_store_spinor(unsigned char* block, size_t Vh, size_t idx, const float (&v)[24])
{
    float n = 0.f;
#pragma unroll
    for (int k = 0; k < 24; k++) n = fmaxf(n, fabsf(v[k]));
    const float scale = n > 0.f ? __fdiv_rn(32767.0f, n) : 0.f;
    int4* q = reinterpret_cast<int4*>(block) + idx;
#pragma unroll
    for (int c = 0; c < 3; c++) q[(size_t)c * Vh] = half_pack8_fast(&v[8 * c], scale);
    reinterpret_cast<float*>(block + Vh * 48)[idx] = n;
}

struct HalfLinks {
    const unsigned char* gauge;
    size_t gblock; /* bytes per (mu, parity) block */
    size_t Vh;
    int parity;
    /* rows 0,1 as codes (scale 32767), row 2 = conj(row0 x row1) / 32767 on the same scale;
     * returns the factor 1/32767 still to be applied */
    template <int MU, int DIR> __device__ __forceinline__ float get(float (&u)[18], int cb, int nb_cb) const
    {
        const unsigned char* blk = gauge + (size_t)(2 * MU + (DIR > 0 ? parity : 1 - parity)) * gblock;
        const size_t i = (size_t)(DIR > 0 ? cb : nb_cb);
        const int4 a = __ldg(reinterpret_cast<const int4*>(blk) + i);
        const int2 b = __ldg(reinterpret_cast<const int2*>(blk + Vh * 16) + i);
        const float d = 1.0f / 32767.0f;
        half_int8(a, &u[0]);
        half_int2(b.x, u[8], u[9]);
        half_int2(b.y, u[10], u[11]);
        reconstruct_row2<float>(u);
#pragma unroll
        for (int k = 12; k < 18; k++) u[k] *= d;
        return d;
    }
};

/* 36 reals of chiral block b of a site's packed clover matrix */
__device__ __forceinline__ void half_load_clover_block(float (&c)[36], const unsigned char* block, size_t Vh, size_t cb, int b)
{
    const int4* q = reinterpret_cast<const int4*>(block) + cb;
    const float n = __ldg(reinterpret_cast<const float*>(block + Vh * 144) + cb);
    const float d = __fdiv_rn(n, 32767.0f);
    float t[40];
#pragma unroll
    for (int k = 0; k < 5; k++) half_unpack8(__ldg(q + (size_t)(4 * b + k) * Vh), d, &t[8 * k]);
#pragma unroll
    for (int k = 0; k < 36; k++) c[k] = t[k + 4 * b]; /* block 1 starts at code 36 = chunk 4, offset 4 */
}

#endif
