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

template <int DAG, int MODE, int OUT_F32>
__global__ void __launch_bounds__(128, 4) hop_half_kernel(const HalfHopArgs A)
{
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= A.geo.Vh) return;
    const size_t Vh = (size_t)A.geo.Vh;
    const Neighbours<float> nb(A.geo, cb, A.parity, A.tb);
    const HalfLinks L = {A.gauge, A.gblock, Vh, A.parity};
    const HalfSpinor src = {A.in, Vh};
    float acc[24];
    hop_site<float, DAG>(acc, L, src, cb, nb);

    if (MODE == HOP_XPAY || MODE == HOP_CLOVER_Z) {
        const HalfSpinor zs = {A.z, Vh};
        float zz[24];
        zs.load(zz, cb);
        if (MODE == HOP_CLOVER_Z) {
            float az[24];
            half_clover_apply(az, A.clover, Vh, (size_t)cb, zz);
#pragma unroll
            for (int i = 0; i < 24; i++) acc[i] = A.a * az[i] + A.b * acc[i];
        } else {
#pragma unroll
            for (int i = 0; i < 24; i++) acc[i] = A.a * zz[i] + A.b * acc[i];
        }
    } else if (MODE == HOP_CLOVER_OUT) {
        float o[24];
        half_clover_apply(o, A.clover, Vh, (size_t)cb, acc);
#pragma unroll
        for (int i = 0; i < 24; i++) acc[i] = o[i];
    }
    if (OUT_F32)
        store_planes<float, 24>(reinterpret_cast<float*>(A.out), Vh, (size_t)cb, acc);
    else
        half_store_spinor(A.out, Vh, (size_t)cb, acc);
}

template <int DAG, int MODE> cudaError_t launch_mode(const HalfHopArgs& A, int out_f32, cudaStream_t st)
{
    const int threads = 128, blocks = (A.geo.Vh + threads - 1) / threads;
    if (out_f32) hop_half_kernel<DAG, MODE, 1><<<blocks, threads, 0, st>>>(A);
    else hop_half_kernel<DAG, MODE, 0><<<blocks, threads, 0, st>>>(A);
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
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= Vh * (size_t)nblocks) return;
    const size_t blk = i / Vh, cb = i - blk * Vh;
    float v[24];
    if (TO_HALF) {
        load_planes_rw<float, 24>(v, f32 + blk * 24 * Vh, Vh, cb);
        half_store_spinor(half + blk * HALF_SPINOR_BYTES * Vh, Vh, cb, v);
    } else {
        const HalfSpinor s = {half + blk * HALF_SPINOR_BYTES * Vh, Vh};
        s.load(v, (int)cb);
        store_planes<float, 24>(f32 + blk * 24 * Vh, Vh, cb, v);
    }
}

/* p = a r + b p (fp32, b == 0: p not read) ; ph = store16(p) */
__global__ void xpay_q16_kernel(float a, const float* r, float b, float* p, unsigned char* ph, size_t Vh, int nblocks)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= Vh * (size_t)nblocks) return;
    const size_t blk = i / Vh, cb = i - blk * Vh;
    float rv[24], pv[24];
    load_planes_rw<float, 24>(rv, r + blk * 24 * Vh, Vh, cb);
    if (b != 0.f) {
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
    cudaError_t e = L.dagger ? launch_dag<1>(A, L.mode, out_f32, ctx->stream) : launch_dag<0>(A, L.mode, out_f32, ctx->stream);
    if (e != cudaSuccess) return qcd_set_error(QCD_ECUDA, "half hop launch: %s", cudaGetErrorString(e));
    ctx->launches++;
    return QCD_OK;
}

int half_convert(qcd_ctx* ctx, void* half, void* f32, size_t Vh, int nblocks, int to_half)
{
    const size_t n = Vh * (size_t)nblocks;
    const int threads = 128, blocks = (int)((n + threads - 1) / threads);
    if (to_half) half_convert_kernel<1><<<blocks, threads, 0, ctx->stream>>>((unsigned char*)half, (float*)f32, Vh, nblocks);
    else half_convert_kernel<0><<<blocks, threads, 0, ctx->stream>>>((unsigned char*)half, (float*)f32, Vh, nblocks);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return qcd_set_error(QCD_ECUDA, "half convert: %s", cudaGetErrorString(e));
    ctx->launches++;
    return QCD_OK;
}

int half_xpay_store(qcd_ctx* ctx, double a, const void* r, double b, void* p, void* ph, size_t Vh, int nblocks)
{
    const size_t n = Vh * (size_t)nblocks;
    const int threads = 128, blocks = (int)((n + threads - 1) / threads);
    xpay_q16_kernel<<<blocks, threads, 0, ctx->stream>>>((float)a, (const float*)r, (float)b, (float*)p, (unsigned char*)ph, Vh, nblocks);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return qcd_set_error(QCD_ECUDA, "half xpay: %s", cudaGetErrorString(e));
    ctx->launches++;
    return QCD_OK;
}
