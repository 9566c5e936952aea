/*
 * layout.cu -- boundary (AoS, lexicographic) <-> internal (checkerboarded SoA) layout
 * kernels: spinor pack / unpack and the gauge load with optional precision conversion
 * and 18 -> 12 real compression.  Setup path, untimed.
 */
#include "half_device.cuh"

namespace {

/* one thread per (parity, cb) */
template <typename T, int UNPACK>
__global__ void spinor_pack_kernel(T* internal, T* boundary, DevGeom g)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 2 * g.Vh) return;
    const int parity = i / g.Vh, cb = i - parity * g.Vh;
    const Coord c = cb_to_coord(g, cb, parity);
    const size_t s = (size_t)c.x + (size_t)g.X * (c.y + (size_t)g.Y * (c.z + (size_t)g.Z * c.t));
    T* blk = internal + (size_t)parity * 24 * g.Vh;
    T v[24];
    if (UNPACK) {
        load_planes_rw<T, 24>(v, blk, (size_t)g.Vh, (size_t)cb);
#pragma unroll
        for (int k = 0; k < 24; k++) boundary[s * 24 + k] = v[k];
    } else {
#pragma unroll
        for (int k = 0; k < 24; k++) v[k] = boundary[s * 24 + k];
        store_planes<T, 24>(blk, (size_t)g.Vh, (size_t)cb, v);
    }
}

/* one thread per (mu, parity, cb) */
template <typename TI, typename T, int RECON>
__global__ void gauge_load_kernel(T* data, const TI* links, DevGeom g, size_t gblock)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 8LL * g.Vh) return;
    const int mu = (int)(i / (2LL * g.Vh));
    const int rem = (int)(i - (long long)mu * 2 * g.Vh);
    const int parity = rem / g.Vh, cb = rem - parity * g.Vh;
    const Coord c = cb_to_coord(g, cb, parity);
    const size_t s = (size_t)c.x + (size_t)g.X * (c.y + (size_t)g.Y * (c.z + (size_t)g.Z * c.t));
    T u[18];
#pragma unroll
    for (int k = 0; k < 18; k++) u[k] = (T)links[(s * 4 + mu) * 18 + k];
    store_link<T, RECON>(data + (size_t)(2 * mu + parity) * gblock, (size_t)g.Vh, (size_t)cb, u);
}

/* 16-bit links (reading H1): codes of the 12 reals of rows 0,1 at scale 32767 */
template <typename TI> __global__ void gauge_load_half_kernel(unsigned char* data, const TI* links, DevGeom g, size_t gblock)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 8LL * g.Vh) return;
    const int mu = (int)(i / (2LL * g.Vh));
    const int rem = (int)(i - (long long)mu * 2 * g.Vh);
    const int parity = rem / g.Vh, cb = rem - parity * g.Vh;
    const Coord c = cb_to_coord(g, cb, parity);
    const size_t s = (size_t)c.x + (size_t)g.X * (c.y + (size_t)g.Y * (c.z + (size_t)g.Z * c.t));
    float u[12];
#pragma unroll
    for (int k = 0; k < 12; k++) u[k] = (float)links[(s * 4 + mu) * 18 + k];
    unsigned char* blk = data + (size_t)(2 * mu + parity) * gblock;
    reinterpret_cast<int4*>(blk)[cb] = half_pack8(&u[0], 32767.0f);
    reinterpret_cast<int2*>(blk + (size_t)g.Vh * 16)[cb] = make_int2(half_pack2(u[8], u[9], 32767.0f), half_pack2(u[10], u[11], 32767.0f));
}

} // namespace

int layout_spinor_pack(qcd_ctx* ctx, void* internal, const void* boundary, const Geom& geo, int prec, int unpack)
{
    const DevGeom g = dev_geom(geo);
    const int threads = 128, blocks = (2 * g.Vh + threads - 1) / threads;
    if (prec == 4) {
        if (unpack) spinor_pack_kernel<float, 1><<<blocks, threads, 0, ctx->stream>>>((float*)internal, (float*)boundary, g);
        else spinor_pack_kernel<float, 0><<<blocks, threads, 0, ctx->stream>>>((float*)internal, (float*)boundary, g);
    } else {
        if (unpack) spinor_pack_kernel<double, 1><<<blocks, threads, 0, ctx->stream>>>((double*)internal, (double*)boundary, g);
        else spinor_pack_kernel<double, 0><<<blocks, threads, 0, ctx->stream>>>((double*)internal, (double*)boundary, g);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return qcd_set_error(QCD_ECUDA, "spinor pack: %s", cudaGetErrorString(e));
    ctx->launches++;
    return QCD_OK;
}

template <typename TI, typename T>
static void gauge_load_launch(qcd_ctx* ctx, const qcd_gauge* gh, const void* links)
{
    const DevGeom g = dev_geom(gh->geo);
    const int threads = 128;
    const long long n = 8LL * g.Vh;
    const int blocks = (int)((n + threads - 1) / threads);
    const size_t gblock = gh->block_bytes / sizeof(T);
    if (gh->reconstruct == 12)
        gauge_load_kernel<TI, T, 12><<<blocks, threads, 0, ctx->stream>>>((T*)gh->data, (const TI*)links, g, gblock);
    else
        gauge_load_kernel<TI, T, 18><<<blocks, threads, 0, ctx->stream>>>((T*)gh->data, (const TI*)links, g, gblock);
}

int layout_gauge_load(qcd_ctx* ctx, const qcd_gauge* gh, const void* links, int prec_in)
{
    if (gh->precision == 2) {
        const DevGeom g = dev_geom(gh->geo);
        const int threads = 128;
        const int blocks = (int)((8LL * g.Vh + threads - 1) / threads);
        if (prec_in == 8) gauge_load_half_kernel<double><<<blocks, threads, 0, ctx->stream>>>((unsigned char*)gh->data, (const double*)links, g, gh->block_bytes);
        else gauge_load_half_kernel<float><<<blocks, threads, 0, ctx->stream>>>((unsigned char*)gh->data, (const float*)links, g, gh->block_bytes);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return qcd_set_error(QCD_ECUDA, "gauge load (16-bit): %s", cudaGetErrorString(e));
        ctx->launches++;
        return QCD_OK;
    }
    if (prec_in == 8 && gh->precision == 8) gauge_load_launch<double, double>(ctx, gh, links);
    else if (prec_in == 8 && gh->precision == 4) gauge_load_launch<double, float>(ctx, gh, links);
    else if (prec_in == 4 && gh->precision == 4) gauge_load_launch<float, float>(ctx, gh, links);
    else gauge_load_launch<float, double>(ctx, gh, links);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return qcd_set_error(QCD_ECUDA, "gauge load: %s", cudaGetErrorString(e));
    ctx->launches++;
    return QCD_OK;
}
