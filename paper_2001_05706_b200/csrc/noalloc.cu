/*
 * noalloc.cu -- qcd_norm2_noalloc: |x|^2 (reductions) for callers that cannot
 * allocate: no qcd_ctx (qcd_init calls cudaMalloc), no cudaMalloc / cudaFree / allocating library routine anywhere on
 * this path.  It is a variant of blas.cu's dot_kernel whose scratch -- one fp64 partial per block and the ticket
 * that elects the last block -- lives in a file-scope __device__ array instead of the ctx's allocation.
 *
 * The array is part of the library image: every GPU that loads libqcd_b200.so holds its NOALLOC_SCRATCH_BYTES
 * (512 KiB + 256 B) until the process exits.  Every call on a device shares it and it keeps the last call's
 * contents, so (i) what must start at zero, the ticket, is cleared on the caller's stream before each launch, the
 * partials are all written before they are read, and (ii) two calls that overlap on one GPU (different streams,
 * or graphs replayed concurrently) race on it: callers serialise them.
 *
 * In host code the array's name is a host-side stand-in, not a device address; the device address is taken once
 * per device with cudaGetSymbolAddress (qcd_noalloc_setup) and that pointer is what the kernel receives.
 */
#include "qcd_device.cuh"

namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_VEC_PER_THREAD = 4;                                  /* 128-bit words per thread                  */
constexpr size_t NA_VEC_PER_BLOCK = (size_t)NA_THREADS * NA_VEC_PER_THREAD; /* 1024 words = 16 KiB of x per block  */
constexpr size_t NA_MAX_BLOCKS = 65536;                               /* => x up to 1 GiB                          */
constexpr size_t NA_TICKET_OFFSET = NA_MAX_BLOCKS * sizeof(double);   /* ticket behind the partials, 256-aligned   */
constexpr size_t NOALLOC_SCRATCH_BYTES = NA_TICKET_OFFSET + 256;
constexpr int NA_MAX_DEVICES = 64;

static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_SCRATCH_BYTES];

/* device address of g_noalloc_scratch per device ordinal, filled in by qcd_noalloc_setup */
unsigned char* g_scratch_addr[NA_MAX_DEVICES];

__device__ __forceinline__ double na_block_sum(double v)
{
    __shared__ double sm[NA_THREADS / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) sm[w] = v;
    __syncthreads();
    double r = 0.0;
    if (w == 0) {
        r = (l < NA_THREADS / 32) ? sm[l] : 0.0;
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) r += __shfl_xor_sync(0xffffffffu, r, o);
    }
    return r; /* valid in thread 0 */
}

/* Block b sums words [b * 1024, (b + 1) * 1024) of x (products and sums in fp64), writes partial[b]; the last block
 * to take a ticket adds the partials in index order: the result depends on nvec only, not on the GPU. */
template <typename T>
__global__ void __launch_bounds__(NA_THREADS) norm2_noalloc_kernel(const T* __restrict__ x, size_t nvec, double* partial, unsigned int* ticket,
                                                                   double* out)
{
    typedef typename Vec<T>::type V;
    const V* xv = reinterpret_cast<const V*>(x);
    const size_t base = (size_t)blockIdx.x * NA_VEC_PER_BLOCK + threadIdx.x;
    V w[NA_VEC_PER_THREAD];
#pragma unroll
    for (int u = 0; u < NA_VEC_PER_THREAD; u++) {
        const size_t i = base + (size_t)u * NA_THREADS;
        if (i < nvec) w[u] = xv[i];
    }
    double s = 0.0;
#pragma unroll
    for (int u = 0; u < NA_VEC_PER_THREAD; u++) {
        const size_t i = base + (size_t)u * NA_THREADS;
        if (i < nvec) {
            T xs[Vec<T>::reals];
            vec_get(w[u], xs);
#pragma unroll
            for (int k = 0; k < Vec<T>::reals; k++) s += (double)xs[k] * (double)xs[k];
        }
    }
    __shared__ bool last;
    const double bs = na_block_sum(s);
    if (threadIdx.x == 0) {
        partial[blockIdx.x] = bs;
        __threadfence();
        last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    double t = 0.0;
    for (unsigned int i = threadIdx.x; i < gridDim.x; i += NA_THREADS) t += __ldcg(partial + i);
    const double r = na_block_sum(t);
    if (threadIdx.x == 0) *out = r;
}

} // namespace

extern "C" {

size_t qcd_noalloc_max_bytes(void) { return NA_MAX_BLOCKS * NA_VEC_PER_BLOCK * 16; }

int qcd_noalloc_setup(int device)
{
    QCD_REQUIRE(device >= 0 && device < NA_MAX_DEVICES, "noalloc_setup: device ordinal %d outside 0..%d", device, NA_MAX_DEVICES - 1);
    QCD_CHECK_CUDA(cudaSetDevice(device));
    unsigned char* p = nullptr;
    QCD_CHECK_CUDA(cudaGetSymbolAddress((void**)&p, g_noalloc_scratch));
    QCD_REQUIRE(p != nullptr && ((uintptr_t)p & 255u) == 0, "noalloc_setup: scratch symbol has no aligned device address");
    g_scratch_addr[device] = p;
    return QCD_OK;
}

int qcd_norm2_noalloc(int device, void* cuda_stream, const void* x, size_t nreal, int precision, double* result_dev)
{
    QCD_REQUIRE(device >= 0 && device < NA_MAX_DEVICES, "norm2_noalloc: device ordinal %d outside 0..%d", device, NA_MAX_DEVICES - 1);
    QCD_REQUIRE(g_scratch_addr[device] != nullptr, "norm2_noalloc: qcd_noalloc_setup(%d) has not been called", device);
    QCD_REQUIRE(precision == 4 || precision == 8, "norm2_noalloc: precision must be 4|8");
    QCD_REQUIRE(x && result_dev && ((uintptr_t)x & 15u) == 0 && ((uintptr_t)result_dev & 7u) == 0,
                "norm2_noalloc: x must be non-NULL and 16-byte aligned, result_dev a non-NULL device double");
    const size_t per = 16 / (size_t)precision;
    QCD_REQUIRE(nreal > 0 && nreal % per == 0, "norm2_noalloc: nreal must be a positive multiple of %zu", per);
    const size_t nvec = nreal / per;
    const size_t blocks = (nvec + NA_VEC_PER_BLOCK - 1) / NA_VEC_PER_BLOCK;
    QCD_REQUIRE(blocks <= NA_MAX_BLOCKS, "norm2_noalloc: %zu bytes of x exceed the %zu the static scratch covers (use qcd_norm2)",
                nreal * (size_t)precision, qcd_noalloc_max_bytes());
    QCD_CHECK_CUDA(cudaSetDevice(device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double* partial = reinterpret_cast<double*>(g_scratch_addr[device]);
    unsigned int* ticket = reinterpret_cast<unsigned int*>(g_scratch_addr[device] + NA_TICKET_OFFSET);
    QCD_CHECK_CUDA(cudaMemsetAsync(ticket, 0, sizeof(unsigned int), st)); /* the array keeps the last call's contents */
    if (precision == 4) norm2_noalloc_kernel<float><<<(unsigned)blocks, NA_THREADS, 0, st>>>((const float*)x, nvec, partial, ticket, result_dev);
    else norm2_noalloc_kernel<double><<<(unsigned)blocks, NA_THREADS, 0, st>>>((const double*)x, nvec, partial, ticket, result_dev);
    QCD_CHECK_CUDA(cudaGetLastError());
    return QCD_OK;
}

} // extern "C"
