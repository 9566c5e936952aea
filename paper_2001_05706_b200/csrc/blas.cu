/*
 * blas.cu -- fused BLAS-1 for the CG ("vector
 * operations" and reductions as their own kernels).  All streams are 128-bit loads /
 * stores; every reduction multiplies and accumulates in fp64 and is deterministic:
 * fixed grid, per-thread strided sum -> warp shuffle tree -> shared-memory tree ->
 * per-block partial -> the last block to finish (ticket) sums the partials in a fixed
 * order and writes the scalar (and derived scalars) to device memory.
 */
#include "qcd_device.cuh"

namespace {

constexpr int BLAS_THREADS = 256;
#ifndef BLAS_UNROLL
#define BLAS_UNROLL 4 /* grid-stride loops unrolled: cg_update fp32 0.88 -> 0.94, fp64 0.91 -> 0.96 of the roofline (1 / 2 / 4 swept) */
#endif
constexpr int BLAS_UNROLL_N = BLAS_UNROLL;
/* The reductions take BLAS_BATCH grid strides at a time and issue all their loads before the first use: a
 * `#pragma unroll` of a grid-stride loop keeps its early-exit test between the copies, and ptxas then leaves
 * one load in flight per thread (SASS of round 1's dot_kernel: LDG, 4 x F2F + DFMA, BRA, LDG, ...).  Measured on
 * B200 (100 MB vectors, rotating operands): norm2 fp32 22.0 -> 20.5 us, fp64 36.5 -> 34.4 us; the same change in
 * axpby / cg_update / cg_xp moved nothing (they have 3 - 6 streams in flight per iteration anyway) and was not kept.
 * What is left of a short reduction is fixed cost: 6.3 us per launch at 16 MB (`bench.py --l2-probe`). */
#ifndef BLAS_BATCH
#define BLAS_BATCH 2 /* 2 / 4 / 8 swept: norm2 the same; redot fp32 34.9 / 37.4 / 34.8 us (4 costs it two resident blocks) */
#endif
constexpr int BLAS_BATCH_N = BLAS_BATCH;

__device__ __forceinline__ double eval(const DevScalar& s)
{
    return s.num ? s.sign * (*s.num / *s.den) : s.val;
}

/* a launch of the solver iteration does nothing while the solver's halt flag is set */
__device__ __forceinline__ bool halted(const int* halt)
{
    return halt && *reinterpret_cast<const volatile int*>(halt) != 0;
}

__device__ __forceinline__ double block_sum(double v)
{
    __shared__ double sm[BLAS_THREADS / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) sm[w] = v;
    __syncthreads();
    double r = 0.0;
    if (w == 0) {
        r = (l < BLAS_THREADS / 32) ? sm[l] : 0.0;
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) r += __shfl_xor_sync(0xffffffffu, r, o);
    }
    return r; /* valid in thread 0 */
}

/* Second stage.  Returns true (in thread 0 of the last block) with the total in *tot. */
__device__ __forceinline__ bool grid_sum(double v, double* partial, unsigned int* ticket, double* tot)
{
    __shared__ bool last;
    const double bs = block_sum(v);
    if (threadIdx.x == 0) {
        partial[blockIdx.x] = bs;
        __threadfence();
        const unsigned int t = atomicInc(ticket, gridDim.x - 1); /* wraps back to 0 */
        last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!last) return false;
    __threadfence();
    /* the partials of up to GRID_SUM_BATCH * BLAS_THREADS blocks are requested together (L2 loads, the other blocks'
     * stores are visible after the fence) and summed in index order: a `volatile` loop paid one L2 round trip per
     * 256 blocks on the launch's critical path */
    constexpr int GRID_SUM_BATCH = 8;
    double pv[GRID_SUM_BATCH];
#pragma unroll
    for (int u = 0; u < GRID_SUM_BATCH; u++) {
        const unsigned int i = threadIdx.x + u * BLAS_THREADS;
        pv[u] = (i < gridDim.x) ? __ldcg(partial + i) : 0.0;
    }
    double s = 0.0;
#pragma unroll
    for (int u = 0; u < GRID_SUM_BATCH; u++) s += pv[u];
    for (unsigned int i = threadIdx.x + GRID_SUM_BATCH * BLAS_THREADS; i < gridDim.x; i += BLAS_THREADS) s += __ldcg(partial + i);
    const double r = block_sum(s);
    if (threadIdx.x == 0) *tot = r;
    return threadIdx.x == 0;
}

template <typename T> __global__ void __launch_bounds__(BLAS_THREADS) axpby_kernel(DevScalar a, const T* __restrict__ x, DevScalar b, T* __restrict__ y, size_t nvec, const int* halt)
{
    pdl_launch_dependents();
    pdl_wait();
    typedef typename Vec<T>::type V;
    if (halted(halt)) return;
    const T aa = (T)eval(a), bb = (T)eval(b);
    const V* xv = reinterpret_cast<const V*>(x);
    V* yv = reinterpret_cast<V*>(y);
#pragma unroll BLAS_UNROLL_N
    for (size_t i = (size_t)blockIdx.x * BLAS_THREADS + threadIdx.x; i < nvec; i += (size_t)gridDim.x * BLAS_THREADS) {
        T xs[Vec<T>::reals], ys[Vec<T>::reals];
        vec_get(xv[i], xs);
        vec_get(yv[i], ys);
#pragma unroll
        for (int k = 0; k < Vec<T>::reals; k++) ys[k] = aa * xs[k] + bb * ys[k];
        yv[i] = vec_make(ys);
    }
}

template <typename T, int TWO>
__global__ void __launch_bounds__(BLAS_THREADS) dot_kernel(const T* __restrict__ x, const T* __restrict__ y, size_t nvec, double* partial, unsigned int* ticket, double* out, const int* halt)
{
    pdl_launch_dependents();
    pdl_wait();
    typedef typename Vec<T>::type V;
    if (halted(halt)) return;
    const V* xv = reinterpret_cast<const V*>(x);
    const V* yv = reinterpret_cast<const V*>(y);
    double s = 0.0;
    const size_t stride = (size_t)gridDim.x * BLAS_THREADS;
    size_t i = (size_t)blockIdx.x * BLAS_THREADS + threadIdx.x;
    for (; i + (BLAS_BATCH_N - 1) * stride < nvec; i += BLAS_BATCH_N * stride) {
        V xb[BLAS_BATCH_N], yb[BLAS_BATCH_N];
#pragma unroll
        for (int u = 0; u < BLAS_BATCH_N; u++) {
            xb[u] = xv[i + u * stride];
            if (TWO) yb[u] = yv[i + u * stride];
        }
#pragma unroll
        for (int u = 0; u < BLAS_BATCH_N; u++) {
            T xs[Vec<T>::reals], ys[Vec<T>::reals];
            vec_get(xb[u], xs);
            if (TWO) vec_get(yb[u], ys);
#pragma unroll
            for (int k = 0; k < Vec<T>::reals; k++) s += (double)xs[k] * (double)(TWO ? ys[k] : xs[k]);
        }
    }
    for (; i < nvec; i += stride) {
        T xs[Vec<T>::reals], ys[Vec<T>::reals];
        vec_get(xv[i], xs);
        if (TWO) vec_get(yv[i], ys);
#pragma unroll
        for (int k = 0; k < Vec<T>::reals; k++) s += (double)xs[k] * (double)(TWO ? ys[k] : xs[k]);
    }
    double tot;
    if (grid_sum(s, partial, ticket, &tot)) *out = tot;
}

template <typename T>
__global__ void __launch_bounds__(BLAS_THREADS) cg_update_kernel(DevScalar a, const T* __restrict__ p, const T* __restrict__ q, T* __restrict__ x, T* __restrict__ r, size_t nvec, double* partial,
                                 unsigned int* ticket, double* out, CgCtl* ctl, int* status)
{
    pdl_launch_dependents();
    pdl_wait();
    typedef typename Vec<T>::type V;
    if (ctl) {
        if (halted(&ctl->halt)) return;
        /* breakdown (reading O6: <p,Np> <= 0 or NaN) is detected before anything is written */
        if (a.num && !(*a.den > 0.0)) {
            if (blockIdx.x == 0 && threadIdx.x == 0) cg_flag_breakdown(ctl, status);
            return;
        }
    }
    const T aa = (T)eval(a);
    const V* pv = reinterpret_cast<const V*>(p);
    const V* qv = reinterpret_cast<const V*>(q);
    V* xv = reinterpret_cast<V*>(x);
    V* rv = reinterpret_cast<V*>(r);
    double s = 0.0;
#pragma unroll BLAS_UNROLL_N
    for (size_t i = (size_t)blockIdx.x * BLAS_THREADS + threadIdx.x; i < nvec; i += (size_t)gridDim.x * BLAS_THREADS) {
        T ps[Vec<T>::reals], qs[Vec<T>::reals], xs[Vec<T>::reals], rs[Vec<T>::reals];
        vec_get(pv[i], ps);
        vec_get(qv[i], qs);
        vec_get(xv[i], xs);
        vec_get(rv[i], rs);
#pragma unroll
        for (int k = 0; k < Vec<T>::reals; k++) {
            xs[k] += aa * ps[k];
            rs[k] -= aa * qs[k];
            s += (double)rs[k] * (double)rs[k];
        }
        xv[i] = vec_make(xs);
        rv[i] = vec_make(rs);
    }
    double tot;
    if (grid_sum(s, partial, ticket, &tot)) {
        *out = tot;
        if (ctl) cg_decide(ctl, status, tot); /* stopping test (O6) / update rule (O7), taken on the device */
    }
}

/* The other half of a CG iteration whose residual update ran in the epilogue of the last hop launch
 * (hop_kernel.cuh, HopArgs::cg_r):  x += alpha p ; p = r + beta p.  `iter` is the iteration the host
 * enqueued this launch for.  While the solver runs (halt == 0) both updates are done.  In the iteration
 * that halted it (converged, or reliable update due: ctl->iter == iter) only x += alpha p is (readings
 * O6 / O7: the stop test and the update decision come after the x update and before the p update);
 * launches enqueued for later iterations, and everything after a breakdown, do nothing. */
template <typename T>
__global__ void __launch_bounds__(BLAS_THREADS) cg_xp_kernel(DevScalar a, DevScalar b, const T* __restrict__ r, T* __restrict__ x, T* __restrict__ p, size_t nvec, const CgCtl* ctl,
                             int iter)
{
    pdl_launch_dependents();
    pdl_wait();
    typedef typename Vec<T>::type V;
    const int h = *reinterpret_cast<const volatile int*>(&ctl->halt);
    if (h == CG_BREAKDOWN || (h != CG_RUN && ctl->iter != iter)) return;
    const bool pupd = (h == CG_RUN);
    const T aa = (T)eval(a), bb = pupd ? (T)eval(b) : (T)0;
    const V* rv = reinterpret_cast<const V*>(r);
    V* xv = reinterpret_cast<V*>(x);
    V* pv = reinterpret_cast<V*>(p);
#pragma unroll BLAS_UNROLL_N
    for (size_t i = (size_t)blockIdx.x * BLAS_THREADS + threadIdx.x; i < nvec; i += (size_t)gridDim.x * BLAS_THREADS) {
        T ps[Vec<T>::reals], xs[Vec<T>::reals];
        vec_get(pv[i], ps);
        vec_get(xv[i], xs);
#pragma unroll
        for (int k = 0; k < Vec<T>::reals; k++) xs[k] += aa * ps[k];
        xv[i] = vec_make(xs);
        if (pupd) {
            T rs[Vec<T>::reals];
            vec_get(rv[i], rs);
#pragma unroll
            for (int k = 0; k < Vec<T>::reals; k++) ps[k] = rs[k] + bb * ps[k];
            pv[i] = vec_make(ps);
        }
    }
}

/* Mixed-precision kernels.  The internal spinor layout is [chunk][cb] with 128-bit
 * chunks, so one fp32 chunk c (2 complex) of site cb corresponds to the fp64 chunks 2c
 * and 2c+1 of the same site: float4 index (blk*6 + c)*Vh + cb  <->  double2 indices
 * (blk*12 + 2c)*Vh + cb and (blk*12 + 2c + 1)*Vh + cb.  Both sides stay coalesced. */
__device__ __forceinline__ size_t hi_index(size_t i, size_t Vh)
{
    const size_t plane = i / Vh, cb = i - plane * Vh; /* plane = blk*6 + c */
    return 2 * plane * Vh + cb;
}

/* y_hi += x_lo ; x_lo = 0   (reliable update, reading O7) */
__global__ void __launch_bounds__(BLAS_THREADS) accumulate_hi_kernel(double* y, float* x, size_t n4, size_t Vh)
{
    pdl_launch_dependents();
    pdl_wait();
    float4* xv = reinterpret_cast<float4*>(x);
    double2* yv = reinterpret_cast<double2*>(y);
    for (size_t i = (size_t)blockIdx.x * BLAS_THREADS + threadIdx.x; i < n4; i += (size_t)gridDim.x * BLAS_THREADS) {
        const float4 v = xv[i];
        const size_t j = hi_index(i, Vh);
        double2 a = yv[j], b = yv[j + Vh];
        a.x += (double)v.x; a.y += (double)v.y; b.x += (double)v.z; b.y += (double)v.w;
        yv[j] = a;
        yv[j + Vh] = b;
        xv[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
}

/* r_hi = b - t ; r_lo = (float) r_hi ; out = |r_hi|^2 */
__global__ void __launch_bounds__(BLAS_THREADS) residual_hi_kernel(double* rh, float* rl, const double* b, const double* t, size_t n4, size_t Vh,
                                   double* partial, unsigned int* ticket, double* out, CgCtl* ctl)
{
    pdl_launch_dependents();
    pdl_wait();
    double s = 0.0;
    const double2* bv = reinterpret_cast<const double2*>(b);
    const double2* tv = reinterpret_cast<const double2*>(t);
    double2* rv = reinterpret_cast<double2*>(rh);
    float4* lv = reinterpret_cast<float4*>(rl);
    for (size_t i = (size_t)blockIdx.x * BLAS_THREADS + threadIdx.x; i < n4; i += (size_t)gridDim.x * BLAS_THREADS) {
        const size_t j = hi_index(i, Vh);
        const double2 b0 = bv[j], b1 = bv[j + Vh], t0 = tv[j], t1 = tv[j + Vh];
        const double2 r0 = make_double2(b0.x - t0.x, b0.y - t0.y), r1 = make_double2(b1.x - t1.x, b1.y - t1.y);
        s += r0.x * r0.x + r0.y * r0.y + r1.x * r1.x + r1.y * r1.y;
        rv[j] = r0;
        rv[j + Vh] = r1;
        lv[i] = make_float4((float)r0.x, (float)r0.y, (float)r1.x, (float)r1.y);
    }
    double tot;
    if (grid_sum(s, partial, ticket, &tot)) {
        *out = tot;
        if (ctl) { /* reading O7: rmax = |r_hi|; stop iff |r_hi| <= tol |b| */
            const double rn = sqrt(tot);
            ctl->rmax = rn;
            ctl->rnorm = rn;
            ctl->halt = (rn <= ctl->thresh) ? CG_CONVERGED : CG_RUN;
        }
    }
}

/* HI_TO_LO: lo = (float) hi ; else hi = (double) lo */
template <int HI_TO_LO> __global__ void __launch_bounds__(BLAS_THREADS) convert_kernel(double* hi, float* lo, size_t n4, size_t Vh)
{
    pdl_launch_dependents();
    pdl_wait();
    float4* lv = reinterpret_cast<float4*>(lo);
    double2* hv = reinterpret_cast<double2*>(hi);
    for (size_t i = (size_t)blockIdx.x * BLAS_THREADS + threadIdx.x; i < n4; i += (size_t)gridDim.x * BLAS_THREADS) {
        const size_t j = hi_index(i, Vh);
        if (HI_TO_LO) {
            const double2 a = hv[j], b = hv[j + Vh];
            lv[i] = make_float4((float)a.x, (float)a.y, (float)b.x, (float)b.y);
        } else {
            const float4 v = lv[i];
            hv[j] = make_double2((double)v.x, (double)v.y);
            hv[j + Vh] = make_double2((double)v.z, (double)v.w);
        }
    }
}

/* ---- multi-shift CG updates: one pass over all shifted systems ------- */
template <typename T>
__global__ void __launch_bounds__(BLAS_THREADS) multishift_x_kernel(MultiShiftCoef cf, T* x, const T* p, size_t fstride_vec, const T* q, T* r,
                                    size_t nvec, double* partial, unsigned int* ticket, double* out)
{
    pdl_launch_dependents();
    pdl_wait();
    typedef typename Vec<T>::type V;
    const V* qv = reinterpret_cast<const V*>(q);
    V* rv = reinterpret_cast<V*>(r);
    const T alpha = (T)cf.alpha;
    double s = 0.0;
#pragma unroll BLAS_UNROLL_N
    for (size_t i = (size_t)blockIdx.x * BLAS_THREADS + threadIdx.x; i < nvec; i += (size_t)gridDim.x * BLAS_THREADS) {
        T qs[Vec<T>::reals], rs[Vec<T>::reals];
        vec_get(qv[i], qs);
        vec_get(rv[i], rs);
#pragma unroll
        for (int k = 0; k < Vec<T>::reals; k++) {
            rs[k] -= alpha * qs[k];
            s += (double)rs[k] * (double)rs[k];
        }
        rv[i] = vec_make(rs);
        for (int j = 0; j < cf.ns; j++) {
            V* xv = reinterpret_cast<V*>(x) + (size_t)j * fstride_vec;
            const V* pv = reinterpret_cast<const V*>(p) + (size_t)j * fstride_vec;
            T xs[Vec<T>::reals], ps[Vec<T>::reals];
            vec_get(xv[i], xs);
            vec_get(pv[i], ps);
            const T a = (T)cf.c[j];
#pragma unroll
            for (int k = 0; k < Vec<T>::reals; k++) xs[k] += a * ps[k];
            xv[i] = vec_make(xs);
        }
    }
    double tot;
    if (grid_sum(s, partial, ticket, &tot)) *out = tot;
}

template <typename T>
__global__ void __launch_bounds__(BLAS_THREADS) multishift_p_kernel(MultiShiftCoef zeta, MultiShiftCoef beta, T* p, size_t fstride_vec, const T* r, size_t nvec)
{
    pdl_launch_dependents();
    pdl_wait();
    typedef typename Vec<T>::type V;
    const V* rv = reinterpret_cast<const V*>(r);
#pragma unroll BLAS_UNROLL_N
    for (size_t i = (size_t)blockIdx.x * BLAS_THREADS + threadIdx.x; i < nvec; i += (size_t)gridDim.x * BLAS_THREADS) {
        T rs[Vec<T>::reals];
        vec_get(rv[i], rs);
        for (int j = 0; j < zeta.ns; j++) {
            V* pv = reinterpret_cast<V*>(p) + (size_t)j * fstride_vec;
            T ps[Vec<T>::reals];
            vec_get(pv[i], ps);
            const T z = (T)zeta.c[j], b = (T)beta.c[j];
#pragma unroll
            for (int k = 0; k < Vec<T>::reals; k++) ps[k] = z * rs[k] + b * ps[k];
            pv[i] = vec_make(ps);
        }
    }
}

/* x_j += cx_j p_j (j < cx.ns) and p_j = zeta_j r + beta_j p_j (j < zeta.ns <= cx.ns) in one pass: the multi-shift
 * iteration whose residual update ran in the operator's epilogue (solver.cu) */
template <typename T>
__global__ void __launch_bounds__(BLAS_THREADS) multishift_xp_kernel(MultiShiftCoef cx, MultiShiftCoef zeta, MultiShiftCoef beta, T* x, T* p, size_t fstride_vec,
                                                                     const T* r, size_t nvec)
{
    pdl_launch_dependents();
    pdl_wait();
    typedef typename Vec<T>::type V;
    const V* rv = reinterpret_cast<const V*>(r);
#pragma unroll 2
    for (size_t i = (size_t)blockIdx.x * BLAS_THREADS + threadIdx.x; i < nvec; i += (size_t)gridDim.x * BLAS_THREADS) {
        T rs[Vec<T>::reals];
        if (zeta.ns > 0) vec_get(rv[i], rs);
        for (int j = 0; j < cx.ns; j++) {
            V* xv = reinterpret_cast<V*>(x) + (size_t)j * fstride_vec;
            V* pv = reinterpret_cast<V*>(p) + (size_t)j * fstride_vec;
            T xs[Vec<T>::reals], ps[Vec<T>::reals];
            vec_get(xv[i], xs);
            vec_get(pv[i], ps);
            const T a = (T)cx.c[j];
#pragma unroll
            for (int k = 0; k < Vec<T>::reals; k++) xs[k] += a * ps[k];
            xv[i] = vec_make(xs);
            if (j < zeta.ns) {
                const T z = (T)zeta.c[j], b = (T)beta.c[j];
#pragma unroll
                for (int k = 0; k < Vec<T>::reals; k++) ps[k] = z * rs[k] + b * ps[k];
                pv[i] = vec_make(ps);
            }
        }
    }
}

int grid_for(const qcd_ctx* ctx, size_t nvec)
{
    size_t b = (nvec + BLAS_THREADS - 1) / BLAS_THREADS;
    const size_t cap = (size_t)ctx->max_blocks;
    if (b > cap) b = cap;
    if (b < 1) b = 1;
    return (int)b;
}

int check_launch(qcd_ctx* ctx, const char* what)
{
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return qcd_set_error(QCD_ECUDA, "%s: %s", what, cudaGetErrorString(e));
    ctx->launches++;
    return QCD_OK;
}

} // namespace

int blas_axpby(qcd_ctx* ctx, DevScalar a, const void* x, DevScalar b, void* y, size_t nreal, int prec, const int* halt)
{
    if (prec == 4) {
        const size_t nv = nreal / 4;
        launch_pdl(axpby_kernel<float>, grid_for(ctx, nv), BLAS_THREADS, ctx->stream, a, (const float*)x, b, (float*)y, nv, halt);
    } else {
        const size_t nv = nreal / 2;
        launch_pdl(axpby_kernel<double>, grid_for(ctx, nv), BLAS_THREADS, ctx->stream, a, (const double*)x, b, (double*)y, nv, halt);
    }
    return check_launch(ctx, "axpby");
}

int blas_norm2(qcd_ctx* ctx, const void* x, size_t nreal, int prec, double* d_out)
{
    if (prec == 4) {
        const size_t nv = nreal / 4;
        launch_pdl(dot_kernel<float, 0>, grid_for(ctx, nv), BLAS_THREADS, ctx->stream, (const float*)x, (const float*)x, nv, ctx->d_partial, ctx->d_ticket, d_out, nullptr);
    } else {
        const size_t nv = nreal / 2;
        launch_pdl(dot_kernel<double, 0>, grid_for(ctx, nv), BLAS_THREADS, ctx->stream, (const double*)x, (const double*)x, nv, ctx->d_partial, ctx->d_ticket, d_out, nullptr);
    }
    return check_launch(ctx, "norm2");
}

int blas_redot(qcd_ctx* ctx, const void* x, const void* y, size_t nreal, int prec, double* d_out, const int* halt)
{
    if (prec == 4) {
        const size_t nv = nreal / 4;
        launch_pdl(dot_kernel<float, 1>, grid_for(ctx, nv), BLAS_THREADS, ctx->stream, (const float*)x, (const float*)y, nv, ctx->d_partial, ctx->d_ticket, d_out, halt);
    } else {
        const size_t nv = nreal / 2;
        launch_pdl(dot_kernel<double, 1>, grid_for(ctx, nv), BLAS_THREADS, ctx->stream, (const double*)x, (const double*)y, nv, ctx->d_partial, ctx->d_ticket, d_out, halt);
    }
    return check_launch(ctx, "redot");
}

int blas_cg_update(qcd_ctx* ctx, DevScalar a, const void* p, const void* q, void* x, void* r, size_t nreal, int prec,
                   double* d_out, CgCtl* ctl, int* status)
{
    if (prec == 4) {
        const size_t nv = nreal / 4;
        launch_pdl(cg_update_kernel<float>, grid_for(ctx, nv), BLAS_THREADS, ctx->stream, a, (const float*)p, (const float*)q, (float*)x, (float*)r, nv,
                                                                                   ctx->d_partial, ctx->d_ticket, d_out, ctl, status);
    } else {
        const size_t nv = nreal / 2;
        launch_pdl(cg_update_kernel<double>, grid_for(ctx, nv), BLAS_THREADS, ctx->stream, a, (const double*)p, (const double*)q, (double*)x, (double*)r, nv,
                                                                                    ctx->d_partial, ctx->d_ticket, d_out, ctl, status);
    }
    return check_launch(ctx, "cg_update");
}

int blas_cg_xp(qcd_ctx* ctx, DevScalar a, DevScalar b, const void* r, void* x, void* p, size_t nreal, int prec, const CgCtl* ctl, int iter)
{
    if (prec == 4) {
        const size_t nv = nreal / 4;
        launch_pdl(cg_xp_kernel<float>, grid_for(ctx, nv), BLAS_THREADS, ctx->stream, a, b, (const float*)r, (float*)x, (float*)p, nv, ctl, iter);
    } else {
        const size_t nv = nreal / 2;
        launch_pdl(cg_xp_kernel<double>, grid_for(ctx, nv), BLAS_THREADS, ctx->stream, a, b, (const double*)r, (double*)x, (double*)p, nv, ctl, iter);
    }
    return check_launch(ctx, "cg_xp");
}

int blas_accumulate_hi(qcd_ctx* ctx, void* y_hi, void* x_lo, size_t nreal, size_t Vh)
{
    const size_t n4 = nreal / 4;
    launch_pdl(accumulate_hi_kernel, grid_for(ctx, n4), BLAS_THREADS, ctx->stream, (double*)y_hi, (float*)x_lo, n4, Vh);
    return check_launch(ctx, "accumulate_hi");
}

int blas_residual_hi(qcd_ctx* ctx, void* r_hi, void* r_lo, const void* b, const void* t, size_t nreal, size_t Vh, double* d_out, CgCtl* ctl)
{
    const size_t n4 = nreal / 4;
    launch_pdl(residual_hi_kernel, grid_for(ctx, n4), BLAS_THREADS, ctx->stream, (double*)r_hi, (float*)r_lo, (const double*)b, (const double*)t, n4, Vh,
                                                                          ctx->d_partial, ctx->d_ticket, d_out, ctl);
    return check_launch(ctx, "residual_hi");
}

int blas_convert(qcd_ctx* ctx, void* dst, int pdst, const void* src, int psrc, size_t nreal, size_t Vh)
{
    if (pdst == psrc) return blas_copy(ctx, dst, src, nreal * (size_t)pdst);
    const size_t n4 = nreal / 4;
    const int g = grid_for(ctx, n4);
    if (pdst == 4)
        launch_pdl(convert_kernel<1>, g, BLAS_THREADS, ctx->stream, (double*)const_cast<void*>(src), (float*)dst, n4, Vh);
    else
        launch_pdl(convert_kernel<0>, g, BLAS_THREADS, ctx->stream, (double*)dst, (float*)const_cast<void*>(src), n4, Vh);
    return check_launch(ctx, "convert");
}

int blas_zero(qcd_ctx* ctx, void* x, size_t bytes)
{
    cudaError_t e = cudaMemsetAsync(x, 0, bytes, ctx->stream);
    if (e != cudaSuccess) return qcd_set_error(QCD_ECUDA, "memset: %s", cudaGetErrorString(e));
    return QCD_OK;
}

int blas_copy(qcd_ctx* ctx, void* dst, const void* src, size_t bytes)
{
    cudaError_t e = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToDevice, ctx->stream);
    if (e != cudaSuccess) return qcd_set_error(QCD_ECUDA, "memcpy: %s", cudaGetErrorString(e));
    return QCD_OK;
}

int blas_multishift_xp(qcd_ctx* ctx, const MultiShiftCoef& cx, const MultiShiftCoef& zeta, const MultiShiftCoef& beta, void* x, void* p, const void* r,
                       size_t nreal, int prec)
{
    if (prec == 4) {
        const size_t nv = nreal / 4;
        launch_pdl(multishift_xp_kernel<float>, grid_for(ctx, nv), BLAS_THREADS, ctx->stream, cx, zeta, beta, (float*)x, (float*)p, nv, (const float*)r, nv);
    } else {
        const size_t nv = nreal / 2;
        launch_pdl(multishift_xp_kernel<double>, grid_for(ctx, nv), BLAS_THREADS, ctx->stream, cx, zeta, beta, (double*)x, (double*)p, nv, (const double*)r, nv);
    }
    return check_launch(ctx, "multishift_xp");
}

int blas_multishift_x(qcd_ctx* ctx, const MultiShiftCoef& cf, void* x, const void* p, const void* q, void* r, size_t nreal, int prec,
                      double* d_out)
{
    if (prec == 4) {
        const size_t nv = nreal / 4;
        launch_pdl(multishift_x_kernel<float>, grid_for(ctx, nv), BLAS_THREADS, ctx->stream, cf, (float*)x, (const float*)p, nv, (const float*)q, (float*)r, nv,
                                                                                      ctx->d_partial, ctx->d_ticket, d_out);
    } else {
        const size_t nv = nreal / 2;
        launch_pdl(multishift_x_kernel<double>, grid_for(ctx, nv), BLAS_THREADS, ctx->stream, cf, (double*)x, (const double*)p, nv, (const double*)q, (double*)r,
                                                                                       nv, ctx->d_partial, ctx->d_ticket, d_out);
    }
    return check_launch(ctx, "multishift_x");
}

int blas_multishift_p(qcd_ctx* ctx, const MultiShiftCoef& zeta, const MultiShiftCoef& beta, void* p, const void* r, size_t nreal, int prec)
{
    if (prec == 4) {
        const size_t nv = nreal / 4;
        launch_pdl(multishift_p_kernel<float>, grid_for(ctx, nv), BLAS_THREADS, ctx->stream, zeta, beta, (float*)p, nv, (const float*)r, nv);
    } else {
        const size_t nv = nreal / 2;
        launch_pdl(multishift_p_kernel<double>, grid_for(ctx, nv), BLAS_THREADS, ctx->stream, zeta, beta, (double*)p, nv, (const double*)r, nv);
    }
    return check_launch(ctx, "multishift_p");
}
