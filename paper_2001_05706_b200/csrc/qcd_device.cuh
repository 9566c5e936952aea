/*
 * qcd_device.cuh -- device helpers: 128-bit field access, checkerboard indexing,
 * SU(3) link loading with 12-real reconstruction (links "suppressed to
 * 12 real numbers to save the memory bandwidth").
 */
#ifndef QCD_DEVICE_CUH
#define QCD_DEVICE_CUH

#include "qcd_internal.h"
#include <cstdlib>

/* programmatic dependent launch (sm_90+): griddepcontrol.launch_dependents lets the next launch of the stream start
 * placing blocks once every block of this grid has executed it; griddepcontrol.wait blocks until the previous grid has
 * completed and its memory operations are visible.  Both are no-ops in a launch without the attribute. */
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

/* QCD_PDL=0 in the environment launches every kernel fully serialised (A/B switch; default on) */
static inline bool pdl_enabled()
{
    static const int on = [] { const char* e = getenv("QCD_PDL"); return (e && atoi(e) == 0) ? 0 : 1; }();
    return on != 0;
}

/* Launch with programmatic stream serialisation.  Only for kernels whose first statements are pdl_launch_dependents();
 * pdl_wait(): such a kernel may be placed while its predecessor in the stream drains and reads or writes nothing
 * before the predecessor has completed.  The launch error, if any, is left for cudaGetLastError(). */
template <typename... Exp, typename... Act>
static inline void launch_pdl_smem(void (*kernel)(Exp...), int grid, int block, size_t smem, cudaStream_t st, Act&&... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3((unsigned)block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = pdl_enabled() ? 1 : 0;
    (void)cudaLaunchKernelEx(&cfg, kernel, static_cast<Exp>(args)...);
}
template <typename... Exp, typename... Act>
static inline void launch_pdl(void (*kernel)(Exp...), int grid, int block, cudaStream_t st, Act&&... args)
{
    launch_pdl_smem(kernel, grid, block, 0, st, static_cast<Act&&>(args)...);
}

template <typename T> struct Vec;
template <> struct Vec<float> {
    typedef float4 type;
    static constexpr int reals = 4;
};
template <> struct Vec<double> {
    typedef double2 type;
    static constexpr int reals = 2;
};

/* number of 128-bit chunks holding n reals */
template <typename T> __host__ __device__ constexpr int chunks_of(int nreal)
{
    return nreal / Vec<T>::reals;
}

__device__ __forceinline__ void vec_get(const float4& v, float* d)
{
    d[0] = v.x; d[1] = v.y; d[2] = v.z; d[3] = v.w;
}
__device__ __forceinline__ void vec_get(const double2& v, double* d)
{
    d[0] = v.x; d[1] = v.y;
}
__device__ __forceinline__ float4 vec_make(const float* d) { return make_float4(d[0], d[1], d[2], d[3]); }
__device__ __forceinline__ double2 vec_make(const double* d) { return make_double2(d[0], d[1]); }

/* load / store NREAL reals of site idx from a [chunk][stride] plane array */
template <typename T, int NREAL>
__device__ __forceinline__ void load_planes(T (&d)[NREAL], const T* __restrict__ base, size_t stride,
                                            size_t idx)
{
    typedef typename Vec<T>::type V;
    const V* p = reinterpret_cast<const V*>(base) + idx;
#pragma unroll
    for (int c = 0; c < NREAL / Vec<T>::reals; c++) {
        V v = __ldg(p + (size_t)c * stride);
        vec_get(v, &d[c * Vec<T>::reals]);
    }
}
/* plain (coherent) load: for buffers that the same kernel also writes elsewhere */
template <typename T, int NREAL>
__device__ __forceinline__ void load_planes_rw(T (&d)[NREAL], const T* base, size_t stride, size_t idx)
{
    typedef typename Vec<T>::type V;
    const V* p = reinterpret_cast<const V*>(base) + idx;
#pragma unroll
    for (int c = 0; c < NREAL / Vec<T>::reals; c++) {
        V v = p[(size_t)c * stride];
        vec_get(v, &d[c * Vec<T>::reals]);
    }
}
/* streaming variants (ld.global.cs / st.global.cs): data touched once per launch, marked
 * evict-first so that it does not displace the neighbour spinors that L2 must keep for reuse */
template <typename T, int NREAL>
__device__ __forceinline__ void load_planes_cs(T (&d)[NREAL], const T* base, size_t stride, size_t idx)
{
    typedef typename Vec<T>::type V;
    const V* p = reinterpret_cast<const V*>(base) + idx;
#pragma unroll
    for (int c = 0; c < NREAL / Vec<T>::reals; c++) {
        V v = __ldcs(p + (size_t)c * stride);
        vec_get(v, &d[c * Vec<T>::reals]);
    }
}
/* L2 prefetch of the NREAL reals of site idx (one line request per 128-bit plane, no register
 * is tied up): used where a thread knows, a whole vector ahead, what it will read next */
template <typename T, int NREAL>
__device__ __forceinline__ void prefetch_planes_l2(const T* base, size_t stride, size_t idx)
{
    typedef typename Vec<T>::type V;
    const V* p = reinterpret_cast<const V*>(base) + idx;
#pragma unroll
    for (int c = 0; c < NREAL / Vec<T>::reals; c++) asm volatile("prefetch.global.L2 [%0];" ::"l"(p + (size_t)c * stride));
}
template <typename T, int NREAL>
__device__ __forceinline__ void store_planes_cs(T* base, size_t stride, size_t idx, const T (&d)[NREAL])
{
    typedef typename Vec<T>::type V;
    V* p = reinterpret_cast<V*>(base) + idx;
#pragma unroll
    for (int c = 0; c < NREAL / Vec<T>::reals; c++) __stcs(p + (size_t)c * stride, vec_make(&d[c * Vec<T>::reals]));
}

template <typename T, int NREAL>
__device__ __forceinline__ void store_planes(T* base, size_t stride, size_t idx, const T (&d)[NREAL])
{
    typedef typename Vec<T>::type V;
    V* p = reinterpret_cast<V*>(base) + idx;
#pragma unroll
    for (int c = 0; c < NREAL / Vec<T>::reals; c++) p[(size_t)c * stride] = vec_make(&d[c * Vec<T>::reals]);
}

/* ---- SU(3) link: u[2*(3*row+col)+reim] ------------------------------------------ */
/* row2 = conj(row0 x row1)  (reading S7) */
template <typename T> __device__ __forceinline__ void reconstruct_row2(T (&u)[18])
{
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
        /* (r0 x r1)_c = r0[c1] r1[c2] - r0[c2] r1[c1] */
        const T ar = u[2 * c1], ai = u[2 * c1 + 1], br = u[6 + 2 * c2], bi = u[6 + 2 * c2 + 1];
        const T cr = u[2 * c2], ci = u[2 * c2 + 1], dr = u[6 + 2 * c1], di = u[6 + 2 * c1 + 1];
        /* one multiply and three fused multiply-adds per real (the bracketed form costs five) */
        T re = ar * br, nim = cr * di;
        re = re - ai * bi;
        nim = nim + ci * dr;
        re = re - cr * dr;
        nim = nim - ar * bi;
        re = re + ci * di;
        nim = nim - ai * br;
        u[12 + 2 * c] = re;
        u[12 + 2 * c + 1] = nim;
    }
}

/* block = base of one (mu, parity) gauge block; Vh sites */
template <typename T, int RECON>
__device__ __forceinline__ void load_link(T (&u)[18], const T* __restrict__ block, size_t Vh, size_t cb)
{
    if (RECON == 12) {
        T r[12];
        load_planes<T, 12>(r, block, Vh, cb);
#pragma unroll
        for (int i = 0; i < 12; i++) u[i] = r[i];
        reconstruct_row2<T>(u);
    } else if (sizeof(T) == 8) {
        load_planes<T, 18>(u, block, Vh, cb);
    } else {
        /* fp32 18-real: 4 float4 planes then one float2 plane */
        T r[16];
        load_planes<T, 16>(r, block, Vh, cb);
#pragma unroll
        for (int i = 0; i < 16; i++) u[i] = r[i];
        const float2* tail = reinterpret_cast<const float2*>(block + 16 * Vh) + cb;
        const float2 v = __ldg(tail);
        u[16] = (T)v.x;
        u[17] = (T)v.y;
    }
}

template <typename T, int RECON>
__device__ __forceinline__ void store_link(T* block, size_t Vh, size_t cb, const T (&u)[18])
{
    if (RECON == 12) {
        T r[12];
#pragma unroll
        for (int i = 0; i < 12; i++) r[i] = u[i];
        store_planes<T, 12>(block, Vh, cb, r);
    } else if (sizeof(T) == 8) {
        store_planes<T, 18>(block, Vh, cb, u);
    } else {
        T r[16];
#pragma unroll
        for (int i = 0; i < 16; i++) r[i] = u[i];
        store_planes<T, 16>(block, Vh, cb, r);
        float2* tail = reinterpret_cast<float2*>(block + 16 * Vh) + cb;
        *tail = make_float2((float)u[16], (float)u[17]);
    }
}

/* ---- solver control on the device -------------------------------------
 * Called by ONE thread once the new |r|^2 of an iteration is known (the last block of the CG
 * update kernel, or of the hop launch with the residual update fused into its epilogue): counts
 * the iteration, takes the stopping test of reading O6 or the reliable-update rule of reading O7,
 * sets ctl->halt and mirrors (iterations done, halt) to the mapped host words the solver polls. */
__device__ __forceinline__ void cg_decide(CgCtl* ctl, int* status, double rho_new)
{
    const double rn = sqrt(rho_new);
    const int it = ctl->iter + 1;
    int h = CG_RUN;
    ctl->rnorm = rn;
    ctl->iter = it;
    if (ctl->delta > 0.0) {
        double rm = ctl->rmax;
        if (rn > rm) { rm = rn; ctl->rmax = rm; }
        if (rn < ctl->delta * rm || rn <= ctl->thresh) h = CG_UPDATE_DUE;
    } else if (rn <= ctl->thresh) {
        h = CG_CONVERGED;
    }
    if (h) ctl->halt = h;
    if (status) {
        volatile int* hs = reinterpret_cast<volatile int*>(status);
        hs[1] = h;
        __threadfence_system();
        hs[0] = it;
    }
}
/* breakdown (reading O6: <p,Np> <= 0 or NaN): flagged by one thread before anything is written */
__device__ __forceinline__ void cg_flag_breakdown(CgCtl* ctl, int* status)
{
    ctl->halt = CG_BREAKDOWN;
    if (status) {
        reinterpret_cast<volatile int*>(status)[1] = CG_BREAKDOWN;
        __threadfence_system();
    }
}

/* ---- checkerboard indexing (reading S3) -------------------------------------------
 * lexicographic s = x + X (y + Y (z + Z t)); parity = (x+y+z+t)&1; cb = s >> 1. */
struct DevGeom {
    int X, Y, Z, T, X2, Vh;
};
static inline DevGeom dev_geom(const Geom& g)
{
    DevGeom d = {g.X, g.Y, g.Z, g.T, g.X2, g.Vh};
    return d;
}

struct Coord {
    int x, y, z, t;
};
__device__ __forceinline__ Coord cb_to_coord(const DevGeom& g, int cb, int parity)
{
    Coord c;
    unsigned r = (unsigned)cb;
    const unsigned xh = r % (unsigned)g.X2;
    r /= (unsigned)g.X2;
    c.y = (int)(r % (unsigned)g.Y);
    r /= (unsigned)g.Y;
    c.z = (int)(r % (unsigned)g.Z);
    c.t = (int)(r / (unsigned)g.Z);
    c.x = 2 * (int)xh + ((c.y + c.z + c.t + parity) & 1);
    return c;
}
__device__ __forceinline__ int coord_to_cb(const DevGeom& g, int x, int y, int z, int t)
{
    return (x + g.X * (y + g.Y * (z + g.Z * t))) >> 1;
}

#endif
