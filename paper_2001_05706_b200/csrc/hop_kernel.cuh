/*
 * hop_kernel.cuh -- the single-parity Wilson hopping term (
 * BASELINE.json north_star formula; "the D-slash", single precision with
 * 12-real links)
 *
 *   (H psi)(x) = sum_mu [ (1 - g_mu) U_mu(x) psi(x+mu) + (1 + g_mu) U_mu(x-mu)^dag psi(x-mu) ]
 *
 * on the sites x of one parity, reading psi on the other parity, with a fused site-local
 * epilogue (xpay, clover apply, clover-inverse apply, Chebyshev step).
 *
 * One thread per output site.  Per direction the thread issues 128-bit loads of the
 * neighbour spinor and of the link (coalesced along cb), projects to a half spinor
 * (DeGrand-Rossi basis, table in DESIGN.md), multiplies the two colour vectors by U or
 * U^dag and accumulates with the spin reconstruction.
 */
#ifndef QCD_HOP_KERNEL_CUH
#define QCD_HOP_KERNEL_CUH

#include "qcd_device.cuh"

template <typename T> struct HopArgs {
    T* out;
    const T* in;
    const T* z;
    T* y;
    T* tm;
    const T* gauge;
    const T* clover;
    size_t gblock; /* reals per (mu, parity) gauge block */
    DevGeom geo;
    int parity;
    T tb;
    T a, b, c0, c1, c2, ck;
    int y_init;
};

/* spin projection: h = rows 0,1 of (1 + S g_mu) psi.  s[2*(3*spin+col)+reim]; h[2*(3*j+col)+reim] */
template <typename T, int MU, int S> __device__ __forceinline__ void project(T (&h)[12], const T (&s)[24])
{
    const T sg = (T)S;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const int r0 = 2 * c, r1 = 2 * (3 + c), r2 = 2 * (6 + c), r3 = 2 * (9 + c);
        if (MU == 0) { /* h0 = p0 + S i p3 ; h1 = p1 + S i p2 */
            h[r0] = s[r0] - sg * s[r3 + 1];
            h[r0 + 1] = s[r0 + 1] + sg * s[r3];
            h[r1] = s[r1] - sg * s[r2 + 1];
            h[r1 + 1] = s[r1 + 1] + sg * s[r2];
        } else if (MU == 1) { /* h0 = p0 - S p3 ; h1 = p1 + S p2 */
            h[r0] = s[r0] - sg * s[r3];
            h[r0 + 1] = s[r0 + 1] - sg * s[r3 + 1];
            h[r1] = s[r1] + sg * s[r2];
            h[r1 + 1] = s[r1 + 1] + sg * s[r2 + 1];
        } else if (MU == 2) { /* h0 = p0 + S i p2 ; h1 = p1 - S i p3 */
            h[r0] = s[r0] - sg * s[r2 + 1];
            h[r0 + 1] = s[r0 + 1] + sg * s[r2];
            h[r1] = s[r1] + sg * s[r3 + 1];
            h[r1 + 1] = s[r1 + 1] - sg * s[r3];
        } else { /* h0 = p0 + S p2 ; h1 = p1 + S p3 */
            h[r0] = s[r0] + sg * s[r2];
            h[r0 + 1] = s[r0 + 1] + sg * s[r2 + 1];
            h[r1] = s[r1] + sg * s[r3];
            h[r1 + 1] = s[r1 + 1] + sg * s[r3 + 1];
        }
    }
}

/* acc += (rows 0..3 of (1 + S g_mu) chi) given its upper half w = (w0, w1) */
template <typename T, int MU, int S> __device__ __forceinline__ void reconstruct_add(T (&acc)[24], const T (&w)[12])
{
    const T sg = (T)S;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const int j0 = 2 * c, j1 = 2 * (3 + c);
        const int r2 = 2 * (6 + c), r3 = 2 * (9 + c);
        acc[j0] += w[j0];
        acc[j0 + 1] += w[j0 + 1];
        acc[j1] += w[j1];
        acc[j1 + 1] += w[j1 + 1];
        if (MU == 0) { /* out2 = -S i w1 ; out3 = -S i w0 */
            acc[r2] += sg * w[j1 + 1];
            acc[r2 + 1] -= sg * w[j1];
            acc[r3] += sg * w[j0 + 1];
            acc[r3 + 1] -= sg * w[j0];
        } else if (MU == 1) { /* out2 = S w1 ; out3 = -S w0 */
            acc[r2] += sg * w[j1];
            acc[r2 + 1] += sg * w[j1 + 1];
            acc[r3] -= sg * w[j0];
            acc[r3 + 1] -= sg * w[j0 + 1];
        } else if (MU == 2) { /* out2 = -S i w0 ; out3 = +S i w1 */
            acc[r2] += sg * w[j0 + 1];
            acc[r2 + 1] -= sg * w[j0];
            acc[r3] -= sg * w[j1 + 1];
            acc[r3 + 1] += sg * w[j1];
        } else { /* out2 = S w0 ; out3 = S w1 */
            acc[r2] += sg * w[j0];
            acc[r2 + 1] += sg * w[j0 + 1];
            acc[r3] += sg * w[j1];
            acc[r3 + 1] += sg * w[j1 + 1];
        }
    }
}

/* w_j = U h_j (ADJ = 0) or U^dag h_j (ADJ = 1), j = 0,1, scaled by sign */
template <typename T, int ADJ>
__device__ __forceinline__ void colour_mul(T (&w)[12], const T (&u)[18], const T (&h)[12], T sign)
{
#pragma unroll
    for (int j = 0; j < 2; j++)
#pragma unroll
        for (int a = 0; a < 3; a++) {
            T re = 0, im = 0;
#pragma unroll
            for (int b = 0; b < 3; b++) {
                const int k = ADJ ? 2 * (3 * b + a) : 2 * (3 * a + b);
                const T ur = u[k], ui = ADJ ? -u[k + 1] : u[k + 1];
                const T hr = h[2 * (3 * j + b)], hi = h[2 * (3 * j + b) + 1];
                re += ur * hr - ui * hi;
                im += ur * hi + ui * hr;
            }
            w[2 * (3 * j + a)] = sign * re;
            w[2 * (3 * j + a) + 1] = sign * im;
        }
}

/* one direction: MU, DIR = +1 forward / -1 backward; SG = projector sign (forward: -1, i.e. 1 - g) */
template <typename T, int RECON, int MU, int DIR, int SG>
__device__ __forceinline__ void hop_dir(T (&acc)[24], const HopArgs<T>& A, int cb, int nb_cb, T sign)
{
    const size_t Vh = (size_t)A.geo.Vh;
    T s[24], u[18], h[12], w[12];
    load_planes<T, 24>(s, A.in, Vh, (size_t)nb_cb);
    if (DIR > 0)
        load_link<T, RECON>(u, A.gauge + (size_t)(2 * MU + A.parity) * A.gblock, Vh, (size_t)cb);
    else
        load_link<T, RECON>(u, A.gauge + (size_t)(2 * MU + (1 - A.parity)) * A.gblock, Vh, (size_t)nb_cb);
    project<T, MU, SG>(h, s);
    colour_mul<T, (DIR < 0)>(w, u, h, sign);
    reconstruct_add<T, MU, SG>(acc, w);
}

/* packed Hermitian 6x6 block times 6-vector; c = 36 reals of one block */
template <typename T> __device__ __forceinline__ void clover_block_apply(T* o, const T* c, const T* v)
{
#pragma unroll
    for (int i = 0; i < 6; i++) {
        T re = c[i] * v[2 * i], im = c[i] * v[2 * i + 1];
#pragma unroll
        for (int j = 0; j < 6; j++) {
            if (j == i) continue;
            const int hi = i > j ? i : j, lo = i > j ? j : i;
            const int k = 6 + 2 * (5 * lo - (lo * (lo - 1)) / 2 + (hi - lo - 1));
            const T lr = c[k], li = (i > j) ? c[k + 1] : -c[k + 1];
            re += lr * v[2 * j] - li * v[2 * j + 1];
            im += lr * v[2 * j + 1] + li * v[2 * j];
        }
        o[2 * i] = re;
        o[2 * i + 1] = im;
    }
}

template <typename T>
__device__ __forceinline__ void clover_apply(T (&o)[24], const T* __restrict__ clov, size_t Vh, size_t cb,
                                             const T (&v)[24])
{
#pragma unroll
    for (int b = 0; b < 2; b++) {
        T c[36];
        load_planes<T, 36>(c, clov + (size_t)36 * b * Vh, Vh, cb);
        clover_block_apply<T>(&o[12 * b], c, &v[12 * b]);
    }
}

template <typename T, int RECON, int DAG, int MODE>
__global__ void __launch_bounds__(128, (sizeof(T) == 4 ? 4 : 2)) hop_kernel(const HopArgs<T> A)
{
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= A.geo.Vh) return;
    const DevGeom& g = A.geo;
    const Coord c = cb_to_coord(g, cb, A.parity);
    const size_t Vh = (size_t)g.Vh;

    /* neighbour checkerboard indices (periodic wrap; reading S3) */
    const int odd = c.x & 1;
    const int xp = odd ? (c.x == g.X - 1 ? cb - (g.X2 - 1) : cb + 1) : cb;
    const int xm = odd ? cb : (c.x == 0 ? cb + (g.X2 - 1) : cb - 1);
    const int sy = g.X2, sz = g.X2 * g.Y, st = g.X2 * g.Y * g.Z;
    const int yp = (c.y == g.Y - 1) ? cb - (g.Y - 1) * sy : cb + sy;
    const int ym = (c.y == 0) ? cb + (g.Y - 1) * sy : cb - sy;
    const int zp = (c.z == g.Z - 1) ? cb - (g.Z - 1) * sz : cb + sz;
    const int zm = (c.z == 0) ? cb + (g.Z - 1) * sz : cb - sz;
    const int tp = (c.t == g.T - 1) ? cb - (g.T - 1) * st : cb + st;
    const int tmn = (c.t == 0) ? cb + (g.T - 1) * st : cb - st;
    const T sgn_tp = (c.t == g.T - 1) ? A.tb : (T)1;
    const T sgn_tm = (c.t == 0) ? A.tb : (T)1;

    /* forward hop carries (1 - g_mu), backward (1 + g_mu); the adjoint swaps them (O4) */
    constexpr int SF = DAG ? +1 : -1;
    constexpr int SB = DAG ? -1 : +1;

    T acc[24];
#pragma unroll
    for (int i = 0; i < 24; i++) acc[i] = 0;

    hop_dir<T, RECON, 0, +1, SF>(acc, A, cb, xp, (T)1);
    hop_dir<T, RECON, 0, -1, SB>(acc, A, cb, xm, (T)1);
    hop_dir<T, RECON, 1, +1, SF>(acc, A, cb, yp, (T)1);
    hop_dir<T, RECON, 1, -1, SB>(acc, A, cb, ym, (T)1);
    hop_dir<T, RECON, 2, +1, SF>(acc, A, cb, zp, (T)1);
    hop_dir<T, RECON, 2, -1, SB>(acc, A, cb, zm, (T)1);
    hop_dir<T, RECON, 3, +1, SF>(acc, A, cb, tp, sgn_tp);
    hop_dir<T, RECON, 3, -1, SB>(acc, A, cb, tmn, sgn_tm);

    if (MODE == HOP_PLAIN) {
        store_planes<T, 24>(A.out, Vh, (size_t)cb, acc);
    } else if (MODE == HOP_XPAY) {
        T zz[24];
        load_planes_rw<T, 24>(zz, A.z, Vh, (size_t)cb);
#pragma unroll
        for (int i = 0; i < 24; i++) acc[i] = A.a * zz[i] + A.b * acc[i];
        store_planes<T, 24>(A.out, Vh, (size_t)cb, acc);
    } else if (MODE == HOP_CLOVER_Z) {
        T zz[24], az[24];
        load_planes_rw<T, 24>(zz, A.z, Vh, (size_t)cb);
        clover_apply<T>(az, A.clover, Vh, (size_t)cb, zz);
#pragma unroll
        for (int i = 0; i < 24; i++) acc[i] = A.a * az[i] + A.b * acc[i];
        store_planes<T, 24>(A.out, Vh, (size_t)cb, acc);
    } else if (MODE == HOP_CLOVER_OUT) {
        T o[24];
        clover_apply<T>(o, A.clover, Vh, (size_t)cb, acc);
        store_planes<T, 24>(A.out, Vh, (size_t)cb, o);
    } else { /* HOP_CHEB: tn = c1 g5 (z + b H in) + c2 tm ; y (+)= ck tn ; tm <- tn  (reading O8) */
        T zz[24], yy[24];
        load_planes_rw<T, 24>(zz, A.z, Vh, (size_t)cb);
#pragma unroll
        for (int i = 0; i < 24; i++) {
            const T g5 = (i < 12) ? (T)1 : (T)-1; /* gamma5 = diag(1,1,-1,-1) */
            acc[i] = A.c1 * g5 * (zz[i] + A.b * acc[i]);
        }
        if (A.c2 != (T)0) {
            T tt[24];
            load_planes_rw<T, 24>(tt, A.tm, Vh, (size_t)cb);
#pragma unroll
            for (int i = 0; i < 24; i++) acc[i] += A.c2 * tt[i];
        }
        if (A.y_init) {
#pragma unroll
            for (int i = 0; i < 24; i++) yy[i] = A.c0 * zz[i] + A.ck * acc[i];
        } else {
            load_planes_rw<T, 24>(yy, A.y, Vh, (size_t)cb);
#pragma unroll
            for (int i = 0; i < 24; i++) yy[i] += A.ck * acc[i];
        }
        store_planes<T, 24>(A.y, Vh, (size_t)cb, yy);
        store_planes<T, 24>(A.tm, Vh, (size_t)cb, acc);
    }
}

template <typename T, int RECON, int DAG> static cudaError_t hop_dispatch_mode(const HopArgs<T>& A, int mode, cudaStream_t st)
{
    const int threads = 128;
    const int blocks = (A.geo.Vh + threads - 1) / threads;
    switch (mode) {
    case HOP_PLAIN: hop_kernel<T, RECON, DAG, HOP_PLAIN><<<blocks, threads, 0, st>>>(A); break;
    case HOP_XPAY: hop_kernel<T, RECON, DAG, HOP_XPAY><<<blocks, threads, 0, st>>>(A); break;
    case HOP_CLOVER_Z: hop_kernel<T, RECON, DAG, HOP_CLOVER_Z><<<blocks, threads, 0, st>>>(A); break;
    case HOP_CLOVER_OUT: hop_kernel<T, RECON, DAG, HOP_CLOVER_OUT><<<blocks, threads, 0, st>>>(A); break;
    case HOP_CHEB: hop_kernel<T, RECON, DAG, HOP_CHEB><<<blocks, threads, 0, st>>>(A); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

template <typename T> static cudaError_t hop_dispatch(const HopArgs<T>& A, int recon, int dagger, int mode, cudaStream_t st)
{
    if (recon == 12)
        return dagger ? hop_dispatch_mode<T, 12, 1>(A, mode, st) : hop_dispatch_mode<T, 12, 0>(A, mode, st);
    return dagger ? hop_dispatch_mode<T, 18, 1>(A, mode, st) : hop_dispatch_mode<T, 18, 0>(A, mode, st);
}

template <typename T> static HopArgs<T> make_hop_args(const qcd_gauge* g, const HopLaunch& L)
{
    HopArgs<T> A;
    A.out = (T*)L.out;
    A.in = (const T*)L.in;
    A.z = (const T*)L.z;
    A.y = (T*)L.y;
    A.tm = (T*)L.tm;
    A.gauge = (const T*)g->data;
    A.clover = (const T*)L.clover;
    A.gblock = g->block_bytes / sizeof(T);
    A.geo = dev_geom(g->geo);
    A.parity = L.out_parity;
    A.tb = (T)g->tb;
    A.a = (T)L.a; A.b = (T)L.b; A.c0 = (T)L.c0; A.c1 = (T)L.c1; A.c2 = (T)L.c2; A.ck = (T)L.ck;
    A.y_init = L.y_init;
    return A;
}

#endif
