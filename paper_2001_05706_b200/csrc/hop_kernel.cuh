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
    const T* tm;   /* Chebyshev: b_{k+2}, own parity (may alias out)            */
    const T* v;    /* Chebyshev: the source vector, own parity                  */
    const T* gauge;
    const T* clover;
    size_t gblock; /* reals per (mu, parity) gauge block */
    size_t vstride; /* Chebyshev multi-rhs: reals between consecutive vectors   */
    int nvec;
    int tblock;     /* multi-rhs: t extent of the traversal tile (divides T)      */
    DevGeom geo;
    int parity;
    T tb;
    T a, b, c1, c2, c3;
    T s5; /* Chebyshev / multi-rhs epilogue: -1 applies gamma5 = diag(1,1,-1,-1), +1 does not */
    /* solver hooks: gate and the norm fused into the epilogue */
    const int* halt;        /* the launch does nothing while *halt != 0 (NULL: always run)     */
    double* norm_out;       /* |out|^2 (+ *norm_add) in fp64, NULL = not wanted                */
    const double* norm_add;
    double* norm_partial;   /* one slot per block                                              */
    unsigned int* norm_ticket;
    /* CG residual update fused into the epilogue (HopLaunch::cg_r) */
    T* cg_r;
    const double* cg_num;
    const double* cg_den;
    CgCtl* cg_ctl;
    int* cg_status;
};

/* |v|^2 of the block's sites, accumulated in fp64.  Deterministic two-level reduction over the grid:
 * every block writes its partial; the last block of each group of HOP_NORM_GROUP consecutive blocks to
 * take the group's ticket sums that group's partials in index order into a group partial, then takes
 * the top ticket, and the last group to do so sums the group partials in index order.  Which block does
 * a sum varies from run to run, what it sums and in which order does not.  (A single last block summing
 * all 16384 partials of a 32^3 x 64 launch with its 64 threads cost 21 us of tail per launch.)
 * Called by every thread of the block (inactive threads pass active = false). */
template <int THREADS> __device__ __forceinline__ double hop_block_sum(double s, double* sm)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads(); /* sm may still be read from the previous use */
    if (l == 0) sm[w] = s;
    __syncthreads();
    double b = 0.0;
#pragma unroll
    for (int i = 0; i < THREADS / 32; i++) b += sm[i];
    return b; /* the same value in every thread */
}

template <typename T, int THREADS>
__device__ __forceinline__ void hop_fused_norm(const HopArgs<T>& A, const T (&v)[24], bool active)
{
    __shared__ double sm[THREADS / 32];
    __shared__ int role; /* 0: done, 1: last block of its group, 2: also last group */
    double s = 0.0;
    if (active) {
#pragma unroll
        for (int i = 0; i < 24; i++) s += (double)v[i] * (double)v[i];
    }
    const double b = hop_block_sum<THREADS>(s, sm);
    const unsigned int nblocks = gridDim.x, ngroups = (nblocks + HOP_NORM_GROUP - 1) / HOP_NORM_GROUP;
    const unsigned int grp = blockIdx.x / HOP_NORM_GROUP;
    const unsigned int first = grp * HOP_NORM_GROUP;
    const unsigned int members = min((unsigned int)HOP_NORM_GROUP, nblocks - first);
    double* group_partial = A.norm_partial + nblocks;
    if (threadIdx.x == 0) {
        A.norm_partial[blockIdx.x] = b;
        __threadfence();
        const unsigned int t = atomicInc(A.norm_ticket + 1 + grp, members - 1); /* wraps back to 0 */
        role = (t == members - 1) ? 1 : 0;
    }
    __syncthreads();
    if (role == 0) return;
    __threadfence();
    double g = 0.0;
    for (unsigned int i = threadIdx.x; i < members; i += THREADS) g += __ldcg(A.norm_partial + first + i);
    g = hop_block_sum<THREADS>(g, sm);
    if (threadIdx.x == 0) {
        group_partial[grp] = g;
        __threadfence();
        const unsigned int t = atomicInc(A.norm_ticket, ngroups - 1);
        role = (t == ngroups - 1) ? 2 : 0;
    }
    __syncthreads();
    if (role != 2) return;
    __threadfence();
    double t = 0.0;
    for (unsigned int i = threadIdx.x; i < ngroups; i += THREADS) t += __ldcg(group_partial + i);
    t = hop_block_sum<THREADS>(t, sm);
    if (threadIdx.x == 0) {
        const double tot = t + (A.norm_add ? *A.norm_add : 0.0);
        *A.norm_out = tot;
        if (A.cg_ctl) cg_decide(A.cg_ctl, A.cg_status, tot);
    }
}

/* epilogue of the launch that computes q = (M^dag M p)(x) for this site: r -= alpha q in place of
 * storing q, alpha = cg_num / cg_den rounded to T (reading O6; O7: alpha = (float)(rho / <p,Np>)) */
template <typename T>
__device__ __forceinline__ void hop_cg_residual(const HopArgs<T>& A, T (&q)[24], size_t Vh, size_t cb, bool active)
{
    const T alpha = (T)(*A.cg_num / *A.cg_den);
    T rr[24];
    load_planes_rw<T, 24>(rr, A.cg_r, Vh, cb);
#pragma unroll
    for (int i = 0; i < 24; i++) q[i] = rr[i] - alpha * q[i];
    if (active) store_planes<T, 24>(A.cg_r, Vh, cb, q);
}

/* ---- where a neighbour spinor comes from ---------------------------------------------- */
template <typename T> struct PlaneSpinor {
    const T* base;
    size_t Vh;
    /* load() and Links::get() return the factor their values still have to be multiplied by
     * (1 here; the 16-bit sources return their scale so that it is applied once, to the
     * colour-multiplied half spinor, instead of to every decoded value) */
    __device__ __forceinline__ T load(T (&s)[24], int idx) const
    {
        load_planes<T, 24>(s, base, Vh, (size_t)idx);
        return (T)1;
    }
};

/* ---- where a direction's link comes from ------------------------------------------- */
template <typename T, int RECON> struct GlobalLinks {
    const T* gauge;
    size_t gblock, Vh;
    int parity;
    template <int MU, int DIR> __device__ __forceinline__ T get(T (&u)[18], int cb, int nb_cb) const
    {
        if (DIR > 0)
            load_link<T, RECON>(u, gauge + (size_t)(2 * MU + parity) * gblock, Vh, (size_t)cb);
        else
            load_link<T, RECON>(u, gauge + (size_t)(2 * MU + (1 - parity)) * gblock, Vh, (size_t)nb_cb);
        return (T)1;
    }
};

/* Per-thread slots in shared memory: slot (d, chunk) of thread tid at [(d*NCH + chunk)*128 + tid]
 * (128-bit words) -> conflict-free LDS.128 / STS.128; only the owning thread touches its slots,
 * so no barrier is needed.  Used by the multi-right-hand-side kernel to load each link from
 * HBM once per block instead of once per vector. */
template <typename T, int RECON> struct SmemLinks {
    typedef typename Vec<T>::type V;
    static constexpr int NCH = (RECON * (int)sizeof(T) + 15) / 16;
    V* slot; /* = smem + threadIdx.x */
    template <int MU, int DIR> __device__ __forceinline__ void put(const T (&u)[18]) const
    {
        constexpr int d = 2 * MU + (DIR < 0 ? 1 : 0);
        T r[NCH * Vec<T>::reals];
#pragma unroll
        for (int i = 0; i < NCH * Vec<T>::reals; i++) r[i] = (i < RECON) ? u[i] : (T)0;
#pragma unroll
        for (int c = 0; c < NCH; c++) slot[(d * NCH + c) * 128] = vec_make(&r[c * Vec<T>::reals]);
    }
    template <int MU, int DIR> __device__ __forceinline__ T get(T (&u)[18], int, int) const
    {
        constexpr int d = 2 * MU + (DIR < 0 ? 1 : 0);
        T r[NCH * Vec<T>::reals];
#pragma unroll
        for (int c = 0; c < NCH; c++) vec_get(slot[(d * NCH + c) * 128], &r[c * Vec<T>::reals]);
#pragma unroll
        for (int i = 0; i < RECON; i++) u[i] = r[i];
        if (RECON == 12) reconstruct_row2<T>(u);
        return (T)1;
    }
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
                /* one fused multiply-add per term: "re += ur*hr - ui*hi" in one statement costs three
                 * instructions (the bracket has to be rounded before it is added) */
                re += ur * hr;
                re -= ui * hi;
                im += ur * hi;
                im += ui * hr;
            }
            w[2 * (3 * j + a)] = sign * re;
            w[2 * (3 * j + a) + 1] = sign * im;
        }
}

/* one direction: MU, DIR = +1 forward / -1 backward; SG = projector sign (forward: -1, i.e. 1 - g) */
template <typename T, int MU, int DIR, int SG, typename Links, typename Src>
__device__ __forceinline__ void hop_dir(T (&acc)[24], const Links& L, const Src& in, int cb, int nb_cb, T sign)
{
    T s[24], u[18], h[12], w[12];
    const T fs = in.load(s, nb_cb);
    const T fu = L.template get<MU, DIR>(u, cb, nb_cb);
    project<T, MU, SG>(h, s);
    colour_mul<T, (DIR < 0)>(w, u, h, sign * fs * fu);
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
            re += lr * v[2 * j];
            re -= li * v[2 * j + 1];
            im += lr * v[2 * j + 1];
            im += li * v[2 * j];
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

/* neighbour checkerboard indices (periodic wrap; reading S3) and t-seam signs (S4) */
template <typename T> struct Neighbours {
    int xp, xm, yp, ym, zp, zm, tp, tm;
    T sgn_tp, sgn_tm;
    __device__ __forceinline__ Neighbours() {} /* filled in by the caller (hop_tile.cu: staged slots instead of cb) */
    __device__ __forceinline__ Neighbours(const DevGeom& g, int cb, int parity, T tb)
    {
        const Coord c = cb_to_coord(g, cb, parity);
        const int odd = c.x & 1;
        xp = odd ? (c.x == g.X - 1 ? cb - (g.X2 - 1) : cb + 1) : cb;
        xm = odd ? cb : (c.x == 0 ? cb + (g.X2 - 1) : cb - 1);
        const int sy = g.X2, sz = g.X2 * g.Y, st = g.X2 * g.Y * g.Z;
        yp = (c.y == g.Y - 1) ? cb - (g.Y - 1) * sy : cb + sy;
        ym = (c.y == 0) ? cb + (g.Y - 1) * sy : cb - sy;
        zp = (c.z == g.Z - 1) ? cb - (g.Z - 1) * sz : cb + sz;
        zm = (c.z == 0) ? cb + (g.Z - 1) * sz : cb - sz;
        tp = (c.t == g.T - 1) ? cb - (g.T - 1) * st : cb + st;
        tm = (c.t == 0) ? cb + (g.T - 1) * st : cb - st;
        sgn_tp = (c.t == g.T - 1) ? tb : (T)1;
        sgn_tm = (c.t == 0) ? tb : (T)1;
    }
};

/* acc = (H in)(cb) (or H^dag): the eight directions */
template <typename T, int DAG, typename Links, typename Src>
__device__ __forceinline__ void hop_site(T (&acc)[24], const Links& L, const Src& in, int cb, const Neighbours<T>& n)
{
    /* forward hop carries (1 - g_mu), backward (1 + g_mu); the adjoint swaps them (O4) */
    constexpr int SF = DAG ? +1 : -1;
    constexpr int SB = DAG ? -1 : +1;
#pragma unroll
    for (int i = 0; i < 24; i++) acc[i] = 0;
    hop_dir<T, 0, +1, SF>(acc, L, in, cb, n.xp, (T)1);
    hop_dir<T, 0, -1, SB>(acc, L, in, cb, n.xm, (T)1);
    hop_dir<T, 1, +1, SF>(acc, L, in, cb, n.yp, (T)1);
    hop_dir<T, 1, -1, SB>(acc, L, in, cb, n.ym, (T)1);
    hop_dir<T, 2, +1, SF>(acc, L, in, cb, n.zp, (T)1);
    hop_dir<T, 2, -1, SB>(acc, L, in, cb, n.zm, (T)1);
    hop_dir<T, 3, +1, SF>(acc, L, in, cb, n.tp, n.sgn_tp);
    hop_dir<T, 3, -1, SB>(acc, L, in, cb, n.tm, n.sgn_tm);
}

#ifndef HOP_THREADS
#define HOP_THREADS 64 /* threads per block of hop_kernel (swept on B200: 32 / 64 / 128 / 256 -> plain 12-real hop 100.7 / 100.9 /
                          102.6 / 104.8 us); the MINBLOCKS targets below are per 128 threads */
#endif
#ifndef HOP_MINBLOCKS_F32
#define HOP_MINBLOCKS_F32 4
#endif
#ifndef HOP_MINBLOCKS_F64
#define HOP_MINBLOCKS_F64 2
#endif

template <typename T, int RECON, int DAG, int MODE>
__global__ void __launch_bounds__(HOP_THREADS, (sizeof(T) == 4 ? HOP_MINBLOCKS_F32 : HOP_MINBLOCKS_F64) * 128 / HOP_THREADS) hop_kernel(const HopArgs<T> A)
{
    /* Programmatic dependent launch (hop_launch_pdl below): the next launch in the stream may place its blocks while
     * this grid's last wave drains and waits here until this grid has completed and its memory is visible.  Measured
     * on B200 (same build, QCD_PDL=0 / 1): bench step 284.1 -> 279.2 us, plain 12-real hop 98.5 -> 96.6 us, 16^3x32
     * Mhat in a loop 16.45 -> 13.71 us per apply.  Hoisting the neighbour table above the wait costs more in
     * registers (12 - 28 bytes of spills) than the overlap returns: 281.5 us. */
    pdl_launch_dependents();
    pdl_wait();
    if (A.halt && *reinterpret_cast<const volatile int*>(A.halt) != 0) return;
    const bool fuse_cg = (MODE == HOP_XPAY || MODE == HOP_CLOVER_Z) && A.cg_r != nullptr;
    if (fuse_cg && !(*A.cg_den > 0.0)) { /* breakdown: nothing is written */
        if (A.cg_ctl && blockIdx.x == 0 && threadIdx.x == 0) cg_flag_breakdown(A.cg_ctl, A.cg_status);
        return;
    }
    int cb = blockIdx.x * blockDim.x + threadIdx.x;
    const bool want_norm = (MODE == HOP_XPAY || MODE == HOP_CLOVER_Z) && A.norm_out != nullptr;
    const bool active = cb < A.geo.Vh;
    if (!active) {
        if (!want_norm) return;
        cb = A.geo.Vh - 1; /* ragged tail of a launch with a fused norm: computes a valid site, stores nothing */
    }
    const size_t Vh = (size_t)A.geo.Vh;
    const Neighbours<T> nb(A.geo, cb, A.parity, A.tb);
    const GlobalLinks<T, RECON> L = {A.gauge, A.gblock, Vh, A.parity};
    const PlaneSpinor<T> src = {A.in, Vh};
    T acc[24];
    hop_site<T, DAG>(acc, L, src, cb, nb);

    if (MODE == HOP_PLAIN) {
        store_planes<T, 24>(A.out, Vh, (size_t)cb, acc);
    } else if (MODE == HOP_XPAY) {
        T zz[24];
        load_planes_rw<T, 24>(zz, A.z, Vh, (size_t)cb);
#pragma unroll
        for (int i = 0; i < 24; i++) acc[i] = A.a * zz[i] + A.b * acc[i];
        if (fuse_cg) hop_cg_residual<T>(A, acc, Vh, (size_t)cb, active);
        else if (active) store_planes<T, 24>(A.out, Vh, (size_t)cb, acc);
        if (want_norm) hop_fused_norm<T, HOP_THREADS>(A, acc, active);
    } else if (MODE == HOP_CLOVER_Z) {
        T zz[24], az[24];
        load_planes_rw<T, 24>(zz, A.z, Vh, (size_t)cb);
        clover_apply<T>(az, A.clover, Vh, (size_t)cb, zz);
#pragma unroll
        for (int i = 0; i < 24; i++) acc[i] = A.a * az[i] + A.b * acc[i];
        if (fuse_cg) hop_cg_residual<T>(A, acc, Vh, (size_t)cb, active);
        else if (active) store_planes<T, 24>(A.out, Vh, (size_t)cb, acc);
        if (want_norm) hop_fused_norm<T, HOP_THREADS>(A, acc, active);
    } else if (MODE == HOP_CLOVER_OUT) {
        T o[24];
        clover_apply<T>(o, A.clover, Vh, (size_t)cb, acc);
        store_planes<T, 24>(A.out, Vh, (size_t)cb, o);
    }
}

/* ---- Chebyshev (Clenshaw) step for nvec right-hand sides -----
 *   out_j = c1 g5 (z_j + b H in_j) + c2 tm_j + c3 v_j          j = 0 .. nvec-1
 * with z_j the own-parity block of the field whose other-parity block is in_j.  The block's
 * 8 x 128 links are read from HBM once, parked in per-thread shared-memory slots and reused
 * for every vector, so the link traffic per site-vector is 8*RECON reals / nvec.  out may alias
 * tm (same index, same thread). */
template <typename T>
__device__ __forceinline__ void cheb_epilogue(const HopArgs<T>& A, T (&acc)[24], size_t off, size_t Vh, int cb)
{
    T zz[24];
    load_planes_cs<T, 24>(zz, A.z + off, Vh, (size_t)cb);
#pragma unroll
    for (int i = 0; i < 24; i++) {
        const T g5 = (i < 12) ? (T)1 : A.s5; /* gamma5 = diag(1,1,-1,-1) when s5 = -1 */
        acc[i] = A.c1 * g5 * (zz[i] + A.b * acc[i]);
    }
    if (A.c3 != (T)0) {
        load_planes_cs<T, 24>(zz, A.v + off, Vh, (size_t)cb);
#pragma unroll
        for (int i = 0; i < 24; i++) acc[i] += A.c3 * zz[i];
    }
    if (A.c2 != (T)0) {
        load_planes_cs<T, 24>(zz, A.tm + off, Vh, (size_t)cb);
#pragma unroll
        for (int i = 0; i < 24; i++) acc[i] += A.c2 * zz[i];
    }
    store_planes_cs<T, 24>(A.out + off, Vh, (size_t)cb, acc);
}

template <typename T, typename Links>
__device__ __forceinline__ void cheb_vector(const HopArgs<T>& A, const Links& L, size_t off, size_t Vh, int cb, const Neighbours<T>& nb)
{
    const PlaneSpinor<T> src = {A.in + off, Vh};
    T acc[24];
    hop_site<T, 0>(acc, L, src, cb, nb);
    cheb_epilogue<T>(A, acc, off, Vh, cb);
}

#ifndef HOP_CHEB_PREFETCH
#define HOP_CHEB_PREFETCH 1
#endif
/* Optional L2 prefetch (prefetch.global.L2, no register tied up) of what a vector of the multi-rhs
 * loop will read: bit 0 the own-site streams z / v / tm of the current vector, bit 2 those of the
 * next vector instead, bit 1 the x neighbours of the next vector, bit 3 all its neighbours.
 * Motivation: 59 % of the ncu stall samples are long-scoreboard waits, the largest at the first
 * use of direction 0 and of z / tm / v, whose loads the compiler cannot hoist across the vector
 * loop.  Measured on B200 (48^3x96, 12 vectors, degree 100): 0 -> 1.40 s, 1 -> 1.35 s, 2 -> 1.47 s,
 * 4 -> 1.44 s, 6 -> 1.57 s, 15 -> 1.84 s; ncu on one 12-vector launch: 6.31 ms -> 6.05 ms with bit 0,
 * DRAM traffic unchanged (36.6 GB).  Requesting neighbours a vector ahead costs more than it hides,
 * and so does letting only one lane per 128-byte line issue the request (bit 0: 1.42 s). */
template <typename T, int WHAT>
__device__ __forceinline__ void cheb_prefetch(const HopArgs<T>& A, size_t off, size_t Vh, int cb, const Neighbours<T>& nb)
{
    if (WHAT & 2) {
        const T* in = A.in + off;
        prefetch_planes_l2<T, 24>(in, Vh, (size_t)nb.xp);
        prefetch_planes_l2<T, 24>(in, Vh, (size_t)nb.xm);
        if (WHAT & 8) {
            prefetch_planes_l2<T, 24>(in, Vh, (size_t)nb.yp);
            prefetch_planes_l2<T, 24>(in, Vh, (size_t)nb.ym);
            prefetch_planes_l2<T, 24>(in, Vh, (size_t)nb.zp);
            prefetch_planes_l2<T, 24>(in, Vh, (size_t)nb.zm);
            prefetch_planes_l2<T, 24>(in, Vh, (size_t)nb.tp);
            prefetch_planes_l2<T, 24>(in, Vh, (size_t)nb.tm);
        }
    }
    if (WHAT & 1) {
        prefetch_planes_l2<T, 24>(A.z + off, Vh, (size_t)cb);
        if (A.c3 != (T)0) prefetch_planes_l2<T, 24>(A.v + off, Vh, (size_t)cb);
        if (A.c2 != (T)0) prefetch_planes_l2<T, 24>(A.tm + off, Vh, (size_t)cb);
    }
}

#ifndef HOP_MRHS_MINBLOCKS_F32
#define HOP_MRHS_MINBLOCKS_F32 4
#endif
/* Traversal order of the multi-rhs kernels: (x,y) fastest, then t inside a tile of tblock slices, then z,
 * then the tiles: with nvec vectors in flight the L2 footprint between the two uses of a +-t neighbour is
 * nvec planes instead of nvec time-slices, and between +-z uses nvec*tblock planes; only the tile faces in
 * t are fetched twice. */
__device__ __forceinline__ int mrhs_site(const DevGeom& g, int tblock, int cb)
{
    if (tblock <= 1) return cb;
    const unsigned P = (unsigned)(g.X2 * g.Y), TB = (unsigned)tblock, Z = (unsigned)g.Z;
    unsigned r = (unsigned)cb;
    const unsigned xy = r % P; r /= P;
    const unsigned tin = r % TB; r /= TB;
    const unsigned z = r % Z; const unsigned tout = r / Z;
    return (int)(xy + P * (z + Z * (tout * TB + tin)));
}

template <typename T, int RECON, typename Slots>
__device__ __forceinline__ void park_links(const Slots& S, const GlobalLinks<T, RECON>& G, int cb, const Neighbours<T>& nb)
{
    T u[18];
    G.template get<0, +1>(u, cb, nb.xp); S.template put<0, +1>(u);
    G.template get<0, -1>(u, cb, nb.xm); S.template put<0, -1>(u);
    G.template get<1, +1>(u, cb, nb.yp); S.template put<1, +1>(u);
    G.template get<1, -1>(u, cb, nb.ym); S.template put<1, -1>(u);
    G.template get<2, +1>(u, cb, nb.zp); S.template put<2, +1>(u);
    G.template get<2, -1>(u, cb, nb.zm); S.template put<2, -1>(u);
    G.template get<3, +1>(u, cb, nb.tp); S.template put<3, +1>(u);
    G.template get<3, -1>(u, cb, nb.tm); S.template put<3, -1>(u);
}

#ifndef HOP_MRHS_MINBLOCKS_F32
#define HOP_MRHS_MINBLOCKS_F32 4
#endif
/* STAGE = 1: nvec > 1, links parked in shared memory; STAGE = 0: one vector, links straight from HBM */
template <typename T, int RECON, int STAGE>
__global__ void __launch_bounds__(128, (sizeof(T) == 4 ? HOP_MRHS_MINBLOCKS_F32 : 2)) hop_cheb_mrhs_kernel(const HopArgs<T> A)
{
    typedef typename Vec<T>::type V;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    pdl_launch_dependents();
    pdl_wait();
    int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= A.geo.Vh) return;
    if (STAGE) cb = mrhs_site(A.geo, A.tblock, cb);
    const size_t Vh = (size_t)A.geo.Vh;
    const Neighbours<T> nb(A.geo, cb, A.parity, A.tb);
    const GlobalLinks<T, RECON> G = {A.gauge, A.gblock, Vh, A.parity};
    if (!STAGE) {
        cheb_vector<T>(A, G, 0, Vh, cb, nb);
        return;
    }
    const SmemLinks<T, RECON> S = {reinterpret_cast<V*>(smem_raw) + threadIdx.x};
    if (HOP_CHEB_PREFETCH & 4) cheb_prefetch<T, 1>(A, 0, Vh, cb, nb);
    park_links<T, RECON, SmemLinks<T, RECON> >(S, G, cb, nb);
    for (int j = 0; j < A.nvec; j++) {
        /* bit 0: own-site streams of this vector now; bit 2: of the next vector instead;
         * bit 1: x neighbours of the next vector; bit 3: all its neighbours */
        if ((HOP_CHEB_PREFETCH & 5) == 1) cheb_prefetch<T, 1>(A, (size_t)j * A.vstride, Vh, cb, nb);
        if ((HOP_CHEB_PREFETCH & 4) && j + 1 < A.nvec) cheb_prefetch<T, 1>(A, (size_t)(j + 1) * A.vstride, Vh, cb, nb);
        if ((HOP_CHEB_PREFETCH & 2) && j + 1 < A.nvec) cheb_prefetch<T, (HOP_CHEB_PREFETCH & 10)>(A, (size_t)(j + 1) * A.vstride, Vh, cb, nb);
        cheb_vector<T>(A, S, (size_t)j * A.vstride, Vh, cb, nb);
    }
}

template <typename T, int RECON> static cudaError_t hop_cheb_launch(const HopArgs<T>& A, cudaStream_t st)
{
    const int threads = 128;
    const int blocks = (A.geo.Vh + threads - 1) / threads;
    if (A.nvec == 1) {
        launch_pdl(hop_cheb_mrhs_kernel<T, RECON, 0>, blocks, threads, st, A);
        return cudaGetLastError();
    }
    const size_t smem = (size_t)8 * SmemLinks<T, RECON>::NCH * 128 * 16;
    /* the attribute is per device and the call is cheap: set it on every launch rather than cache it per process */
    cudaError_t e = cudaFuncSetAttribute(hop_cheb_mrhs_kernel<T, RECON, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    launch_pdl_smem(hop_cheb_mrhs_kernel<T, RECON, 1>, blocks, threads, smem, st, A);
    return cudaGetLastError();
}

template <typename T, int RECON, int DAG, int MODE> static cudaError_t hop_launch_pdl(const HopArgs<T>& A, int blocks, int threads, cudaStream_t st)
{
    launch_pdl(hop_kernel<T, RECON, DAG, MODE>, blocks, threads, st, A);
    return cudaGetLastError();
}

template <typename T, int RECON, int DAG> static cudaError_t hop_dispatch_mode(const HopArgs<T>& A, int mode, cudaStream_t st)
{
    const int threads = HOP_THREADS;
    const int blocks = (A.geo.Vh + threads - 1) / threads;
    switch (mode) {
    case HOP_PLAIN: return hop_launch_pdl<T, RECON, DAG, HOP_PLAIN>(A, blocks, threads, st);
    case HOP_XPAY: return hop_launch_pdl<T, RECON, DAG, HOP_XPAY>(A, blocks, threads, st);
    case HOP_CLOVER_Z: return hop_launch_pdl<T, RECON, DAG, HOP_CLOVER_Z>(A, blocks, threads, st);
    case HOP_CLOVER_OUT: return hop_launch_pdl<T, RECON, DAG, HOP_CLOVER_OUT>(A, blocks, threads, st);
    default: return cudaErrorInvalidValue;
    }
}

/* out(cb) = C(cb) in(cb) on one parity, C = A or A^-1 (two packed Hermitian 6x6 blocks per site).
 * Site-local, so out may be in.  Used by the even-odd source preparation / solution reconstruction (reading O5). */
template <typename T>
__global__ void __launch_bounds__(128) clover_site_kernel(T* out, const T* in, const T* __restrict__ clov, int Vh)
{
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= Vh) return;
    T v[24], o[24];
    load_planes_rw<T, 24>(v, in, (size_t)Vh, (size_t)cb);
    clover_apply<T>(o, clov, (size_t)Vh, (size_t)cb, v);
    store_planes<T, 24>(out, (size_t)Vh, (size_t)cb, o);
}

template <typename T> static cudaError_t clover_site_launch(void* out, const void* in, const void* clov, int Vh, cudaStream_t st)
{
    clover_site_kernel<T><<<(Vh + 127) / 128, 128, 0, st>>>((T*)out, (const T*)in, (const T*)clov, Vh);
    return cudaGetLastError();
}

template <typename T> static cudaError_t hop_dispatch(const HopArgs<T>& A, int recon, int dagger, int mode, cudaStream_t st)
{
    if (mode == HOP_CHEB) return recon == 12 ? hop_cheb_launch<T, 12>(A, st) : hop_cheb_launch<T, 18>(A, st);
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
    A.tm = (const T*)L.tm;
    A.v = (const T*)L.v;
    A.vstride = L.vstride;
    A.nvec = L.nvec;
    A.tblock = 1;
    /* t-tile of the multi-rhs traversal: swept on B200 (48^3x96, 12 vectors): 1 -> 1.45 s, 2 -> 1.41,
     * 4 -> 1.36, 8 -> 1.36, 16 -> 1.38, 32 -> 1.42; tiling y and z as well changes nothing (1.35-1.39) */
    for (int tbk = 8; tbk > 1; tbk >>= 1)
        if (g->geo.T % tbk == 0 && g->geo.T > tbk) { A.tblock = tbk; break; }
    A.gauge = (const T*)g->data;
    A.clover = (const T*)L.clover;
    A.gblock = g->block_bytes / sizeof(T);
    A.geo = dev_geom(g->geo);
    A.parity = L.out_parity;
    A.tb = (T)g->tb;
    A.a = (T)L.a; A.b = (T)L.b; A.c1 = (T)L.c1; A.c2 = (T)L.c2; A.c3 = (T)L.c3;
    A.s5 = (L.s5 == 0.0) ? (T)-1 : (T)L.s5;
    A.halt = L.halt;
    A.norm_out = L.norm_out;
    A.norm_add = L.norm_add;
    A.norm_partial = g->ctx->d_hop_partial;
    A.norm_ticket = g->ctx->d_hop_ticket; /* [0] the groups' ticket, [1 + g] group g's */
    A.cg_r = (T*)L.cg_r;
    A.cg_num = L.cg_num;
    A.cg_den = L.cg_den;
    A.cg_ctl = L.cg_ctl;
    A.cg_status = L.cg_status;
    return A;
}

#endif
