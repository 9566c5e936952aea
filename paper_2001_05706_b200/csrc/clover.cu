/*
 * clover.cu -- clover term construction (BASELINE.json configs[2]:
 * "clover field built from the plaquette field-strength F_munu with csw=1.0"; readings
 * O3/S9 in DESIGN.md).  Setup path: untimed, parity-checked.
 *
 *   Q_mn(x)  = sum of the four plaquette leaves in the (m,n) plane around x
 *   Fhat_mn  = (Q_mn - Q_mn^dag)/8
 *   A(x)     = 1 + kappa*csw * sum_{m<n} i sigma_mn (x) Fhat_mn(x),  sigma_mn = (i/2)[g_m, g_n]
 *
 * sigma_mn is block diagonal in chirality (gamma5 = diag(1,1,-1,-1)), so A is two
 * Hermitian 6x6 blocks, stored as 6 real diagonal + 15 complex lower entries each.
 * All arithmetic here is fp64 whatever the storage precision.
 */
#include <math.h>
#include <type_traits>

#include "half_device.cuh"

namespace {

struct cplx {
    double re, im;
};
__host__ __device__ inline cplx cmul(cplx a, cplx b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
__host__ __device__ inline cplx cadd(cplx a, cplx b) { return {a.re + b.re, a.im + b.im}; }
__host__ __device__ inline cplx csub(cplx a, cplx b) { return {a.re - b.re, a.im - b.im}; }
__host__ __device__ inline cplx cconj(cplx a) { return {a.re, -a.im}; }

/* i * sigma_mn, planes (01,02,03,12,13,23), 4x4 each; filled by the host at first use */
__constant__ cplx c_isigma[6][4][4];

/* DeGrand-Rossi gamma matrices (BASELINE.json configs[0]); entries are 0, +-1, +-i:
 * code 0 = 0, 1 = +1, 2 = -1, 3 = +i, 4 = -i. */
const int h_gamma_code[4][4][4] = {
    /* gamma_x */ {{0, 0, 0, 3}, {0, 0, 3, 0}, {0, 4, 0, 0}, {4, 0, 0, 0}},
    /* gamma_y */ {{0, 0, 0, 2}, {0, 0, 1, 0}, {0, 1, 0, 0}, {2, 0, 0, 0}},
    /* gamma_z */ {{0, 0, 3, 0}, {0, 0, 0, 4}, {4, 0, 0, 0}, {0, 3, 0, 0}},
    /* gamma_t */ {{0, 0, 1, 0}, {0, 0, 0, 1}, {1, 0, 0, 0}, {0, 1, 0, 0}}};

int upload_sigma()
{
    static bool done = false;
    cplx g[4][4][4];
    const cplx code[5] = {{0, 0}, {1, 0}, {-1, 0}, {0, 1}, {0, -1}};
    for (int m = 0; m < 4; m++)
        for (int i = 0; i < 4; i++)
            for (int j = 0; j < 4; j++) g[m][i][j] = code[h_gamma_code[m][i][j]];
    cplx is[6][4][4];
    int pl = 0;
    for (int m = 0; m < 4; m++)
        for (int n = m + 1; n < 4; n++, pl++)
            for (int i = 0; i < 4; i++)
                for (int j = 0; j < 4; j++) {
                    cplx c = {0, 0};
                    for (int k = 0; k < 4; k++) c = cadd(c, csub(cmul(g[m][i][k], g[n][k][j]), cmul(g[n][i][k], g[m][k][j])));
                    /* sigma = (i/2) [g_m, g_n];  i*sigma = -(1/2)[g_m, g_n] */
                    is[pl][i][j] = {-0.5 * c.re, -0.5 * c.im};
                }
    (void)done;
    cudaError_t e = cudaMemcpyToSymbol(c_isigma, is, sizeof(is));
    return e == cudaSuccess ? 0 : -1;
}

struct M3 {
    cplx m[9];
};
__device__ inline M3 mul(const M3& a, const M3& b)
{
    M3 c;
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            cplx s = {0, 0};
#pragma unroll
            for (int k = 0; k < 3; k++) s = cadd(s, cmul(a.m[3 * i + k], b.m[3 * k + j]));
            c.m[3 * i + j] = s;
        }
    return c;
}
__device__ inline M3 dag(const M3& a)
{
    M3 c;
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) c.m[3 * i + j] = cconj(a.m[3 * j + i]);
    return c;
}

/* c = a b, a b^dag (DB) */
template <int DB> __device__ __forceinline__ M3 mulx(const M3& a, const M3& b)
{
    M3 c;
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            cplx s = {0, 0};
#pragma unroll
            for (int k = 0; k < 3; k++) s = cadd(s, cmul(a.m[3 * i + k], DB ? cconj(b.m[3 * j + k]) : b.m[3 * k + j]));
            c.m[3 * i + j] = s;
        }
    return c;
}

template <typename T, int RECON> struct LinkReader {
    const T* data;
    size_t gblock;
    DevGeom g;
    /* U_mu at site c shifted by dm in direction m and dn in direction n (periodic); the
     * shifts are -1, 0 or +1 */
    __device__ __forceinline__ M3 get(int mu, const Coord& c, int m, int dm, int n, int dn) const
    {
        int x[4] = {c.x, c.y, c.z, c.t};
        const int L[4] = {g.X, g.Y, g.Z, g.T};
#pragma unroll
        for (int k = 0; k < 4; k++) { /* selects, not indexing: m and n are loop variables of a rolled loop */
            const int sh = (k == m ? dm : 0) + (k == n ? dn : 0);
            int v = x[k] + sh;
            v = v < 0 ? v + L[k] : (v >= L[k] ? v - L[k] : v);
            x[k] = v;
        }
        const int parity = (x[0] + x[1] + x[2] + x[3]) & 1;
        const int cb = coord_to_cb(g, x[0], x[1], x[2], x[3]);
        T u[18];
        load_link<T, RECON>(u, data + (size_t)(2 * mu + parity) * gblock, (size_t)g.Vh, (size_t)cb);
        M3 r;
#pragma unroll
        for (int k = 0; k < 9; k++) r.m[k] = {(double)u[2 * k], (double)u[2 * k + 1]};
        return r;
    }
};

__host__ __device__ constexpr int tri_index(int hi, int lo) { return 5 * lo - (lo * (lo - 1)) / 2 + (hi - lo - 1); }

/* Packed Hermitian 6x6 block (the storage format): p[0..5] the diagonal, p[6 + 2 t], p[7 + 2 t] = Re, Im of a[hi][lo],
 * t = tri_index(hi, lo), hi > lo.  In-place inverse through p = L D L^dag (L unit lower triangular, D real), M = L^-1,
 * p^-1 = M^dag D^-1 M; every index is a compile-time constant, the 36 reals stay in registers.  No pivoting:
 * A = 1 + kappa csw C is positive definite for every physical (kappa, csw); a vanishing or non-finite pivot
 * reports the block as singular. */
__device__ __forceinline__ cplx pk_get(const double (&p)[36], int hi, int lo) { return {p[6 + 2 * tri_index(hi, lo)], p[7 + 2 * tri_index(hi, lo)]}; }
__device__ __forceinline__ void pk_set(double (&p)[36], int hi, int lo, cplx v)
{
    p[6 + 2 * tri_index(hi, lo)] = v.re;
    p[7 + 2 * tri_index(hi, lo)] = v.im;
}
__device__ __forceinline__ bool invert_packed(double (&p)[36])
{
    bool ok = true;
    /* p = L D L^dag in place: diagonal <- 1 / d_j, lower triangle <- L */
#pragma unroll
    for (int j = 0; j < 6; j++) {
        double dj = p[j];
#pragma unroll
        for (int k = 0; k < j; k++) {
            const cplx l = pk_get(p, j, k);
            dj -= (l.re * l.re + l.im * l.im) / p[k];
        }
        ok = ok && (fabs(dj) > 1e-300) && (fabs(dj) < 1e300);
        const double dinv = 1.0 / dj;
#pragma unroll
        for (int i = j + 1; i < 6; i++) {
            cplx v = pk_get(p, i, j);
#pragma unroll
            for (int k = 0; k < j; k++) {
                const cplx t = cmul(pk_get(p, i, k), cconj(pk_get(p, j, k)));
                v.re -= t.re / p[k];
                v.im -= t.im / p[k];
            }
            pk_set(p, i, j, {v.re * dinv, v.im * dinv});
        }
        p[j] = dinv;
    }
    /* lower triangle <- M = L^-1, column by column (column j needs L of the columns to its right, still in place) */
#pragma unroll
    for (int j = 0; j < 6; j++)
#pragma unroll
        for (int i = j + 1; i < 6; i++) {
            cplx v = pk_get(p, i, j);
#pragma unroll
            for (int k = j + 1; k < i; k++) v = cadd(v, cmul(pk_get(p, i, k), pk_get(p, k, j)));
            pk_set(p, i, j, {-v.re, -v.im});
        }
    /* p <- M^dag D^-1 M, row by row from the top: entry (i,j) needs rows >= i only, its own row only at (i,j) itself */
#pragma unroll
    for (int i = 0; i < 6; i++) {
#pragma unroll
        for (int j = 0; j < i; j++) {
            const cplx mij = pk_get(p, i, j);
            cplx s = {mij.re * p[i], mij.im * p[i]};
#pragma unroll
            for (int k = i + 1; k < 6; k++) {
                const cplx t = cmul(cconj(pk_get(p, k, i)), pk_get(p, k, j));
                s.re += t.re * p[k];
                s.im += t.im * p[k];
            }
            pk_set(p, i, j, s);
        }
        double s = p[i];
#pragma unroll
        for (int k = i + 1; k < 6; k++) {
            const cplx m = pk_get(p, k, i);
            s += (m.re * m.re + m.im * m.im) * p[k];
        }
        p[i] = s;
    }
    return ok;
}

template <typename TS> __device__ __forceinline__ void store_block(TS* blk, size_t Vh, size_t cb, int b, const double (&p)[36])
{
    TS r[36];
#pragma unroll
    for (int k = 0; k < 36; k++) r[k] = (TS)p[k];
    store_planes<TS, 36>(blk + (size_t)36 * b * Vh, Vh, cb, r);
}

/* tag type: 16-bit storage (reading H1) */
struct HalfTag {};

/* both chiral blocks of a site (72 reals) -> int16 codes + site norm */
__device__ __forceinline__ void store_site_half(unsigned char* blk, size_t Vh, size_t cb, const double (&p0)[36], const double (&p1)[36])
{
    float r[72];
#pragma unroll
    for (int k = 0; k < 36; k++) { r[k] = (float)p0[k]; r[36 + k] = (float)p1[k]; }
    float n = 0.f;
#pragma unroll
    for (int k = 0; k < 72; k++) n = fmaxf(n, fabsf(r[k]));
    const float scale = n > 0.f ? __fdiv_rn(32767.0f, n) : 0.f;
    int4* q = reinterpret_cast<int4*>(blk) + cb;
#pragma unroll
    for (int c = 0; c < 9; c++) q[(size_t)c * Vh] = half_pack8(&r[8 * c], scale);
    reinterpret_cast<float*>(blk + Vh * 144)[cb] = n;
}

/* One thread per site.  The six planes, the four leaves of each and all matrix indices are unrolled, so the two
 * packed blocks (72 reals) and the running products live in registers: round 1's kernel kept two dense 6x6 complex
 * blocks and the Gauss-Jordan work matrix in 1744 B of dynamically indexed local memory per thread, which
 * fell out of L2 next to the streamed links (ncu: 21 GB of DRAM traffic for 2.4 GB of links and output). */
template <typename T, int RECON, typename TS>
__global__ void __launch_bounds__(64) clover_build_kernel(LinkReader<T, RECON> R, TS* A, TS* Ainv, size_t cblock, double coeff, int* bad)
{
    const DevGeom& g = R.g;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 2 * g.Vh) return;
    const int parity = i / g.Vh, cb = i - parity * g.Vh;
    const Coord c = cb_to_coord(g, cb, parity);

    double P[2][36];
#pragma unroll
    for (int b = 0; b < 2; b++)
#pragma unroll
        for (int k = 0; k < 36; k++) P[b][k] = 0.0;

#pragma unroll 1
    for (int pl = 0; pl < 6; pl++) {
        {
            const int m = pl < 3 ? 0 : (pl < 5 ? 1 : 2), n = pl < 3 ? pl + 1 : (pl < 5 ? pl - 1 : 3);
            /* the four leaves, each a closed loop x -> ... -> x, counter-clockwise in (m,n) */
            M3 q = mulx<1>(mulx<1>(mulx<0>(R.get(m, c, m, 0, n, 0), R.get(n, c, m, 1, n, 0)), R.get(m, c, m, 0, n, 1)), R.get(n, c, m, 0, n, 0));
            M3 l = mulx<0>(mulx<1>(mulx<1>(R.get(n, c, m, 0, n, 0), R.get(m, c, m, -1, n, 1)), R.get(n, c, m, -1, n, 0)), R.get(m, c, m, -1, n, 0));
#pragma unroll
            for (int k = 0; k < 9; k++) q.m[k] = cadd(q.m[k], l.m[k]);
            l = mulx<0>(mulx<0>(mulx<1>(dag(R.get(m, c, m, -1, n, 0)), R.get(n, c, m, -1, n, -1)), R.get(m, c, m, -1, n, -1)), R.get(n, c, m, 0, n, -1));
#pragma unroll
            for (int k = 0; k < 9; k++) q.m[k] = cadd(q.m[k], l.m[k]);
            l = mulx<1>(mulx<0>(mulx<0>(dag(R.get(n, c, m, 0, n, -1)), R.get(m, c, m, 0, n, -1)), R.get(n, c, m, 1, n, -1)), R.get(m, c, m, 0, n, 0));
#pragma unroll
            for (int k = 0; k < 9; k++) q.m[k] = cadd(q.m[k], l.m[k]);
            /* Fhat = (Q - Q^dag)/8;  C += (i sigma_mn) (x) Fhat, chirality block by block, lower triangle only */
#pragma unroll
            for (int b = 0; b < 2; b++)
#pragma unroll
                for (int s = 0; s < 2; s++)
#pragma unroll
                    for (int sp = 0; sp <= s; sp++) {
                        const cplx sg = c_isigma[pl][2 * b + s][2 * b + sp];
#pragma unroll
                        for (int a = 0; a < 3; a++)
#pragma unroll
                            for (int bb = 0; bb < 3; bb++) {
                                const int row = 3 * s + a, col = 3 * sp + bb;
                                if (row < col) continue;
                                const cplx dq = csub(q.m[3 * a + bb], cconj(q.m[3 * bb + a]));
                                const cplx f = {0.125 * dq.re, 0.125 * dq.im};
                                const cplx v = cmul(sg, f);
                                if (row == col) P[b][row] += v.re;
                                else { P[b][6 + 2 * tri_index(row, col)] += v.re; P[b][7 + 2 * tri_index(row, col)] += v.im; }
                            }
                    }
        }
    }

#pragma unroll
    for (int b = 0; b < 2; b++)
#pragma unroll
        for (int k = 0; k < 36; k++) P[b][k] = P[b][k] * coeff + (k < 6 ? 1.0 : 0.0);
    constexpr bool HALF = std::is_same<TS, HalfTag>::value;
    if constexpr (HALF) store_site_half(reinterpret_cast<unsigned char*>(A) + (size_t)parity * cblock, (size_t)g.Vh, (size_t)cb, P[0], P[1]);
    else {
        store_block<TS>(A + (size_t)parity * cblock, (size_t)g.Vh, (size_t)cb, 0, P[0]);
        store_block<TS>(A + (size_t)parity * cblock, (size_t)g.Vh, (size_t)cb, 1, P[1]);
    }
    if (!invert_packed(P[0])) atomicAdd(bad, 1);
    if (!invert_packed(P[1])) atomicAdd(bad, 1);
    if constexpr (HALF) store_site_half(reinterpret_cast<unsigned char*>(Ainv) + (size_t)parity * cblock, (size_t)g.Vh, (size_t)cb, P[0], P[1]);
    else {
        store_block<TS>(Ainv + (size_t)parity * cblock, (size_t)g.Vh, (size_t)cb, 0, P[0]);
        store_block<TS>(Ainv + (size_t)parity * cblock, (size_t)g.Vh, (size_t)cb, 1, P[1]);
    }
}

/* expand packed blocks to dense 12x12 complex per site, boundary site order, fp64 */
template <typename TS> __global__ void clover_unpack_kernel(double* dense, const TS* C, size_t cblock, DevGeom g)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 2 * g.Vh) return;
    const int parity = i / g.Vh, cb = i - parity * g.Vh;
    const Coord c = cb_to_coord(g, cb, parity);
    const size_t s = (size_t)c.x + (size_t)g.X * (c.y + (size_t)g.Y * (c.z + (size_t)g.Z * c.t));
    double* d = dense + s * 288;
    for (int k = 0; k < 288; k++) d[k] = 0.0;
    for (int b = 0; b < 2; b++) {
        TS r[36];
        load_planes_rw<TS, 36>(r, C + (size_t)parity * cblock + (size_t)36 * b * g.Vh, (size_t)g.Vh, (size_t)cb);
        for (int ii = 0; ii < 6; ii++) {
            const int row = 6 * b + ii;
            d[(row * 12 + row) * 2] = (double)r[ii];
            for (int jj = 0; jj < ii; jj++) {
                const int col = 6 * b + jj;
                const int k = 6 + 2 * tri_index(ii, jj);
                d[(row * 12 + col) * 2] = (double)r[k];
                d[(row * 12 + col) * 2 + 1] = (double)r[k + 1];
                d[(col * 12 + row) * 2] = (double)r[k];
                d[(col * 12 + row) * 2 + 1] = -(double)r[k + 1];
            }
        }
    }
}

__global__ void clover_unpack_half_kernel(double* dense, const unsigned char* C, size_t cblock, DevGeom g)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 2 * g.Vh) return;
    const int parity = i / g.Vh, cb = i - parity * g.Vh;
    const Coord c = cb_to_coord(g, cb, parity);
    const size_t s = (size_t)c.x + (size_t)g.X * (c.y + (size_t)g.Y * (c.z + (size_t)g.Z * c.t));
    double* d = dense + s * 288;
    for (int k = 0; k < 288; k++) d[k] = 0.0;
    for (int b = 0; b < 2; b++) {
        float r[36];
        half_load_clover_block(r, C + (size_t)parity * cblock, (size_t)g.Vh, (size_t)cb, b);
        for (int ii = 0; ii < 6; ii++) {
            const int row = 6 * b + ii;
            d[(row * 12 + row) * 2] = (double)r[ii];
            for (int jj = 0; jj < ii; jj++) {
                const int col = 6 * b + jj;
                const int k = 6 + 2 * tri_index(ii, jj);
                d[(row * 12 + col) * 2] = (double)r[k];
                d[(row * 12 + col) * 2 + 1] = (double)r[k + 1];
                d[(col * 12 + row) * 2] = (double)r[k];
                d[(col * 12 + row) * 2 + 1] = -(double)r[k + 1];
            }
        }
    }
}

template <typename T, int RECON>
cudaError_t build_launch(qcd_ctx* ctx, const qcd_gauge* gh, const qcd_clover* c, int* d_bad)
{
    LinkReader<T, RECON> R;
    R.data = (const T*)gh->data;
    R.gblock = gh->block_bytes / sizeof(T);
    R.g = dev_geom(gh->geo);
    const int threads = 64, blocks = (2 * R.g.Vh + threads - 1) / threads;
    const double coeff = c->kappa * c->csw;
    if (c->precision == 2) {
        /* cblock in bytes; A, Ainv addressed as bytes inside the kernel */
        HalfTag* A = (HalfTag*)c->data;
        clover_build_kernel<T, RECON, HalfTag><<<blocks, threads, 0, ctx->stream>>>(R, A, (HalfTag*)((unsigned char*)c->data + 2 * c->block_bytes),
                                                                                 c->block_bytes, coeff, d_bad);
    } else if (c->precision == 4) {
        const size_t cblock = c->block_bytes / 4;
        float* A = (float*)c->data;
        clover_build_kernel<T, RECON, float><<<blocks, threads, 0, ctx->stream>>>(R, A, A + 2 * cblock, cblock, coeff, d_bad);
    } else {
        const size_t cblock = c->block_bytes / 8;
        double* A = (double*)c->data;
        clover_build_kernel<T, RECON, double><<<blocks, threads, 0, ctx->stream>>>(R, A, A + 2 * cblock, cblock, coeff, d_bad);
    }
    return cudaGetLastError();
}

} // namespace

int clover_build(qcd_ctx* ctx, const qcd_gauge* g, const qcd_clover* c)
{
    if (upload_sigma() != 0) return qcd_set_error(QCD_ECUDA, "clover: constant upload failed");
    int* d_bad = reinterpret_cast<int*>(ctx->d_ticket + 8);
    QCD_CHECK_CUDA(cudaMemsetAsync(d_bad, 0, sizeof(int), ctx->stream));
    cudaError_t e;
    if (g->precision == 4)
        e = (g->reconstruct == 12) ? build_launch<float, 12>(ctx, g, c, d_bad) : build_launch<float, 18>(ctx, g, c, d_bad);
    else
        e = (g->reconstruct == 12) ? build_launch<double, 12>(ctx, g, c, d_bad) : build_launch<double, 18>(ctx, g, c, d_bad);
    if (e != cudaSuccess) return qcd_set_error(QCD_ECUDA, "clover build: %s", cudaGetErrorString(e));
    ctx->launches++;
    int bad = 0;
    QCD_CHECK_CUDA(cudaMemcpyAsync(&bad, d_bad, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    QCD_CHECK_CUDA(cudaStreamSynchronize(ctx->stream));
    if (bad) return qcd_set_error(QCD_EBREAKDOWN, "clover: %d singular 6x6 blocks", bad);
    return QCD_OK;
}

int clover_unpack(qcd_ctx* ctx, void* dense, const qcd_clover* c, int which)
{
    const DevGeom g = dev_geom(c->geo);
    const int threads = 64, blocks = (2 * g.Vh + threads - 1) / threads;
    if (c->precision == 2) {
        clover_unpack_half_kernel<<<blocks, threads, 0, ctx->stream>>>((double*)dense, (const unsigned char*)c->data + (which ? 2 * c->block_bytes : 0),
                                                                     c->block_bytes, g);
    } else if (c->precision == 4) {
        const size_t cblock = c->block_bytes / 4;
        clover_unpack_kernel<float><<<blocks, threads, 0, ctx->stream>>>((double*)dense, (const float*)c->data + (which ? 2 * cblock : 0), cblock, g);
    } else {
        const size_t cblock = c->block_bytes / 8;
        clover_unpack_kernel<double><<<blocks, threads, 0, ctx->stream>>>((double*)dense, (const double*)c->data + (which ? 2 * cblock : 0), cblock, g);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return qcd_set_error(QCD_ECUDA, "clover unpack: %s", cudaGetErrorString(e));
    ctx->launches++;
    return QCD_OK;
}
