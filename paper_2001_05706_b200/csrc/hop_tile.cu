/*
 * hop_tile.cu -- the multi-right-hand-side hopping term with the neighbour spinors of a 4-D
 * tile staged through shared memory (BASELINE.json north_star (2):
 * "neighbour spinors staged through shared memory"; PAPER.md:155 many-vector overlap workload).
 *
 *   out_j = c1 g5 (z_j + b H in_j) + c2 tm_j + c3 v_j        j = 0 .. nvec-1   (mode HOP_CHEB)
 *
 * Why.  ncu on the round-1 kernel (one thread per site, 128 consecutive sites per block, every
 * neighbour read through L1/L2; profiles/hop_cheb_mrhs_r2.md): 897 B per site-vector cross the
 * L2 -> SM fabric for 512 B of algorithmic traffic, 9.6 TB/s at 1.59 GHz, and the kernel's time follows
 * those bytes (HBM is at 74 %).  Each input spinor is wanted by 8 output sites; when a block
 * owns a compact 4-D tile most of those sites are its own, so it fetches the tile's rows once
 * per vector into shared memory (cp.async, 16 B per request, no registers) and the neighbour
 * reads that fall inside the tile become conflict-free LDS.128 with immediate offsets.
 *
 * Block = NG groups of NT threads on one tile of NT = WX x WY x WZ x WT output sites of one
 * parity (WX counts checkerboard columns, i.e. 2 WX lattice sites in x).  Thread (g, s) works on
 * site s for the vectors g, g + NG, g + 2 NG, ...: NG vectors are in flight per tile, each group
 * with its own staging buffers, all groups sharing the parked links.  Shared memory:
 *   links  8 directions x 3 chunks x NT float4   parked once, reused by every group and vector
 *   core   NG x 6 chunks x CORE float4           the tile's other-parity rows, one vector per group
 *   own    NG x NOWN x 6 chunks x NT float4      the site-local streams z, tm, v of that vector
 *   tab    CORE ints                             checkerboard index of every staged slot
 * Staged rows: each of the tile's WY WZ WT rows with the one x-halo column it needs (a row whose
 * output sites sit at even x needs the column to its left, at odd x the one to its right).  The
 * six faces are NOT staged: a face element is wanted exactly once, so it is read straight from
 * global memory by the one thread that wants it.  For (8,4,2,2): 144 staged slots + 320 face reads
 * for 128 outputs = 3.6 fetches per output site instead of 8 x (1 - L1 hit rate).
 * A group's core buffer is free as soon as its neighbour reads are done, so the next vector's rows
 * are requested before the site-local epilogue of the current one runs; the epilogue's own streams
 * were requested a whole vector earlier and are read from shared memory.
 */
#include "hop_kernel.cuh"

#include <stdlib.h>

namespace {

template <int WX_, int WY_, int WZ_, int WT_> struct Tile {
    static constexpr int WX = WX_, WY = WY_, WZ = WZ_, WT = WT_;
    static constexpr int NT = WX * WY * WZ * WT; /* output sites */
    static constexpr int ROW = WX + 1;           /* a row with the x-halo column it needs */
    static constexpr int CORE = WT * WZ * WY * ROW;
    static constexpr int NCH = 3; /* 12-real fp32 link = 3 float4 */
    __host__ __device__ static constexpr size_t smem(int ng, int nown)
    {
        return (size_t)(8 * NCH * NT + ng * 6 * (2 * CORE + nown * NT)) * 16 + (size_t)CORE * 4;
    }
    __host__ __device__ static constexpr int core(int lt, int lz, int ly) { return ((lt * WZ + lz) * WY + ly) * ROW; }
};

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
/* wait until at most N of this thread's committed groups are still in flight */
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
/* barrier among the `count` threads of one group (barrier 0 is __syncthreads) */
__device__ __forceinline__ void group_sync(int id, int count)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory");
}

__device__ __forceinline__ int wrap(int v, int n) { return v < 0 ? v + n : (v >= n ? v - n : v); }

/* checkerboard index (other parity) of staged slot i of the tile at (x0,y0,z0,t0) */
template <typename TL>
__device__ __forceinline__ int slot_cb(int i, int x0, int y0, int z0, int t0, const DevGeom& g, int parity)
{
    const int k = i % TL::ROW;
    int r = i / TL::ROW;
    const int ly = r % TL::WY; r /= TL::WY;
    const int lz = r % TL::WZ, lt = r / TL::WZ;
    const int y = y0 + ly, z = z0 + lz, t = t0 + lt;
    /* the OUTPUT sites of this row sit at x = 2 x2 + rp; their x+ / x- neighbours are the inputs at
     * x2 + rp and x2 - 1 + rp: columns k - 1 + rp, k = 0 .. WX, of the row are wanted */
    const int rp = (y + z + t + parity) & 1;
    const int x2 = wrap(x0 + k - 1 + rp, g.X2);
    return x2 + g.X2 * (y + g.Y * (z + g.Z * t));
}

/* neighbour spinor: idx >= 0 is a staged slot, idx < 0 is ~cb of a face site read from global memory */
template <int CORE> struct TileSpinor {
    const float4* buf;
    const float4* in;
    size_t Vh;
    __device__ __forceinline__ float load(float (&s)[24], int idx) const
    {
        if (idx >= 0) {
            const float4* p = buf + idx;
#pragma unroll
            for (int c = 0; c < 6; c++) vec_get(p[c * CORE], &s[4 * c]);
        } else {
            const float4* p = in + (size_t)(~idx);
#pragma unroll
            for (int c = 0; c < 6; c++) vec_get(__ldg(p + (size_t)c * Vh), &s[4 * c]);
        }
        return 1.f;
    }
};

/* per-site link slots, as SmemLinks of hop_kernel.cuh but for NT sites */
template <int NT> struct TileLinks {
    float4* slot; /* = links + site */
    template <int MU, int DIR> __device__ __forceinline__ void put(const float (&u)[18]) const
    {
        constexpr int d = 2 * MU + (DIR < 0 ? 1 : 0);
#pragma unroll
        for (int c = 0; c < 3; c++) slot[(d * 3 + c) * NT] = vec_make(&u[4 * c]);
    }
    template <int MU, int DIR> __device__ __forceinline__ float get(float (&u)[18], int, int) const
    {
        constexpr int d = 2 * MU + (DIR < 0 ? 1 : 0);
#pragma unroll
        for (int c = 0; c < 3; c++) vec_get(slot[(d * 3 + c) * NT], &u[4 * c]);
        reconstruct_row2<float>(u);
        return 1.f;
    }
};

/* own-site stream k of the epilogue (0: z, 1: tm, 2: v): from shared memory when staged, else from global */
template <int NT, int NOWN, int K>
__device__ __forceinline__ void own_load(float (&d)[24], const float4* own, const float* g, size_t Vh, size_t cb)
{
    if (K < NOWN) {
#pragma unroll
        for (int c = 0; c < 6; c++) vec_get(own[(K * 6 + c) * NT], &d[4 * c]);
    } else {
        load_planes_cs<float, 24>(d, g, Vh, cb);
    }
}

template <typename TL, int NG, int NOWN>
__global__ void __launch_bounds__(TL::NT * NG, 1) hop_mrhs_tile_kernel(const HopArgs<float> A, int nbx, int nby, int nbz, int tgroup)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4* links = reinterpret_cast<float4*>(smem_raw);
    float4* stage0 = links + 8 * TL::NCH * TL::NT;
    int* tab = reinterpret_cast<int*>(stage0 + NG * 6 * (2 * TL::CORE + NOWN * TL::NT));
    const DevGeom& g = A.geo;
    const size_t Vh = (size_t)g.Vh;

    /* tile order: (x, y) fastest, then t inside a group of `tgroup` tiles, then z, then the groups:
     * between the two uses of a t-face by neighbouring tiles only nvec xy-layers of tiles pass through
     * L2, between the uses of a z-face nvec * tgroup of them (same idea as the round-1 traversal) */
    unsigned r = blockIdx.x;
    const int bx = r % nbx; r /= nbx;
    const int by = r % nby; r /= nby;
    const int tin = r % tgroup; r /= tgroup;
    const int bz = r % nbz;
    const int bt = (r / nbz) * tgroup + tin;
    const int x0 = bx * TL::WX, y0 = by * TL::WY, z0 = bz * TL::WZ, t0 = bt * TL::WT;

    const int grp = threadIdx.x / TL::NT, tid = threadIdx.x % TL::NT;
    const int lx = tid % TL::WX;
    const int ly = (tid / TL::WX) % TL::WY;
    const int lz = (tid / (TL::WX * TL::WY)) % TL::WZ;
    const int lt = tid / (TL::WX * TL::WY * TL::WZ);
    const int x2 = x0 + lx, y = y0 + ly, z = z0 + lz, t = t0 + lt;
    const int sy = g.X2, sz = g.X2 * g.Y, st = g.X2 * g.Y * g.Z;
    const int cb = x2 + sy * y + sz * z + st * t;
    const int rp = (y + z + t + A.parity) & 1; /* this output site sits at x = 2 x2 + rp */

    for (int i = threadIdx.x; i < TL::CORE; i += TL::NT * NG) tab[i] = slot_cb<TL>(i, x0, y0, z0, t0, g, A.parity);

    /* where this site's eight neighbours are.  Column c of a staged row with parity q is slot
     * c + 1 - q: in this site's own row (q = rp) the x+ / x- inputs at columns lx + rp and lx - 1 + rp
     * are slots lx + 1 and lx; a row one step away in y, z or t has q = 1 - rp and the input at
     * column lx (same x2, same x) is slot lx + rp.  Outside the tile: ~cb of the face site. */
    Neighbours<float> ns;
    const int row = TL::core(lt, lz, ly), o = lx + rp;
    ns.xp = row + lx + 1;
    ns.xm = row + lx;
    ns.yp = (ly + 1 < TL::WY) ? TL::core(lt, lz, ly + 1) + o : ~(cb + sy * (wrap(y + 1, g.Y) - y));
    ns.ym = (ly > 0) ? TL::core(lt, lz, ly - 1) + o : ~(cb + sy * (wrap(y - 1, g.Y) - y));
    ns.zp = (lz + 1 < TL::WZ) ? TL::core(lt, lz + 1, ly) + o : ~(cb + sz * (wrap(z + 1, g.Z) - z));
    ns.zm = (lz > 0) ? TL::core(lt, lz - 1, ly) + o : ~(cb + sz * (wrap(z - 1, g.Z) - z));
    ns.tp = (lt + 1 < TL::WT) ? TL::core(lt + 1, lz, ly) + o : ~(cb + st * (wrap(t + 1, g.T) - t));
    ns.tm = (lt > 0) ? TL::core(lt - 1, lz, ly) + o : ~(cb + st * (wrap(t - 1, g.T) - t));
    ns.sgn_tp = (t == g.T - 1) ? A.tb : 1.f;
    ns.sgn_tm = (t == 0) ? A.tb : 1.f;
    __syncthreads();

    float4* core0 = stage0 + grp * 6 * (2 * TL::CORE + NOWN * TL::NT); /* two row buffers, then the own-site slots */
    float4* own = core0 + 12 * TL::CORE + tid;

    /* request the tile rows of vector j (other-parity block) into row buffer b */
    auto stage_core = [&](int j, int b) {
        if (j < A.nvec) {
            const float4* in = reinterpret_cast<const float4*>(A.in + (size_t)j * A.vstride);
            float4* core = core0 + b * 6 * TL::CORE;
            for (int i = tid; i < TL::CORE; i += TL::NT) {
                const float4* p = in + tab[i];
#pragma unroll
                for (int ch = 0; ch < 6; ch++) cp_async16(core + ch * TL::CORE + i, p + (size_t)ch * Vh);
            }
        }
        cp_async_commit(); /* always: the group count per iteration is what the waits below rely on */
    };
    /* request this site's own streams of vector j: z, tm, v in that order, the first NOWN of them into
     * shared memory, the others towards L2 */
    auto stage_own = [&](int j) {
        if (j < A.nvec) {
            const size_t off = (size_t)j * A.vstride;
            const float* sp[3] = {A.z + off, A.tm + off, A.v + off};
            const bool used[3] = {true, A.c2 != 0.f, A.c3 != 0.f};
#pragma unroll
            for (int k = 0; k < 3; k++) {
                if (!used[k]) continue;
                if (k < NOWN) {
                    const float4* p = reinterpret_cast<const float4*>(sp[k]) + cb;
#pragma unroll
                    for (int ch = 0; ch < 6; ch++) cp_async16(own + (k * 6 + ch) * TL::NT, p + (size_t)ch * Vh);
                } else {
                    prefetch_planes_l2<float, 24>(sp[k], Vh, (size_t)cb);
                }
            }
        }
        cp_async_commit();
    };

    /* the first vector's rows and own streams are requested before the links are fetched */
    stage_core(grp, 0);
    stage_own(grp);

    /* park the 8 links of every site, the directions dealt out among the groups: forward links at
     * (own parity, cb), backward links at (other parity, the backward neighbour's cb) */
    const TileLinks<TL::NT> S = {links + tid};
    {
        const GlobalLinks<float, 12> G = {A.gauge, A.gblock, Vh, A.parity};
        auto nbcb = [&](int idx) { return idx >= 0 ? tab[idx] : ~idx; };
        float u[18];
        if (0 % NG == grp) { G.template get<0, +1>(u, cb, 0); S.template put<0, +1>(u); }
        if (1 % NG == grp) { G.template get<0, -1>(u, cb, nbcb(ns.xm)); S.template put<0, -1>(u); }
        if (2 % NG == grp) { G.template get<1, +1>(u, cb, 0); S.template put<1, +1>(u); }
        if (3 % NG == grp) { G.template get<1, -1>(u, cb, nbcb(ns.ym)); S.template put<1, -1>(u); }
        if (4 % NG == grp) { G.template get<2, +1>(u, cb, 0); S.template put<2, +1>(u); }
        if (5 % NG == grp) { G.template get<2, -1>(u, cb, nbcb(ns.zm)); S.template put<2, -1>(u); }
        if (6 % NG == grp) { G.template get<3, +1>(u, cb, 0); S.template put<3, +1>(u); }
        if (7 % NG == grp) { G.template get<3, -1>(u, cb, nbcb(ns.tm)); S.template put<3, -1>(u); }
    }
    __syncthreads(); /* links parked by all groups */

    /* Per vector, in this thread's commit order: rows(j) | own(j) | rows(j + NG).  rows(j + NG) go
     * into the other row buffer at the top of iteration j, a whole iteration before they are read;
     * own(j + NG) is requested when the epilogue of j has consumed the slots, a whole hop before
     * it is read. */
    int b = 0;
    for (int j = grp; j < A.nvec; j += NG, b ^= 1) {
        const size_t off = (size_t)j * A.vstride;
        const TileSpinor<TL::CORE> src = {core0 + b * 6 * TL::CORE, reinterpret_cast<const float4*>(A.in + off), Vh};
        stage_core(j + NG, b ^ 1);
        cp_async_wait<2>(); /* rows(j) have landed (this thread's requests) */
        group_sync(1 + grp, TL::NT);
        float acc[24], zz[24];
        hop_site<float, 0>(acc, S, src, cb, ns);
        group_sync(1 + grp, TL::NT); /* the group is done with row buffer b: the next iteration may refill it */

        cp_async_wait<1>(); /* own(j) has landed */
        own_load<TL::NT, NOWN, 0>(zz, own, A.z + off, Vh, (size_t)cb);
#pragma unroll
        for (int i = 0; i < 24; i++) {
            const float g5 = (i < 12) ? 1.f : A.s5; /* gamma5 = diag(1,1,-1,-1) when s5 = -1 */
            acc[i] = A.c1 * g5 * (zz[i] + A.b * acc[i]);
        }
        if (A.c2 != 0.f) {
            own_load<TL::NT, NOWN, 1>(zz, own, A.tm + off, Vh, (size_t)cb);
#pragma unroll
            for (int i = 0; i < 24; i++) acc[i] += A.c2 * zz[i];
        }
        if (A.c3 != 0.f) {
            own_load<TL::NT, NOWN, 2>(zz, own, A.v + off, Vh, (size_t)cb);
#pragma unroll
            for (int i = 0; i < 24; i++) acc[i] += A.c3 * zz[i];
        }
        store_planes_cs<float, 24>(A.out + off, Vh, (size_t)cb, acc);
        stage_own(j + NG); /* this thread alone reads its own slots: no barrier needed */
    }
    cp_async_wait<0>();
}

template <typename TL> bool tile_fits(const DevGeom& g)
{
    return g.X2 % TL::WX == 0 && g.Y % TL::WY == 0 && g.Z % TL::WZ == 0 && g.T % TL::WT == 0;
}

template <typename TL, int NG, int NOWN> cudaError_t launch_tile(const HopArgs<float>& A, cudaStream_t st)
{
    const DevGeom& g = A.geo;
    const int nbx = g.X2 / TL::WX, nby = g.Y / TL::WY, nbz = g.Z / TL::WZ, nbt = g.T / TL::WT;
    int tgroup = 1;
    for (int tg = 4; tg > 1; tg >>= 1)
        if (nbt % tg == 0 && nbt > tg) { tgroup = tg; break; }
    cudaError_t e = cudaFuncSetAttribute(hop_mrhs_tile_kernel<TL, NG, NOWN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TL::smem(NG, NOWN));
    if (e != cudaSuccess) return e;
    hop_mrhs_tile_kernel<TL, NG, NOWN><<<nbx * nby * nbz * nbt, TL::NT * NG, TL::smem(NG, NOWN), st>>>(A, nbx, nby, nbz, tgroup);
    return cudaGetLastError();
}

} // namespace

/* Runs the multi-rhs Chebyshev / Wilson step with the tiled kernel when it is asked for and applies
 * (fp32, 12-real links, more than one vector, extents divisible by a tile shape); *handled = false
 * otherwise and the caller uses hop_cheb_mrhs_kernel.
 * OPT-IN (QCD_MRHS_TILE=1): measured on B200 at 48^3 x 96, 12 vectors x degree 100, this kernel moves
 * 19 % fewer bytes across the L2 -> SM fabric (46.4 against 57.1 GB per launch) but runs 1.62 - 1.74 s
 * against 1.34 s for hop_cheb_mrhs_kernel: with one 512-thread block per SM its barriers and the exposed
 * latency of whatever is not staged cost more than the traffic saves (profiles/hop_cheb_mrhs_r2.md).
 * It stays in the tree, parity-tested, as the shared-memory staging experiment north_star (2) names. */
cudaError_t hop_tile_launch_f32(const qcd_gauge* g, const HopLaunch& L, cudaStream_t st, bool* handled)
{
    *handled = false;
    if (L.mode != HOP_CHEB || L.nvec < 2 || g->reconstruct != 12) return cudaSuccess;
    const char* env = getenv("QCD_MRHS_TILE");
    if (!env || atoi(env) != 1) return cudaSuccess;
    const HopArgs<float> A = make_hop_args<float>(g, L);
    typedef Tile<8, 4, 2, 2> T8;
    typedef Tile<4, 4, 4, 2> T4;
    const char* v = getenv("QCD_MRHS_VARIANT"); /* sweep knob: "<groups><own streams staged>" */
    const int variant = v ? atoi(v) : 40;
    if (tile_fits<T8>(A.geo)) {
        *handled = true;
        switch (variant) {
        case 32: return launch_tile<T8, 3, 2>(A, st);
        case 31: return launch_tile<T8, 3, 1>(A, st);
        case 41: return launch_tile<T8, 4, 1>(A, st);
        default: return launch_tile<T8, 4, 0>(A, st);
        }
    }
    if (tile_fits<T4>(A.geo)) {
        *handled = true;
        return launch_tile<T4, 4, 0>(A, st);
    }
    return cudaSuccess;
}
