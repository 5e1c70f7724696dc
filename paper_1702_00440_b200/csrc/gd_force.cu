// gd_force.cu -- softened direct-summation acceleration + jerk (Eq. 3 P:145 and its time derivative, sign per
// fn. 11 P:188) of the listed sinks from ALL np predicted source records (step vii-c).
//
//   r = xp_j - xp_i ; w = vp_j - vp_i ; s = r.r + eps^2 ; q = s^(-1/2)
//   a_i += m_j q^3 r ;   jerk_i += m_j q^3 ( w - 3 (r.w) q^2 r )
//
// Bound: the plain FP64 pipe.  One pair = 31 FP64-pipe instructions (6 DADD, 3+3 DFMA/DMUL for s and r.w,
// 5 for the reciprocal square root refinement, 5 DMUL, 9 DFMA) + 1 MUFU.RSQ64H; counted as 60 flop by the
// convention of BASELINE.json.  Two kernels:
//
//   k_force_ipar   (large active sets)  one sink per (thread, register block); sources staged in shared memory
//                  by TMA bulk copies (cp.async.bulk + mbarrier, GD_STAGES-deep ring) and read by broadcast.
//                  Grid = i-tiles x j-splits; the j-split only exists to fill 148 SMs evenly.
//   k_force_jsplit (small active sets)  one register block of sinks per WARP, the lanes stride over the sources;
//                  partial sums are combined by warp shuffles, shared memory across the warps of a CTA, DSMEM
//                  across the CTAs of a cluster, and a fixed-order pass across clusters.
//
// Every combination order is fixed by the launch geometry, never by timing: results are run-to-run identical.
// The self pair (j == i) contributes exactly zero for eps > 0 (r = w = 0, q finite); for eps = 0 the s == 0
// case is masked to q = 0 (reading R10).  Zero-mass padding records contribute exactly zero.
#include "gd_common.cuh"
#include <cooperative_groups.h>
namespace cg = cooperative_groups;

#define GD_STAGES 2
#define GD_IPAR_THREADS 128
#define GD_JS_THREADS 256
#define GD_JS_WARPS (GD_JS_THREADS / 32)

// ---------------------------------------------------------------------------------------------------------
// q = s^(-1/2): MUFU.RSQ64H seed (relative error ~2^-21: it sees the upper 32 bits of s only) followed by one
// third-order step  y <- y + y e (1/2 + 3/8 e),  e = 1 - s y^2   (error 5/16 e^3 ~ 2^-60: below 1 ulp).
// EPS0 = true (eps == 0): s == 0 for coincident particles and the self pair, masked to q = 0.  With eps > 0, s >= eps^2
// is a normal number and the mask is compiled out (the host picks EPS0 whenever eps^2 is zero or denormal).
template <bool EPS0>
__device__ __forceinline__ double gd_rsqrt(double s)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(s));
    if (EPS0) {
        if (__double2hiint(s) == 0) y = 0.0;                     // contribute nothing instead of inf * 0
    }
    double t = s * y;
    double e = fma(-t, y, 1.0);
    double p = fma(0.375, e, 0.5);
    double g = y * e;
    return fma(g, p, y);
}

struct gd_src { double x, y, z, m, vx, vy, vz; };
struct gd_acc { double ax, ay, az, jx, jy, jz; };

template <bool EPS0>
__device__ __forceinline__ void gd_pair(const gd_src &i, const gd_src &j, double eps2, gd_acc &o)
{
    double rx = j.x - i.x, ry = j.y - i.y, rz = j.z - i.z;
    double wx = j.vx - i.vx, wy = j.vy - i.vy, wz = j.vz - i.vz;
    double s = fma(rx, rx, fma(ry, ry, fma(rz, rz, eps2)));
    double rw = fma(rx, wx, fma(ry, wy, rz * wz));
    double q = gd_rsqrt<EPS0>(s);
    double q2 = q * q;
    double mq3 = (j.m * q) * q2;
    double b3 = -3.0 * (rw * q2);
    o.ax = fma(mq3, rx, o.ax);
    o.ay = fma(mq3, ry, o.ay);
    o.az = fma(mq3, rz, o.az);
    o.jx = fma(mq3, fma(b3, rx, wx), o.jx);
    o.jy = fma(mq3, fma(b3, ry, wy), o.jy);
    o.jz = fma(mq3, fma(b3, rz, wz), o.jz);
}

__device__ __forceinline__ gd_src gd_load_sink(const gd_dev &d, int32_t i)
{
    double2 xy = __ldg(d.pxy + i), zm = __ldg(d.pzm + i), vxy = __ldg(d.vxy + i);
    double vz = __ldg(d.vz + i);
    return gd_src{xy.x, xy.y, zm.x, zm.y, vxy.x, vxy.y, vz};
}

// ---- mbarrier / TMA bulk-copy primitives (PTX; SASS: SYNCS.*, UBLKCP) ---------------------------------
__device__ __forceinline__ uint32_t gd_smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void gd_mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(gd_smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void gd_mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(gd_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void gd_mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(gd_smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void gd_bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     gd_smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(gd_smem_u32(bar))
                 : "memory");
}

// One shared-memory stage: the four SoA planes of GD_TILE_J consecutive source records (14 KB).
struct __align__(128) gd_tile {
    double2 pxy[GD_TILE_J];
    double2 pzm[GD_TILE_J];
    double2 vxy[GD_TILE_J];
    double vz[GD_TILE_J];
};

// cnt records starting at j0 (both multiples of GD_UNIT_J: every copy is 16-byte aligned and a multiple of 16 bytes)
__device__ __forceinline__ void gd_issue_tile(gd_tile *st, uint64_t *bar, const gd_dev &d, int64_t j0, int cnt)
{
    const uint32_t c = (uint32_t)cnt;
    gd_mbar_expect_tx(bar, c * 56u);
    gd_bulk_g2s(st->pxy, d.pxy + j0, c * 16u, bar);
    gd_bulk_g2s(st->pzm, d.pzm + j0, c * 16u, bar);
    gd_bulk_g2s(st->vxy, d.vxy + j0, c * 16u, bar);
    gd_bulk_g2s(st->vz, d.vz + j0, c * 8u, bar);
}

// ---------------------------------------------------------------------------------------------------------
// i-parallel kernel.  CTA = 4 warps arranged as WI x WJ (WI * WJ = 4).  The CTA owns an i-tile of TI = 32 * BI * WI
// sinks (sink k = tile0 + (b * WI + wi) * 32 + lane: coalesced output) and the source range of its j-split
// (blockIdx.y), given in units of GD_UNIT_J records.  The range is streamed through a GD_STAGES-deep ring of
// shared-memory stages of up to GD_TILE_J records, filled by TMA bulk copies that one elected thread issues;
// the WJ warps of one sink group each take a contiguous 1/WJ of every stage and are combined in shared memory
// in wj order.  n_split == 1 writes a_out / j_out directly; otherwise partial[split][k][6], and the LAST CTA of
// an i-tile to arrive (ticket) sums the splits in split order -- the order is fixed, whoever does it.
template <int BI, int WJ, bool EPS0>
__global__ void __launch_bounds__(GD_IPAR_THREADS, (BI == 1 ? 8 : (BI == 2 ? 5 : 2)))
k_force_ipar(gd_dev d, const int32_t *__restrict__ idx, int n_act, int n_units, int units_per_split, int n_split,
             double eps2, double *__restrict__ a_out, double *__restrict__ j_out)
{
    constexpr int WI = 4 / WJ;
    constexpr int TI = 32 * BI * WI;
    __shared__ gd_tile tile[GD_STAGES];
    __shared__ __align__(8) uint64_t full[GD_STAGES];
    __shared__ double red[(WJ > 1 ? (WJ - 1) * WI * BI * 6 * 32 : 1)];
    __shared__ bool s_last;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wi = warp % WI, wj = warp / WI;
    const int split = blockIdx.y;
    const int j_begin = split * units_per_split * GD_UNIT_J;
    const int j_end = min(n_units, (split + 1) * units_per_split) * GD_UNIT_J;
    const int my_tiles = (j_end - j_begin + GD_TILE_J - 1) / GD_TILE_J;

    if (tid == 0) {
        for (int s = 0; s < GD_STAGES; ++s) gd_mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
        for (int s = 0; s < GD_STAGES && s < my_tiles; ++s) {
            int j0 = j_begin + s * GD_TILE_J;
            gd_issue_tile(&tile[s], &full[s], d, j0, min(GD_TILE_J, j_end - j0));
        }
    }

    gd_src si[BI];
    gd_acc acc[BI];
    const int k0 = blockIdx.x * TI + wi * 32 + lane;
#pragma unroll
    for (int b = 0; b < BI; ++b) {
        int k = min(k0 + b * (32 * WI), n_act - 1);                // tail lanes recompute the last sink, never store
        int32_t i = idx ? __ldg(idx + k) : k;
        si[b] = gd_load_sink(d, i);
        acc[b] = gd_acc{0, 0, 0, 0, 0, 0};
    }

    for (int t = 0; t < my_tiles; ++t) {
        const int s = t % GD_STAGES;
        const int cnt = min(GD_TILE_J, j_end - (j_begin + t * GD_TILE_J));   // multiple of GD_UNIT_J
        gd_mbar_wait(&full[s], (uint32_t)((t / GD_STAGES) & 1));
        const gd_tile &T = tile[s];
        const int per = cnt / WJ;
        const int jb = wj * per, je = jb + per;
#pragma unroll 2
        for (int jj = jb; jj < je; ++jj) {
            double2 xy = T.pxy[jj], zm = T.pzm[jj], vxy = T.vxy[jj];
            gd_src sj{xy.x, xy.y, zm.x, zm.y, vxy.x, vxy.y, T.vz[jj]};
#pragma unroll
            for (int b = 0; b < BI; ++b) gd_pair<EPS0>(si[b], sj, eps2, acc[b]);
        }
        __syncthreads();                                         // every warp is done with stage s
        if (tid == 0 && t + GD_STAGES < my_tiles) {
            int j0 = j_begin + (t + GD_STAGES) * GD_TILE_J;
            gd_issue_tile(&tile[s], &full[s], d, j0, min(GD_TILE_J, j_end - j0));
        }
    }

    // warps wj = 1..WJ-1 of a sink group -> warp wj = 0, in wj order
    if (WJ > 1) {
        if (wj > 0) {
#pragma unroll
            for (int b = 0; b < BI; ++b) {
                double *r = red + ((((wj - 1) * WI + wi) * BI + b) * 6) * 32 + lane;
                r[0] = acc[b].ax; r[32] = acc[b].ay; r[64] = acc[b].az;
                r[96] = acc[b].jx; r[128] = acc[b].jy; r[160] = acc[b].jz;
            }
        }
        __syncthreads();
        if (wj == 0) {
#pragma unroll
            for (int p = 1; p < WJ; ++p) {
#pragma unroll
                for (int b = 0; b < BI; ++b) {
                    const double *r = red + ((((p - 1) * WI + wi) * BI + b) * 6) * 32 + lane;
                    acc[b].ax += r[0]; acc[b].ay += r[32]; acc[b].az += r[64];
                    acc[b].jx += r[96]; acc[b].jy += r[128]; acc[b].jz += r[160];
                }
            }
        }
    }

    if (wj == 0) {
#pragma unroll
        for (int b = 0; b < BI; ++b) {
            int k = k0 + b * (32 * WI);
            if (k >= n_act) continue;
            if (n_split == 1) {
                a_out[3 * (int64_t)k + 0] = acc[b].ax; a_out[3 * (int64_t)k + 1] = acc[b].ay; a_out[3 * (int64_t)k + 2] = acc[b].az;
                j_out[3 * (int64_t)k + 0] = acc[b].jx; j_out[3 * (int64_t)k + 1] = acc[b].jy; j_out[3 * (int64_t)k + 2] = acc[b].jz;
            } else {
                double2 *p = reinterpret_cast<double2 *>(d.partial + ((int64_t)split * n_act + k) * 6);
                __stcg(p + 0, make_double2(acc[b].ax, acc[b].ay));
                __stcg(p + 1, make_double2(acc[b].az, acc[b].jx));
                __stcg(p + 2, make_double2(acc[b].jy, acc[b].jz));
            }
        }
    }
    if (n_split == 1) return;

    // the last CTA of this i-tile folds the splits, in split order
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        unsigned int tk = atomicAdd(&d.tile_ticket[blockIdx.x], 1u);
        s_last = (tk == (unsigned int)n_split - 1u);
        if (s_last) d.tile_ticket[blockIdx.x] = 0u;              // every CTA of the tile has arrived: re-arm
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    const int kt0 = blockIdx.x * TI;
    const int rows = min(TI, n_act - kt0);
    for (int e = tid; e < rows * 6; e += GD_IPAR_THREADS) {
        const double *p = d.partial + (int64_t)kt0 * 6 + e;
        double s = 0.0;
#pragma unroll 8
        for (int q = 0; q < n_split; ++q) s += __ldcg(p + (int64_t)q * n_act * 6);
        int k = kt0 + e / 6, comp = e % 6;
        double *o = comp < 3 ? a_out : j_out;
        o[3 * (int64_t)k + comp % 3] = s;
    }
}

// ---------------------------------------------------------------------------------------------------------
// j-split kernel (small active sets: too few sinks to fill the machine with i-tiles).  CTA = 8 warps that ALL own
// the same i-tile of TI = 32 * BI sinks (sink k = tile0 + b * 32 + lane) and split the CTA's source range between
// them: the range is streamed through the same TMA-filled shared-memory stages as above and every warp takes a
// contiguous 1/8 of each stage.  blockIdx.x = source chunk, blockIdx.y = i-tile; a cluster is cdim consecutive
// CTAs along x (same sinks, neighbouring chunks).  Reduction, every level in a fixed order:
//   8 warps -> CTA (shared memory, warp order) -> cluster (DSMEM, rank order, by rank 0)
//   -> clusters (global partials; the last cluster of an i-tile to arrive folds them in cluster order).
template <int BI, bool EPS0>
__global__ void __launch_bounds__(GD_JS_THREADS, 2)
k_force_jsplit(gd_dev d, const int32_t *__restrict__ idx, int n_act, int n_units, int units_per_cta, int cdim,
               double eps2, double *__restrict__ a_out, double *__restrict__ j_out)
{
    constexpr int TI = 32 * BI;
    constexpr int NE = TI * 6;                                     // sums per i-tile; element e = (b * 6 + c) * 32 + lane
    __shared__ gd_tile tile[GD_STAGES];
    __shared__ __align__(8) uint64_t full[GD_STAGES];
    __shared__ double cta[NE];
    static_assert(sizeof(double) * GD_JS_WARPS * NE <= sizeof(gd_tile) * GD_STAGES, "warp sums reuse the stage memory");
    __shared__ bool s_last;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int j_begin = min(n_units, (int)blockIdx.x * units_per_cta) * GD_UNIT_J;
    const int j_end = min(n_units, ((int)blockIdx.x + 1) * units_per_cta) * GD_UNIT_J;
    const int my_tiles = (j_end - j_begin + GD_TILE_J - 1) / GD_TILE_J;     // 0 for the padding CTAs of the last cluster

    if (tid == 0) {
        for (int s = 0; s < GD_STAGES; ++s) gd_mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
        for (int s = 0; s < GD_STAGES && s < my_tiles; ++s) {
            int j0 = j_begin + s * GD_TILE_J;
            gd_issue_tile(&tile[s], &full[s], d, j0, min(GD_TILE_J, j_end - j0));
        }
    }

    gd_src si[BI];
    gd_acc acc[BI];
    const int k0 = blockIdx.y * TI + lane;
#pragma unroll
    for (int b = 0; b < BI; ++b) {
        int k = min(k0 + b * 32, n_act - 1);
        int32_t i = idx ? __ldg(idx + k) : k;
        si[b] = gd_load_sink(d, i);
        acc[b] = gd_acc{0, 0, 0, 0, 0, 0};
    }

    for (int t = 0; t < my_tiles; ++t) {
        const int s = t % GD_STAGES;
        const int cnt = min(GD_TILE_J, j_end - (j_begin + t * GD_TILE_J));   // multiple of GD_UNIT_J = 8 per warp
        gd_mbar_wait(&full[s], (uint32_t)((t / GD_STAGES) & 1));
        const gd_tile &T = tile[s];
        const int per = cnt / GD_JS_WARPS;
        const int jb = warp * per, je = jb + per;
#pragma unroll 2
        for (int jj = jb; jj < je; ++jj) {
            double2 xy = T.pxy[jj], zm = T.pzm[jj], vxy = T.vxy[jj];
            gd_src sj{xy.x, xy.y, zm.x, zm.y, vxy.x, vxy.y, T.vz[jj]};
#pragma unroll
            for (int b = 0; b < BI; ++b) gd_pair<EPS0>(si[b], sj, eps2, acc[b]);
        }
        if (t + GD_STAGES < my_tiles) {
            __syncthreads();                                     // every warp is done with stage s
            if (tid == 0) {
                int j0 = j_begin + (t + GD_STAGES) * GD_TILE_J;
                gd_issue_tile(&tile[s], &full[s], d, j0, min(GD_TILE_J, j_end - j0));
            }
        }
    }

    // 8 warps -> CTA, in warp order (the warp sums reuse the stage memory once every warp has left the source loop)
    __syncthreads();
    double *red = reinterpret_cast<double *>(tile);
#pragma unroll
    for (int b = 0; b < BI; ++b) {
        double *r = red + warp * NE + b * 192 + lane;
        r[0] = acc[b].ax; r[32] = acc[b].ay; r[64] = acc[b].az;
        r[96] = acc[b].jx; r[128] = acc[b].jy; r[160] = acc[b].jz;
    }
    __syncthreads();
    for (int e = tid; e < NE; e += GD_JS_THREADS) {
        double s = red[e];
#pragma unroll
        for (int w = 1; w < GD_JS_WARPS; ++w) s += red[w * NE + e];
        cta[e] = s;
    }
    cg::cluster_group cluster = cg::this_cluster();
    if (cdim > 1) cluster.sync(); else __syncthreads();
    const unsigned rank = (cdim > 1) ? cluster.block_rank() : 0;
    const int n_clusters = gridDim.x / cdim;
    const int cl = blockIdx.x / cdim;
    if (rank == 0) {
        for (int e = tid; e < NE; e += GD_JS_THREADS) {
            double s = cta[e];
            for (int r = 1; r < cdim; ++r) s += cluster.map_shared_rank(cta, r)[e];     // DSMEM read of CTA r's sums
            int k = blockIdx.y * TI + (e / 192) * 32 + (e & 31), comp = (e >> 5) % 6;
            if (k < n_act) {
                if (n_clusters == 1) {
                    double *o = comp < 3 ? a_out : j_out;
                    o[3 * (int64_t)k + comp % 3] = s;
                } else {
                    __stcg(d.partial + ((int64_t)cl * n_act + k) * 6 + comp, s);
                }
            }
        }
    }
    if (n_clusters > 1 && rank == 0) {
        // the last cluster of this i-tile folds the clusters, in cluster order
        __threadfence();
        __syncthreads();
        if (tid == 0) {
            unsigned int tk = atomicAdd(&d.tile_ticket[blockIdx.y], 1u);
            s_last = (tk == (unsigned int)n_clusters - 1u);
            if (s_last) d.tile_ticket[blockIdx.y] = 0u;
        }
        __syncthreads();
        if (s_last) {
            __threadfence();
            for (int e = tid; e < NE; e += GD_JS_THREADS) {
                int k = blockIdx.y * TI + (e / 192) * 32 + (e & 31), comp = (e >> 5) % 6;
                if (k >= n_act) continue;
                const double *p = d.partial + (int64_t)k * 6 + comp;
                double s = 0.0;
#pragma unroll 8
                for (int q = 0; q < n_clusters; ++q) s += __ldcg(p + (int64_t)q * n_act * 6);
                double *o = comp < 3 ? a_out : j_out;
                o[3 * (int64_t)k + comp % 3] = s;
            }
        }
    }
    if (cdim > 1) cluster.sync();                   // keep every CTA's shared memory alive until rank 0 has read it
}

// ---------------------------------------------------------------------------------------------------------
// Host side: launch geometry.

// i-parallel variants, largest i-tile first: {BI, WJ} -> TI = 32 * BI * (4 / WJ)
struct gd_ipar_variant { int bi, wj, ti, resident; };
static gd_ipar_variant g_ipar[] = {{2, 1, 256, 0}, {1, 1, 128, 0}, {1, 2, 64, 0}, {1, 4, 32, 0}};
#define GD_IPAR_NVAR 4

template <int BI, int WJ>
static cudaError_t gd_launch_ipar(gd_ctx *c, dim3 grid, const int32_t *idx, int n_act, int n_units, int ups, int n_split,
                                  double *a_out, double *j_out)
{
    if (c->eps2 < 2.3e-308)
        k_force_ipar<BI, WJ, true><<<grid, GD_IPAR_THREADS, 0, c->stream>>>(c->d, idx, n_act, n_units, ups, n_split, c->eps2, a_out, j_out);
    else
        k_force_ipar<BI, WJ, false><<<grid, GD_IPAR_THREADS, 0, c->stream>>>(c->d, idx, n_act, n_units, ups, n_split, c->eps2, a_out, j_out);
    return cudaGetLastError();
}

static int gd_ipar_resident(int v)
{
    int r = 0;
    cudaError_t e = cudaSuccess;
    switch (v) {
    case 0: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&r, k_force_ipar<2, 1, false>, GD_IPAR_THREADS, 0); break;
    case 1: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&r, k_force_ipar<1, 1, false>, GD_IPAR_THREADS, 0); break;
    case 2: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&r, k_force_ipar<1, 2, false>, GD_IPAR_THREADS, 0); break;
    default: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&r, k_force_ipar<1, 4, false>, GD_IPAR_THREADS, 0); break;
    }
    return (e == cudaSuccess && r > 0) ? r : 1;
}

// Cost model of one launch, in source units per SM: CTAs are dealt round-robin to the SMs, an SM's time is the
// work of the CTAs it gets (the FP64 pipe is shared) plus a fixed cost per CTA, stretched when it holds too few
// warps to cover the FP64 latency.
static double gd_ipar_cost(int64_t i_tiles, int n_units, int s, int sms, int resident, int bi)
{
    const double fixed_units = 1.5;                              // CTA start-up + first TMA round trip, in units of 64 sources
    int64_t ctas = i_tiles * s;
    int64_t per_sm = (ctas + sms - 1) / sms;
    int ups = (n_units + s - 1) / s;
    double conc = (double)(per_sm < resident ? per_sm : resident);
    double chains = conc * 4.0 * bi;                             // independent pair chains per SM
    double eff = chains >= 24.0 ? 1.0 : chains / 24.0;
    return (double)per_sm * (ups + fixed_units) * bi / eff;
}

static int gd_force_ipar(gd_ctx *c, const int32_t *idx, int64_t n_act, double *a_out, double *j_out)
{
    const int n_units = (int)(c->np / GD_UNIT_J);
    int v = c->ipar_variant;
    if (v < 0 || v >= GD_IPAR_NVAR) {
        // the largest i-tile that still yields enough CTAs to occupy every SM
        for (v = 0; v < GD_IPAR_NVAR - 1; ++v) {
            int64_t i_tiles = (n_act + g_ipar[v].ti - 1) / g_ipar[v].ti;
            int64_t s_cap = n_units / 2 > 0 ? n_units / 2 : 1;
            if (i_tiles * s_cap >= 4 * (int64_t)c->sm_count) break;
        }
    }
    gd_ipar_variant &V = g_ipar[v];
    if (!V.resident) V.resident = gd_ipar_resident(v);
    const int64_t i_tiles = (n_act + V.ti - 1) / V.ti;
    int64_t s_max = c->pcap / n_act;
    if (s_max > n_units) s_max = n_units;
    if (s_max > 1024) s_max = 1024;
    if (s_max < 1) s_max = 1;
    int n_split = 1;
    if (c->ipar_split > 0) {
        n_split = (int)(c->ipar_split < s_max ? c->ipar_split : s_max);
    } else {
        double best = 1e300;
        for (int s = 1; s <= s_max; ++s) {
            double cost = gd_ipar_cost(i_tiles, n_units, s, c->sm_count, V.resident, V.bi);
            if (cost < best * (1.0 - 1e-9)) { best = cost; n_split = s; }
        }
    }
    int ups = (n_units + n_split - 1) / n_split;
    n_split = (n_units + ups - 1) / ups;
    dim3 grid((unsigned)i_tiles, (unsigned)n_split);
    cudaError_t e;
    switch (v) {
    case 0: e = gd_launch_ipar<2, 1>(c, grid, idx, (int)n_act, n_units, ups, n_split, a_out, j_out); break;
    case 1: e = gd_launch_ipar<1, 1>(c, grid, idx, (int)n_act, n_units, ups, n_split, a_out, j_out); break;
    case 2: e = gd_launch_ipar<1, 2>(c, grid, idx, (int)n_act, n_units, ups, n_split, a_out, j_out); break;
    default: e = gd_launch_ipar<1, 4>(c, grid, idx, (int)n_act, n_units, ups, n_split, a_out, j_out); break;
    }
    if (e != cudaSuccess) return gd_fail_cuda(c, e, "k_force_ipar");
    c->launches += 1;
    c->last_force_kernel = 1;
    c->last_geom[0] = v; c->last_geom[1] = (int)i_tiles; c->last_geom[2] = n_split; c->last_geom[3] = ups;
    return 0;
}

template <int BI>
static cudaError_t gd_launch_jsplit(gd_ctx *c, cudaLaunchConfig_t *cfg, const int32_t *idx, int n_act, int n_units, int upc,
                                    int cdim, double *a_out, double *j_out)
{
    if (c->eps2 < 2.3e-308)
        return cudaLaunchKernelEx(cfg, k_force_jsplit<BI, true>, c->d, idx, n_act, n_units, upc, cdim, c->eps2, a_out, j_out);
    return cudaLaunchKernelEx(cfg, k_force_jsplit<BI, false>, c->d, idx, n_act, n_units, upc, cdim, c->eps2, a_out, j_out);
}

static int gd_force_jsplit(gd_ctx *c, const int32_t *idx, int64_t n_act, double *a_out, double *j_out)
{
    const int n_units = (int)(c->np / GD_UNIT_J);
    const int bi = (c->js_bi == 1 || c->js_bi == 2) ? c->js_bi : (n_act > 4 * 32 ? 2 : 1);
    const int ti = 32 * bi;
    const int64_t i_tiles = (n_act + ti - 1) / ti;
    // source chunks per i-tile: about js_ctas_per_sm CTAs (8 warps each) per SM over the whole grid
    int64_t jc = c->ipar_split > 0 ? c->ipar_split : ((int64_t)c->js_ctas_per_sm * c->sm_count + i_tiles - 1) / i_tiles;
    if (jc > n_units) jc = n_units;
    if (jc > c->pcap / n_act) jc = c->pcap / n_act;
    if (jc < 1) jc = 1;
    int upc = (int)((n_units + jc - 1) / jc);
    jc = (n_units + upc - 1) / upc;
    int cdim = 1;
    while (cdim < 8 && cdim * 2 <= jc) cdim *= 2;
    if (c->js_cluster > 0 && c->js_cluster < cdim) cdim = c->js_cluster;
    const int64_t gx = ((jc + cdim - 1) / cdim) * cdim;          // padding CTAs of the last cluster get an empty range

    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)gx, (unsigned)i_tiles);
    cfg.blockDim = dim3(GD_JS_THREADS);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = c->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)cdim;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    cudaError_t e = (bi == 2) ? gd_launch_jsplit<2>(c, &cfg, idx, (int)n_act, n_units, upc, cdim, a_out, j_out)
                              : gd_launch_jsplit<1>(c, &cfg, idx, (int)n_act, n_units, upc, cdim, a_out, j_out);
    if (e != cudaSuccess) return gd_fail_cuda(c, e, "k_force_jsplit");
    c->launches += 1;
    c->last_force_kernel = 2;
    c->last_geom[0] = 10 * bi + cdim; c->last_geom[1] = (int)i_tiles; c->last_geom[2] = (int)gx; c->last_geom[3] = upc;
    return 0;
}

int gdk_force(gd_ctx *c, const int32_t *idx, int64_t n_act, double *a_out, double *j_out)
{
    if (n_act <= 0) return 0;
    const bool js = n_act <= c->jsplit_max_nact;
    const int slot = gd_prof_begin(c);
    int rc = js ? gd_force_jsplit(c, idx, n_act, a_out, j_out) : gd_force_ipar(c, idx, n_act, a_out, j_out);
    gd_prof_end(c, slot, js ? 1 : 0, (double)n_act * (double)c->n);
    return rc;
}
