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
#include "gd_pair.cuh"
#include <cooperative_groups.h>
#include <limits.h>
#include <stdlib.h>
namespace cg = cooperative_groups;

#define GD_STAGES 2
#define GD_IPAR_THREADS 128
// the large-set i-parallel kernel: sinks per thread, resident CTAs per SM it is compiled for (register budget), and
// the unrolling of its source loop -- tuning knobs (measured on B200: see DESIGN.md section 5)
#ifndef GD_L_BI
#define GD_L_BI 2
#endif
#ifndef GD_IPAR_L_CTAS
#define GD_IPAR_L_CTAS 3
#endif
#ifndef GD_IPAR_UNROLL
#define GD_IPAR_UNROLL 2
#endif
#define GD_PRAGMA_(x) _Pragma(#x)
#define GD_PRAGMA_UNROLL(n) GD_PRAGMA_(unroll n)
#define GD_JS_THREADS 256
#define GD_JS_WARPS (GD_JS_THREADS / 32)
#define GD_JS_CLUSTER 8
#define GD_JS_MAX_CPT 16          // clusters per i-tile: more only lengthens the fold


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
// Launch arguments common to both force kernels.  The active count comes either from the host (n_act) or from
// device memory (n_act_dev != NULL: the block-step graph, where the host never learns it); a kernel runs only
// if lo < n_act <= hi, so that the graph can enqueue every kernel and let the device pick one.
struct gd_fargs {
    const int32_t *idx;              // sink list (NULL: sink k = particle k)
    const long long *n_act_dev;
    int n_act, lo, hi;
    int n_units;                     // np / GD_UNIT_J
    const int2 *geom;                // i-parallel: [i_tiles] -> {source splits, units per split}
    double eps2;
    double *a_out, *j_out;           // [n_act,3]
};

__device__ __forceinline__ int gd_active_count(const gd_fargs &fa)
{
    return fa.n_act_dev ? (int)__ldcg(fa.n_act_dev) : fa.n_act;
}

// ---------------------------------------------------------------------------------------------------------
// i-parallel kernel.  CTA = 4 warps arranged as WI x WJ (WI * WJ = 4).  A work unit is (i-tile, source split): an
// i-tile of TI = 32 * BI * WI sinks (sink k = tile0 + (b * WI + wi) * 32 + lane: coalesced output) against the
// source range of one split, given in units of GD_UNIT_J records.  The grid is persistent (a multiple of the SM
// count); CTA c takes units c, c + gridDim.x, ...; the number of splits per i-tile count comes from a table the
// host fills at init (gd_ipar_table), so the geometry follows a device-resident n_act without a host round trip.
// A unit's range is streamed through a GD_STAGES-deep ring of shared-memory stages of up to GD_TILE_J records,
// filled by TMA bulk copies that one elected thread issues; the WJ warps of one sink group each take a contiguous
// 1/WJ of every stage and are combined in shared memory in wj order.  One split writes a_out / j_out directly;
// otherwise partial[split][k][6], and the LAST unit of an i-tile to finish (ticket) sums the splits in a fixed
// order -- whoever does it.
template <int BI, int WJ, bool EPS0>
__global__ void __launch_bounds__(GD_IPAR_THREADS, (BI == 1 ? 7 : GD_IPAR_L_CTAS))
k_force_ipar(gd_dev d, gd_fargs fa)
{
    constexpr int WI = 4 / WJ;
    constexpr int TI = 32 * BI * WI;
    constexpr int NE = TI * 6;
    constexpr bool PAR_FOLD = (NE * 4 * sizeof(double) <= sizeof(gd_tile) * GD_STAGES);
    __shared__ gd_tile tile[GD_STAGES];
    __shared__ __align__(8) uint64_t full[GD_STAGES];
    __shared__ double red[(WJ > 1 ? (WJ - 1) * WI * BI * 6 * 32 : 1)];
    __shared__ bool s_last;
    __shared__ int s_next;

    const int n_act = gd_active_count(fa);
    if (n_act <= fa.lo || n_act > fa.hi) return;
    const int i_tiles = (n_act + TI - 1) / TI;
    const int2 geom = __ldg(fa.geom + i_tiles);
    const int n_split = geom.x, units_per_split = geom.y;
    const int n_work = i_tiles * n_split;
    if ((int)blockIdx.x >= n_work) return;                       // only when n_work < gridDim.x: no dynamic hand-out then

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wi = warp % WI, wj = warp / WI;
    if (tid == 0) {
        for (int s = 0; s < GD_STAGES; ++s) gd_mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // units are handed out dynamically once every CTA has had its first one: blockIdx.x, then gridDim.x + ticket.
    // Which CTA computes a unit does not affect the result (a unit's partial sums go to a fixed slot).
    const bool dynamic = n_work > (int)gridDim.x;
    uint32_t it = 0;                                             // stages consumed so far: ring position and parity
    int u = blockIdx.x;
    while (u < n_work) {
        const int i_tile = u / n_split, split = u - i_tile * n_split;
        const int j_begin = split * units_per_split * GD_UNIT_J;
        const int j_end = min(fa.n_units, (split + 1) * units_per_split) * GD_UNIT_J;
        const int my_tiles = (j_end - j_begin + GD_TILE_J - 1) / GD_TILE_J;
        if (tid == 0) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the stages may have held fold scratch
            for (int s = 0; s < GD_STAGES && s < my_tiles; ++s) {
                int j0 = j_begin + s * GD_TILE_J;
                uint32_t st = (it + s) % GD_STAGES;
                gd_issue_tile(&tile[st], &full[st], d, j0, min(GD_TILE_J, j_end - j0));
            }
        }

        gd_src si[BI];
        gd_acc acc[BI];
        const int k0 = i_tile * TI + wi * 32 + lane;
#pragma unroll
        for (int b = 0; b < BI; ++b) {
            int k = min(k0 + b * (32 * WI), n_act - 1);            // tail lanes recompute the last sink, never store
            int32_t i = fa.idx ? __ldg(fa.idx + k) : k;
            si[b] = gd_load_sink(d, i);
            acc[b] = gd_acc{0, 0, 0, 0, 0, 0};
        }

        for (int t = 0; t < my_tiles; ++t, ++it) {
            const uint32_t s = it % GD_STAGES;
            const int cnt = min(GD_TILE_J, j_end - (j_begin + t * GD_TILE_J));   // multiple of GD_UNIT_J
            gd_mbar_wait(&full[s], (it / GD_STAGES) & 1u);
            const gd_tile &T = tile[s];
            const int per = cnt / WJ;
            const int jb = wj * per, je = jb + per;
            GD_PRAGMA_UNROLL(GD_IPAR_UNROLL)
            for (int jj = jb; jj < je; ++jj) {
                double2 xy = T.pxy[jj], zm = T.pzm[jj], vxy = T.vxy[jj];
                gd_src sj{xy.x, xy.y, zm.x, zm.y, vxy.x, vxy.y, T.vz[jj]};
#pragma unroll
                for (int b = 0; b < BI; ++b) gd_pair<EPS0>(si[b], sj, fa.eps2, acc[b]);
            }
            __syncthreads();                                     // every warp is done with stage s
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
                    double *a = fa.a_out + 3 * (int64_t)k, *j = fa.j_out + 3 * (int64_t)k;
                    a[0] = acc[b].ax; a[1] = acc[b].ay; a[2] = acc[b].az;
                    j[0] = acc[b].jx; j[1] = acc[b].jy; j[2] = acc[b].jz;
                } else {
                    double2 *p = reinterpret_cast<double2 *>(d.partial + ((int64_t)split * n_act + k) * 6);
                    __stcg(p + 0, make_double2(acc[b].ax, acc[b].ay));
                    __stcg(p + 1, make_double2(acc[b].az, acc[b].jx));
                    __stcg(p + 2, make_double2(acc[b].jy, acc[b].jz));
                }
            }
        }
        // the last unit of this i-tile to finish folds the splits; the same barrier hands out the next unit
        if (n_split > 1) __threadfence();
        __syncthreads();
        if (tid == 0) {
            s_last = false;
            if (n_split > 1) {
                unsigned int tk = atomicAdd(&d.tile_ticket[i_tile], 1u);
                s_last = (tk == (unsigned int)n_split - 1u);
                if (s_last) d.tile_ticket[i_tile] = 0u;          // every unit of the tile has arrived: re-arm
            }
            s_next = dynamic ? (int)gridDim.x + (int)atomicAdd(&d.work[0], 1u) : n_work;
        }
        __syncthreads();
        u = s_next;
        if (s_last) {
            __threadfence();
            const int kt0 = i_tile * TI;
            const int ne = min(TI, n_act - kt0) * 6;             // the tile's sums are contiguous in every split's rows
            const double *p0 = d.partial + (int64_t)kt0 * 6;
            const int64_t stride = (int64_t)n_act * 6;
            if (PAR_FOLD) {
                // warp g sums the splits [g * qn, (g + 1) * qn) in order; the four warp sums are added in warp order
                double *fold = reinterpret_cast<double *>(tile);
                const int qn = (n_split + 3) / 4;
                const int qb = min(n_split, warp * qn), qe = min(n_split, qb + qn);
                for (int e = lane; e < ne; e += 32) {
                    double s = 0.0;
#pragma unroll 8
                    for (int q = qb; q < qe; ++q) s += __ldcg(p0 + q * stride + e);
                    fold[warp * NE + e] = s;
                }
                __syncthreads();
                for (int e = tid; e < ne; e += GD_IPAR_THREADS) {
                    double s = ((fold[e] + fold[NE + e]) + fold[2 * NE + e]) + fold[3 * NE + e];
                    int k = kt0 + e / 6, comp = e % 6;
                    double *o = comp < 3 ? fa.a_out : fa.j_out;
                    o[3 * (int64_t)k + comp % 3] = s;
                }
            } else {
                for (int e = tid; e < ne; e += GD_IPAR_THREADS) {
                    double s = 0.0;
#pragma unroll 8
                    for (int q = 0; q < n_split; ++q) s += __ldcg(p0 + q * stride + e);
                    int k = kt0 + e / 6, comp = e % 6;
                    double *o = comp < 3 ? fa.a_out : fa.j_out;
                    o[3 * (int64_t)k + comp % 3] = s;
                }
            }
        }
        __syncthreads();                                         // s_last, s_next and the fold scratch are reused by the next unit
    }
    // the last CTA to run out of units re-arms the work counter for the next launch
    if (dynamic && tid == 0) {
        unsigned int done = atomicAdd(&d.work[1], 1u);
        if (done == gridDim.x - 1) { d.work[0] = 0u; d.work[1] = 0u; __threadfence(); }
    }
}

// ---------------------------------------------------------------------------------------------------------
// j-split kernel (small active sets: too few sinks to fill the machine with i-tiles).  CTA = 8 warps that ALL own
// the same i-tile of 32 sinks (sink k = tile0 + lane) and split the CTA's source range between them: the range
// is streamed through the same TMA-filled shared-memory stages as above and every warp takes a contiguous 1/8
// of each stage.  The grid is one row of clusters of GD_JS_CLUSTER CTAs, sized from the SM count; with
// cpt = clusters / i_tiles clusters per i-tile (computed on the device from n_act), cluster c owns i-tile c / cpt
// and the (c % cpt)-th part of the sources, of which its CTAs take consecutive chunks.  Reduction, every level
// in a fixed order:
//   8 warps -> CTA (shared memory, warp order) -> cluster (DSMEM, rank order, by rank 0)
//   -> clusters of the i-tile (global partials; the last cluster to arrive folds them in cluster order).
template <bool EPS0>
__global__ void __launch_bounds__(GD_JS_THREADS, 2)
k_force_jsplit(gd_dev d, gd_fargs fa)
{
    constexpr int NE = 32 * 6;                                     // sums per i-tile; element e = c * 32 + lane
    __shared__ gd_tile tile[GD_STAGES];
    __shared__ __align__(8) uint64_t full[GD_STAGES];
    __shared__ double cta[NE];
    __shared__ bool s_last;
    static_assert(sizeof(double) * GD_JS_WARPS * NE <= sizeof(gd_tile) * GD_STAGES, "warp sums reuse the stage memory");

    const int n_act = gd_active_count(fa);
    if (n_act <= fa.lo || n_act > fa.hi) return;
    cg::cluster_group cluster = cg::this_cluster();
    const int cdim = (int)cluster.num_blocks();
    const int rank = (int)cluster.block_rank();
    const int n_clusters = gridDim.x / cdim;
    const int i_tiles = (n_act + 31) / 32;                         // <= n_clusters (the host bounds hi)
    int cpt = n_clusters / i_tiles;                                // clusters per i-tile
    cpt = max(1, min(min(cpt, GD_JS_MAX_CPT), fa.n_units / cdim)); // at least one unit per CTA where the sources allow it; bounded fold
    const int c = blockIdx.x / cdim;
    const int i_tile = c / cpt, part = c - i_tile * cpt;
    if (i_tile >= i_tiles) return;                                 // whole clusters leave together
    const int chunks = cpt * cdim;
    const int upc = (fa.n_units + chunks - 1) / chunks;            // units per CTA
    const int chunk = part * cdim + rank;
    const int j_begin = min(fa.n_units, chunk * upc) * GD_UNIT_J;
    const int j_end = min(fa.n_units, (chunk + 1) * upc) * GD_UNIT_J;
    const int my_tiles = (j_end - j_begin + GD_TILE_J - 1) / GD_TILE_J;     // 0 if the sources ran out before this chunk

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
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

    const int k0 = i_tile * 32 + lane;
    gd_src si;
    gd_acc acc = gd_acc{0, 0, 0, 0, 0, 0};
    {
        int k = min(k0, n_act - 1);
        int32_t i = fa.idx ? __ldg(fa.idx + k) : k;
        si = gd_load_sink(d, i);
    }

    for (int t = 0; t < my_tiles; ++t) {
        const int s = t % GD_STAGES;
        const int cnt = min(GD_TILE_J, j_end - (j_begin + t * GD_TILE_J));   // multiple of GD_UNIT_J = 8 per warp
        gd_mbar_wait(&full[s], (uint32_t)((t / GD_STAGES) & 1));
        const gd_tile &T = tile[s];
        const int per = cnt / GD_JS_WARPS;
        const int jb = warp * per, je = jb + per;
#pragma unroll 4
        for (int jj = jb; jj < je; ++jj) {
            double2 xy = T.pxy[jj], zm = T.pzm[jj], vxy = T.vxy[jj];
            gd_src sj{xy.x, xy.y, zm.x, zm.y, vxy.x, vxy.y, T.vz[jj]};
            gd_pair<EPS0>(si, sj, fa.eps2, acc);
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
    {
        double *r = red + warp * NE + lane;
        r[0] = acc.ax; r[32] = acc.ay; r[64] = acc.az;
        r[96] = acc.jx; r[128] = acc.jy; r[160] = acc.jz;
    }
    __syncthreads();
    if (tid < NE) {
        double s = red[tid];
#pragma unroll
        for (int w = 1; w < GD_JS_WARPS; ++w) s += red[w * NE + tid];
        cta[tid] = s;
    }
    cluster.sync();
    if (rank == 0) {
        const int comp = tid >> 5, k = k0;                       // threads 0..191: element (comp, lane)
        const bool mine = tid < NE && k < n_act;
        double s = 0.0;
        if (tid < NE) {
            s = cta[tid];
            for (int r = 1; r < cdim; ++r) s += cluster.map_shared_rank(cta, r)[tid];   // DSMEM read of CTA r's sums
        }
        if (cpt == 1) {
            if (mine) (comp < 3 ? fa.a_out : fa.j_out)[3 * (int64_t)k + comp % 3] = s;
        } else {
            if (mine) __stcg(d.partial + ((int64_t)part * n_act + k) * 6 + comp, s);
            // the last cluster of this i-tile to arrive folds the clusters, in cluster order
            __threadfence();
            __syncthreads();
            if (tid == 0) {
                unsigned int tk = atomicAdd(&d.tile_ticket[i_tile], 1u);
                s_last = (tk == (unsigned int)cpt - 1u);
                if (s_last) d.tile_ticket[i_tile] = 0u;
            }
            __syncthreads();
            if (s_last) {
                // warp w sums the clusters w, w + 8, ... in order (all loads in flight at once); then the eight
                // warp sums are added in warp order
                __threadfence();
                const int ne = min(32, n_act - i_tile * 32) * 6;    // the tile's sums are contiguous in every part's rows
                const double *p0 = d.partial + (int64_t)i_tile * 32 * 6;
                const int64_t stride = (int64_t)n_act * 6;
                for (int e = lane; e < ne; e += 32) {
                    double f = 0.0;
#pragma unroll 5
                    for (int q = warp; q < cpt; q += GD_JS_WARPS) f += __ldcg(p0 + q * stride + e);
                    red[warp * NE + e] = f;
                }
                __syncthreads();
                if (tid < ne) {
                    double f = red[tid];
#pragma unroll
                    for (int w = 1; w < GD_JS_WARPS; ++w) f += red[w * NE + tid];
                    int kk = i_tile * 32 + tid / 6, cc = tid % 6;
                    (cc < 3 ? fa.a_out : fa.j_out)[3 * (int64_t)kk + cc % 3] = f;
                }
            }
        }
    }
    cluster.sync();                                  // keep every CTA's shared memory alive until rank 0 has read it
}

// ---------------------------------------------------------------------------------------------------------
// Host side.  Three launch shapes, all independent of n_act (so they can sit in a captured graph):
//   j-split        n_act <= js_hi                  one row of js_clusters clusters of GD_JS_CLUSTER CTAs
//   i-parallel S   js_hi < n_act <= ipar_s_hi      k_force_ipar<1, 4> (i-tile of 32 sinks), persistent grid
//   i-parallel L   ipar_s_hi < n_act               k_force_ipar<2, 1> (i-tile of 256 sinks), persistent grid
#define GD_TI_S 32
#define GD_TI_L (128 * GD_L_BI)

// Cost of covering i_tiles i-tiles with s source splits, in SM cycles: work units are dealt evenly to the SMs, an
// SM's FP64 pipe (64 lanes) is shared by the units it holds, a unit's start-up latency overlaps with the other
// units resident on the SM, and the fold of the splits comes last.
static double gd_ipar_cost(int64_t i_tiles, int n_units, int s, int sms, int resident, int bi, int ti, bool par_fold)
{
    const int64_t work = i_tiles * s;
    const int64_t per_sm = (work + sms - 1) / sms;
    const int ups = (n_units + s - 1) / s;
    const double conc = (double)(per_sm < resident ? per_sm : resident);
    const double chains = conc * bi;                             // independent pair chains per SM sub-partition
    const double eff = chains >= 8.0 ? 1.0 : chains / 8.0;
    const double pair_cycles = (double)per_sm * ups * GD_UNIT_J * ti * 31.0 / 64.0 / eff;
    const double startup = 4000.0 * (double)((per_sm + resident - 1) / resident);
    const double fold = s > 1 ? 1400.0 * (1.0 + (par_fold ? s / 32 : s / 8)) : 0.0;
    return pair_cycles + startup + fold;
}

static void gd_fill_geom(int2 *tab, int64_t max_tiles, int n_units, int64_t pcap, int sms, int resident, int bi, int ti, bool par_fold)
{
    tab[0] = make_int2(1, n_units);
    for (int64_t i_tiles = 1; i_tiles <= max_tiles; ++i_tiles) {
        int64_t s_max = pcap / (i_tiles * ti);
        if (s_max > n_units) s_max = n_units;
        if (s_max > 1024) s_max = 1024;
        if (s_max < 1 || i_tiles >= 16 * (int64_t)sms * resident) s_max = 1;
        int best_s = 1;
        double best = 1e300;
        for (int sp = 1; sp <= s_max; ++sp) {
            double cost = gd_ipar_cost(i_tiles, n_units, sp, sms, resident, bi, ti, par_fold);
            if (cost < best * (1.0 - 1e-9)) { best = cost; best_s = sp; }
        }
        int ups = (n_units + best_s - 1) / best_s;
        tab[i_tiles] = make_int2((n_units + ups - 1) / ups, ups);
    }
}

int gdk_force_setup(gd_ctx *c)
{
    const int n_units = (int)(c->np / GD_UNIT_J);
    int res_s = 0, res_l = 0;
    GD_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&res_s, k_force_ipar<1, 4, false>, GD_IPAR_THREADS, 0));
    GD_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&res_l, k_force_ipar<GD_L_BI, 1, false>, GD_IPAR_THREADS, 0));
    if (res_s < 1) res_s = 1;
    if (res_l < 1) res_l = 1;
    c->grid_s = c->sm_count * res_s;
    c->grid_l = c->sm_count * res_l;
    c->js_clusters = (2 * c->sm_count) / GD_JS_CLUSTER;
    if (c->js_clusters < 1) c->js_clusters = 1;
    const int64_t tiles_s = c->np / GD_TI_S + 1, tiles_l = c->np / GD_TI_L + 1;
    free(c->h_geom_s);
    free(c->h_geom_l);
    c->h_geom_s = (int *)malloc(sizeof(int2) * (size_t)(tiles_s + 1));
    c->h_geom_l = (int *)malloc(sizeof(int2) * (size_t)(tiles_l + 1));
    if (!c->h_geom_s || !c->h_geom_l) return gd_fail_cuda(c, cudaErrorMemoryAllocation, "gdk_force_setup");
    gd_fill_geom((int2 *)c->h_geom_s, tiles_s, n_units, c->pcap, c->sm_count, res_s, 1, GD_TI_S, true);
    gd_fill_geom((int2 *)c->h_geom_l, tiles_l, n_units, c->pcap, c->sm_count, res_l, GD_L_BI, GD_TI_L, false);
    // the host copies stay alive in the context, so the copies need no synchronisation here
    GD_CUDA(c, cudaMemcpyAsync(c->d.geom_s, c->h_geom_s, sizeof(int2) * (size_t)(tiles_s + 1), cudaMemcpyHostToDevice, c->stream));
    GD_CUDA(c, cudaMemcpyAsync(c->d.geom_l, c->h_geom_l, sizeof(int2) * (size_t)(tiles_l + 1), cudaMemcpyHostToDevice, c->stream));
    return 0;
}

static gd_fargs gd_make_fargs(gd_ctx *c, const int32_t *idx, int64_t n_act, bool dev, int lo, int hi, const int2 *geom,
                              double *a_out, double *j_out)
{
    gd_fargs fa;
    fa.idx = idx;
    fa.n_act_dev = dev ? (const long long *)(c->d.cell + 1) : nullptr;
    fa.n_act = (int)n_act;
    fa.lo = lo;
    fa.hi = hi;
    fa.n_units = (int)(c->np / GD_UNIT_J);
    fa.geom = geom;
    fa.eps2 = c->eps2;
    fa.a_out = a_out;
    fa.j_out = j_out;
    return fa;
}

static int gd_launch_jsplit(gd_ctx *c, const gd_fargs &fa, int clusters)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(clusters * GD_JS_CLUSTER));
    cfg.blockDim = dim3(GD_JS_THREADS);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = c->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = GD_JS_CLUSTER;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    cudaError_t e = (c->eps2 < 2.3e-308) ? cudaLaunchKernelEx(&cfg, k_force_jsplit<true>, c->d, fa)
                                         : cudaLaunchKernelEx(&cfg, k_force_jsplit<false>, c->d, fa);
    if (e != cudaSuccess) return gd_fail_cuda(c, e, "k_force_jsplit");
    c->launches += 1;
    return 0;
}

template <int BI, int WJ>
static int gd_launch_ipar(gd_ctx *c, const gd_fargs &fa, int grid)
{
    if (c->eps2 < 2.3e-308)
        k_force_ipar<BI, WJ, true><<<grid, GD_IPAR_THREADS, 0, c->stream>>>(c->d, fa);
    else
        k_force_ipar<BI, WJ, false><<<grid, GD_IPAR_THREADS, 0, c->stream>>>(c->d, fa);
    GD_LAUNCH_CHECK(c, "k_force_ipar");
    return 0;
}

static inline int gd_js_hi(const gd_ctx *c)
{
    int64_t cap = (int64_t)32 * c->js_clusters;
    if (cap > c->pcap / c->js_clusters) cap = c->pcap / c->js_clusters;
    return (int)(c->jsplit_max_nact < cap ? c->jsplit_max_nact : cap);
}

static inline int gd_s_hi(const gd_ctx *c)
{
    int js = gd_js_hi(c);
    int64_t v = c->ipar_small_max_nact;
    if (v > c->np) v = c->np;
    return (int)(v > js ? v : js);
}

// explicit form: the host knows n_act and launches the one kernel that covers it
int gdk_force(gd_ctx *c, const int32_t *idx, int64_t n_act, double *a_out, double *j_out)
{
    if (n_act <= 0) return 0;
    const int js_hi = gd_js_hi(c), s_hi = gd_s_hi(c);
    const int kind = n_act <= gdk_slice_hi(c) ? 4 : (n_act <= js_hi ? 1 : (n_act <= s_hi ? 2 : 0));
    const int slot = gd_prof_begin(c);
    int rc;
    if (kind == 4) {
        rc = gdk_force_slice(c, idx, n_act, a_out, j_out, false);
        c->last_geom[0] = 4; c->last_geom[1] = c->slice_grid; c->last_geom[2] = c->slice_S; c->last_geom[3] = c->slice_passes;
    } else if (kind == 1) {
        int64_t i_tiles = (n_act + 31) / 32;
        rc = gd_launch_jsplit(c, gd_make_fargs(c, idx, n_act, false, 0, INT_MAX, nullptr, a_out, j_out), c->js_clusters);
        c->last_geom[0] = 1; c->last_geom[1] = (int)i_tiles; c->last_geom[2] = c->js_clusters / (int)i_tiles; c->last_geom[3] = 0;
    } else if (kind == 2) {
        int64_t i_tiles = (n_act + GD_TI_S - 1) / GD_TI_S;
        int grid = (int)(i_tiles * 1024 < c->grid_s ? i_tiles * 1024 : c->grid_s);
        rc = gd_launch_ipar<1, 4>(c, gd_make_fargs(c, idx, n_act, false, 0, INT_MAX, c->d.geom_s, a_out, j_out), grid);
        c->last_geom[0] = 2; c->last_geom[1] = (int)i_tiles; c->last_geom[2] = c->h_geom_s[2 * i_tiles]; c->last_geom[3] = c->h_geom_s[2 * i_tiles + 1];
    } else {
        int64_t i_tiles = (n_act + GD_TI_L - 1) / GD_TI_L;
        int grid = (int)(i_tiles * 1024 < c->grid_l ? i_tiles * 1024 : c->grid_l);
        rc = gd_launch_ipar<GD_L_BI, 1>(c, gd_make_fargs(c, idx, n_act, false, 0, INT_MAX, c->d.geom_l, a_out, j_out), grid);
        c->last_geom[0] = 0; c->last_geom[1] = (int)i_tiles; c->last_geom[2] = c->h_geom_l[2 * i_tiles]; c->last_geom[3] = c->h_geom_l[2 * i_tiles + 1];
    }
    c->last_force_kernel = kind == 4 ? 4 : (kind == 1 ? 2 : (kind == 2 ? 3 : 1));
    gd_prof_end(c, slot, kind, (double)n_act * (double)c->n);
    return rc;
}

// graph form: n_act lives in device memory (cell[1]); all three kernels are enqueued and the device picks one
int gdk_force_dev(gd_ctx *c)
{
    const int js_hi = gd_js_hi(c), s_hi = gd_s_hi(c);
    int rc = 0;
    // the same ranges as gdk_force: k_force_slice (kernel + fold, both reading the count on the device) takes the
    // active sets up to its limit, the kernels behind it start above `lo`
    int lo = (int)gdk_slice_hi(c);
    if (lo > 0) rc = gdk_force_slice(c, c->d.idx, lo, c->d.a1, c->d.j1, true);
    if (!rc && js_hi > lo) {
        rc = gd_launch_jsplit(c, gd_make_fargs(c, c->d.idx, 0, true, lo, js_hi, nullptr, c->d.a1, c->d.j1), c->js_clusters);
        lo = js_hi;
    }
    if (!rc && s_hi > lo) {
        rc = gd_launch_ipar<1, 4>(c, gd_make_fargs(c, c->d.idx, 0, true, lo, s_hi, c->d.geom_s, c->d.a1, c->d.j1), c->grid_s);
        lo = s_hi;
    }
    if (!rc && lo < c->np)
        rc = gd_launch_ipar<GD_L_BI, 1>(c, gd_make_fargs(c, c->d.idx, 0, true, lo, INT_MAX, c->d.geom_l, c->d.a1, c->d.j1), c->grid_l);
    return rc;
}
