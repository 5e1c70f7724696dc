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
__device__ __forceinline__ double gd_rsqrt(double s)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(s));
    // s == 0 (coincident particles with eps = 0, or denormal): contribute nothing instead of inf * 0
    if (__double2hiint(s) == 0) y = 0.0;
    double t = s * y;
    double e = fma(-t, y, 1.0);
    double p = fma(0.375, e, 0.5);
    double g = y * e;
    return fma(g, p, y);
}

struct gd_src { double x, y, z, m, vx, vy, vz; };
struct gd_acc { double ax, ay, az, jx, jy, jz; };

__device__ __forceinline__ void gd_pair(const gd_src &i, const gd_src &j, double eps2, gd_acc &o)
{
    double rx = j.x - i.x, ry = j.y - i.y, rz = j.z - i.z;
    double wx = j.vx - i.vx, wy = j.vy - i.vy, wz = j.vz - i.vz;
    double s = fma(rx, rx, fma(ry, ry, fma(rz, rz, eps2)));
    double rw = fma(rx, wx, fma(ry, wy, rz * wz));
    double q = gd_rsqrt(s);
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
#define GD_TILE_BYTES (GD_TILE_J * 56u)

__device__ __forceinline__ void gd_issue_tile(gd_tile *st, uint64_t *bar, const gd_dev &d, int64_t j0)
{
    gd_mbar_expect_tx(bar, GD_TILE_BYTES);
    gd_bulk_g2s(st->pxy, d.pxy + j0, GD_TILE_J * 16u, bar);
    gd_bulk_g2s(st->pzm, d.pzm + j0, GD_TILE_J * 16u, bar);
    gd_bulk_g2s(st->vxy, d.vxy + j0, GD_TILE_J * 16u, bar);
    gd_bulk_g2s(st->vz, d.vz + j0, GD_TILE_J * 8u, bar);
}

// ---------------------------------------------------------------------------------------------------------
// i-parallel kernel.  blockIdx.x = i-tile of BI * 128 sinks (sink k = tile0 + b * 128 + tid: coalesced output),
// blockIdx.y = j-split s covering source tiles [s * tiles_per_split, ...).  n_split == 1 writes a_out/j_out
// ([n_act,3]) directly; otherwise partial[s][k][6] and k_reduce_partials finishes in split order.
template <int BI>
__global__ void __launch_bounds__(GD_IPAR_THREADS)
k_force_ipar(gd_dev d, const int32_t *__restrict__ idx, int n_act, int n_tiles, int tiles_per_split, int n_split,
             double eps2, double *__restrict__ a_out, double *__restrict__ j_out)
{
    __shared__ gd_tile tile[GD_STAGES];
    __shared__ __align__(8) uint64_t full[GD_STAGES];

    const int tid = threadIdx.x;
    const int split = blockIdx.y;
    const int t_begin = split * tiles_per_split;
    const int t_end = min(n_tiles, t_begin + tiles_per_split);
    const int my_tiles = t_end - t_begin;

    if (tid == 0) {
        for (int s = 0; s < GD_STAGES; ++s) gd_mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
        for (int s = 0; s < GD_STAGES && s < my_tiles; ++s)
            gd_issue_tile(&tile[s], &full[s], d, (int64_t)(t_begin + s) * GD_TILE_J);
    }

    gd_src si[BI];
    gd_acc acc[BI];
    const int k0 = blockIdx.x * (BI * GD_IPAR_THREADS) + tid;
#pragma unroll
    for (int b = 0; b < BI; ++b) {
        int k = min(k0 + b * GD_IPAR_THREADS, n_act - 1);          // tail lanes recompute the last sink, never store
        int32_t i = idx ? __ldg(idx + k) : k;
        si[b] = gd_load_sink(d, i);
        acc[b] = gd_acc{0, 0, 0, 0, 0, 0};
    }

    for (int t = 0; t < my_tiles; ++t) {
        const int s = t % GD_STAGES;
        gd_mbar_wait(&full[s], (uint32_t)((t / GD_STAGES) & 1));
        const gd_tile &T = tile[s];
#pragma unroll 2
        for (int jj = 0; jj < GD_TILE_J; ++jj) {
            double2 xy = T.pxy[jj], zm = T.pzm[jj], vxy = T.vxy[jj];
            gd_src sj{xy.x, xy.y, zm.x, zm.y, vxy.x, vxy.y, T.vz[jj]};
#pragma unroll
            for (int b = 0; b < BI; ++b) gd_pair(si[b], sj, eps2, acc[b]);
        }
        __syncthreads();                                         // every warp is done with stage s
        if (tid == 0 && t + GD_STAGES < my_tiles)
            gd_issue_tile(&tile[s], &full[s], d, (int64_t)(t_begin + t + GD_STAGES) * GD_TILE_J);
    }

#pragma unroll
    for (int b = 0; b < BI; ++b) {
        int k = k0 + b * GD_IPAR_THREADS;
        if (k >= n_act) continue;
        if (n_split == 1) {
            a_out[3 * (int64_t)k + 0] = acc[b].ax; a_out[3 * (int64_t)k + 1] = acc[b].ay; a_out[3 * (int64_t)k + 2] = acc[b].az;
            j_out[3 * (int64_t)k + 0] = acc[b].jx; j_out[3 * (int64_t)k + 1] = acc[b].jy; j_out[3 * (int64_t)k + 2] = acc[b].jz;
        } else {
            double2 *p = reinterpret_cast<double2 *>(d.partial + ((int64_t)split * n_act + k) * 6);
            p[0] = make_double2(acc[b].ax, acc[b].ay);
            p[1] = make_double2(acc[b].az, acc[b].jx);
            p[2] = make_double2(acc[b].jy, acc[b].jz);
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// j-split kernel.  CTA = 8 warps arranged as wi x wj (wi * wj = 8): warp (a, b) owns sink group
// g = blockIdx.y * wi + a (BI sinks, the same in every lane) and the lanes of the wj warps stride over the
// CTA's source chunk [blockIdx.x * chunk, ...).  Cluster = cdim consecutive CTAs along x (same sink groups,
// neighbouring chunks).  Reduction: lanes (shuffle) -> warps b = 0..wj-1 (shared memory, in order) -> CTAs of
// the cluster (DSMEM, rank order) -> clusters (k_reduce_partials, in order) unless there is a single cluster.
template <int BI>
__global__ void __launch_bounds__(GD_JS_THREADS)
k_force_jsplit(gd_dev d, const int32_t *__restrict__ idx, int n_act, int np, int chunk, int wi, int cdim,
               double eps2, double *__restrict__ a_out, double *__restrict__ j_out)
{
    __shared__ double red[GD_JS_WARPS][BI * 6];      // per-warp sums
    __shared__ double cta[GD_JS_WARPS][BI * 6];      // per-group CTA sums (first wi rows used)

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int wj = GD_JS_WARPS / wi;
    const int wa = warp % wi, wb = warp / wi;
    const int g = blockIdx.y * wi + wa;

    gd_src si[BI];
    gd_acc acc[BI];
#pragma unroll
    for (int b = 0; b < BI; ++b) {
        int k = min(g * BI + b, n_act - 1);
        int32_t i = idx ? __ldg(idx + k) : k;
        si[b] = gd_load_sink(d, i);
        acc[b] = gd_acc{0, 0, 0, 0, 0, 0};
    }

    const int j_begin = blockIdx.x * chunk;
    const int j_end = min(np, j_begin + chunk);
    const int stride = 32 * wj;
    int j = j_begin + wb * 32 + lane;
    // software pipeline: the next source record is in flight while the current one is consumed
    double2 xy, zm, vxy;
    double vz;
    if (j < j_end) { xy = __ldg(d.pxy + j); zm = __ldg(d.pzm + j); vxy = __ldg(d.vxy + j); vz = __ldg(d.vz + j); }
    while (j < j_end) {
        gd_src sj{xy.x, xy.y, zm.x, zm.y, vxy.x, vxy.y, vz};
        int jn = j + stride;
        if (jn < j_end) { xy = __ldg(d.pxy + jn); zm = __ldg(d.pzm + jn); vxy = __ldg(d.vxy + jn); vz = __ldg(d.vz + jn); }
#pragma unroll
        for (int b = 0; b < BI; ++b) gd_pair(si[b], sj, eps2, acc[b]);
        j = jn;
    }

    // lanes -> warp
#pragma unroll
    for (int b = 0; b < BI; ++b) {
        double v[6] = {acc[b].ax, acc[b].ay, acc[b].az, acc[b].jx, acc[b].jy, acc[b].jz};
#pragma unroll
        for (int c = 0; c < 6; ++c) {
            double x = v[c];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
            if (lane == 0) red[warp][b * 6 + c] = x;
        }
    }
    __syncthreads();
    // warps of one group -> CTA (fixed order wb = 0..wj-1)
    if (threadIdx.x < wi * BI * 6) {
        int a = threadIdx.x / (BI * 6), e = threadIdx.x % (BI * 6);
        double s = 0.0;
        for (int b = 0; b < wj; ++b) s += red[b * wi + a][e];
        cta[a][e] = s;
    }
    cg::cluster_group cluster = cg::this_cluster();
    if (cdim > 1) cluster.sync(); else __syncthreads();
    const unsigned rank = (cdim > 1) ? cluster.block_rank() : 0;
    if (rank == 0 && threadIdx.x < wi * BI * 6) {
        int a = threadIdx.x / (BI * 6), e = threadIdx.x % (BI * 6);
        double s = cta[a][e];
        for (int r = 1; r < cdim; ++r) {
            const double *remote = cluster.map_shared_rank(&cta[0][0], r);     // DSMEM read of CTA r's sums
            s += remote[a * (BI * 6) + e];
        }
        int k = (blockIdx.y * wi + a) * BI + e / 6, comp = e % 6;
        if (k < n_act) {
            int n_clusters = gridDim.x / cdim;
            if (n_clusters == 1) {
                double *o = comp < 3 ? a_out : j_out;
                o[3 * (int64_t)k + comp % 3] = s;
            } else {
                int cl = blockIdx.x / cdim;
                d.partial[((int64_t)cl * n_act + k) * 6 + comp] = s;
            }
        }
    }
    if (cdim > 1) cluster.sync();                   // keep every CTA's shared memory alive until rank 0 has read it
}

// out[k][c] = sum_{s = 0..n_split-1} partial[s][k][c], in that order
__global__ void __launch_bounds__(256) k_reduce_partials(const double *__restrict__ partial, int n_act, int n_split,
                                                         double *__restrict__ a_out, double *__restrict__ j_out)
{
    int64_t e = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (e >= (int64_t)n_act * 6) return;
    double s = 0.0;
    for (int p = 0; p < n_split; ++p) s += partial[(int64_t)p * n_act * 6 + e];
    int64_t k = e / 6;
    int comp = (int)(e % 6);
    double *o = comp < 3 ? a_out : j_out;
    o[3 * k + comp % 3] = s;
}

// ---------------------------------------------------------------------------------------------------------
// Host side: launch geometry.
#define GD_IPAR_BI 2
#define GD_JS_BI 4

// smallest split count in [1, s_max] whose grid fills the machine to >= 95 % of its last wave (else the best seen)
static int gd_pick_split(int64_t units, int64_t slots, int s_max)
{
    int best = 1;
    double best_eff = 0.0;
    for (int s = 1; s <= s_max; ++s) {
        int64_t ctas = units * s;
        int64_t waves = (ctas + slots - 1) / slots;
        double eff = (double)ctas / (double)(waves * slots);
        if (eff > best_eff + 1e-9) { best_eff = eff; best = s; }
        if (eff >= 0.95) return s;
    }
    return best;
}

static int gd_force_ipar(gd_ctx *c, const int32_t *idx, int64_t n_act, double *a_out, double *j_out)
{
    const int n_tiles = (int)(c->np / GD_TILE_J);
    const int64_t i_tiles = (n_act + GD_IPAR_BI * GD_IPAR_THREADS - 1) / (GD_IPAR_BI * GD_IPAR_THREADS);
    static int ctas_per_sm = 0;
    if (!ctas_per_sm) {
        GD_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas_per_sm, k_force_ipar<GD_IPAR_BI>, GD_IPAR_THREADS, 0));
        if (ctas_per_sm < 1) ctas_per_sm = 1;
    }
    const int64_t slots = (int64_t)c->sm_count * ctas_per_sm;
    int s_max = (int)((c->pcap / n_act) < 64 ? (c->pcap / n_act) : 64);
    if (s_max > n_tiles / 4) s_max = n_tiles / 4;               // keep >= 4 source tiles per CTA
    if (s_max < 1) s_max = 1;
    int n_split = (i_tiles >= 16 * slots) ? 1 : gd_pick_split(i_tiles, slots, s_max);
    int tiles_per_split = (n_tiles + n_split - 1) / n_split;
    n_split = (n_tiles + tiles_per_split - 1) / tiles_per_split;
    dim3 grid((unsigned)i_tiles, (unsigned)n_split);
    k_force_ipar<GD_IPAR_BI><<<grid, GD_IPAR_THREADS, 0, c->stream>>>(c->d, idx, (int)n_act, n_tiles, tiles_per_split,
                                                                        n_split, c->eps2, a_out, j_out);
    GD_LAUNCH_CHECK(c, "k_force_ipar");
    if (n_split > 1) {
        k_reduce_partials<<<(unsigned)((n_act * 6 + 255) / 256), 256, 0, c->stream>>>(c->d.partial, (int)n_act, n_split, a_out, j_out);
        GD_LAUNCH_CHECK(c, "k_reduce_partials");
    }
    c->last_force_kernel = 1;
    return 0;
}

static int gd_force_jsplit(gd_ctx *c, const int32_t *idx, int64_t n_act, double *a_out, double *j_out)
{
    const int64_t groups = (n_act + GD_JS_BI - 1) / GD_JS_BI;
    int wi = 1;
    while (wi < GD_JS_WARPS && wi < groups) wi *= 2;
    const int wj = GD_JS_WARPS / wi;
    const int64_t gy = (groups + wi - 1) / wi;
    // CTAs along the source axis: fill the SMs, but leave every lane at least two sources
    int64_t sx_cap = c->np / (64 * wj);
    if (sx_cap < 1) sx_cap = 1;
    if (sx_cap > c->pcap / n_act) sx_cap = c->pcap / n_act;
    int64_t sx = (int64_t)c->sm_count / gy;
    if (sx < 1) sx = 1;
    if (sx > sx_cap) sx = sx_cap;
    int cdim = 1;
    if (sx >= 4) { cdim = 4; sx = (sx / 4) * 4; }
    else if (sx >= 2) { cdim = 2; sx = 2; }
    int chunk = (int)((c->np + sx - 1) / sx);
    chunk = ((chunk + 31) / 32) * 32;
    const int n_clusters = (int)(sx / cdim);

    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)sx, (unsigned)gy);
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
    GD_CUDA(c, cudaLaunchKernelEx(&cfg, k_force_jsplit<GD_JS_BI>, c->d, idx, (int)n_act, (int)c->np, chunk, wi, cdim,
                                  c->eps2, a_out, j_out));
    c->launches += 1;
    if (n_clusters > 1) {
        k_reduce_partials<<<(unsigned)((n_act * 6 + 255) / 256), 256, 0, c->stream>>>(c->d.partial, (int)n_act, n_clusters, a_out, j_out);
        GD_LAUNCH_CHECK(c, "k_reduce_partials");
    }
    c->last_force_kernel = 2;
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
