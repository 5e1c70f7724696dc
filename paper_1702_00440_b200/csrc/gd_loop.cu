// gd_loop.cu -- persistent block-step loop: the whole cycle  next_block -> predict -> force/jerk
// -> correct + time step for the SMALL active sets that dominate the step count under block time
// steps ("N_act << N"), as ONE cooperative kernel that stays resident and iterates on the device.
//
// Why: with n_act ~ 10..100 a block step is 1 us of FP64 work behind ~35 us of launches and dependent round trips
// when every stage is its own kernel.  Here a block step costs two grid barriers.
//
// Decomposition (j-split over the whole machine, Fig. 3 P:173 turned inside out): CTA c OWNS the particle slice
// [c S, (c+1) S): it alone reads and writes their state, keeps their t_i + dt_i and their predicted records in
// shared memory, and evaluates the partial a, jerk of EVERY active sink against its own S sources.  Per block step:
//
//   [publish]  (owner, after its particles changed)  L_c = min of its t_i + dt_i; its candidates {i : t_i + dt_i = L_c},
//              ascending, predicted to L_c, go to its segment of `rec` with L_c and their count
//   -- grid barrier --
//   [force]    every CTA: t+ = min_c L_c; the active list is the concatenation, in CTA order (= ascending index), of
//              the segments with L_c = t+; predict own slice to t+ (shared memory); partial sums of all sinks over
//              own sources (lanes stride over sources, register blocks of 4 sinks, fixed-tree warp reduction)
//              -> partial[c][k][6]
//   -- grid barrier --
//   [correct]  owners of the active particles: sum the partials over c in ascending order, Hermite corrector,
//              Aarseth criterion, block rule, commit; then [publish] again
//
// The loop leaves (without touching the state) when the next active set is larger than `hi` -- the host-enqueued
// stage kernels take that step -- or when t_end / max_steps is reached.  All arithmetic on the discrete decisions
// is the code of gd_hermite.cuh, the pair term is gd_pair.cuh: the same functions the stage kernels run.
// Every summation order is fixed by the geometry (never by timing): results are run-to-run identical.
#include "gd_common.cuh"
#include "gd_hermite.cuh"
#include "gd_pair.cuh"
#include <limits.h>

#ifndef GD_LP_THREADS
#define GD_LP_THREADS 256          // threads of the one CTA per SM (a multiple of 32; tuning knob)
#endif
#define GD_LP_WARPS (GD_LP_THREADS / 32)
#ifndef GD_LP_PROFILE
#define GD_LP_PROFILE 1            // 1: k_block_loop also exists as an instantiation with timers, launched when the "loop_timers"
#endif                             //    option is set (the default instantiation has none); 0: no timers at all (the ns of
                                   //    gd_get_loop_profile / gd_get_loop_histogram stay 0)
#ifndef GD_LP_ITEM_UNROLL
#define GD_LP_ITEM_UNROLL 2        // unrolling of the round loop of a lanes-over-sources item
#endif
#ifndef GD_LP_WIDE_UNROLL
#define GD_LP_WIDE_UNROLL 4        // unrolling of the source loop of the wide sink tiles (measured: 2 -> 4 gains 1 - 3 %)
#endif
#define GD_LP_PRAGMA_(x) _Pragma(#x)
#define GD_LP_PRAGMA_UNROLL(n) GD_LP_PRAGMA_(unroll n)
#define GD_LP_MAX_GRID 256          // CTAs (one per SM); bounds the shared tables
// Thread `tid` of every CTA handles CTA `tid`'s published minimum and candidate count, and the step's owners are counted
// with one __syncthreads_count over those threads: every tid < G has to exist.
static_assert(GD_LP_THREADS >= GD_LP_MAX_GRID, "k_block_loop reads one CTA's {L, count} per thread: GD_LP_THREADS must cover GD_LP_MAX_GRID");
static_assert(GD_LP_THREADS % 32 == 0 && GD_LP_THREADS <= 1024, "GD_LP_THREADS: a multiple of 32, at most 1024");
#define GD_LP_MAX_SMALL 256         // largest active set of the lanes-over-sources mapping (bounds the position map)

struct gd_largs {
    int n;                           // particles; CTA c owns [c n / G, (c + 1) n / G)
    int S;                           // slice capacity in shared memory (multiple of 32)
    int hi;                          // largest active set the loop takes
    int cap;                         // positions the partial-sum scratch holds: partial[cap][G][6]
    int small_hi;                    // n_act <= small_hi: lanes over sources; above: lanes over sinks
    int wc_hi;                       // [correct]: up to wc_hi own active particles a warp each, above a thread each
    int state;                       // != 0: the own state is resident in shared memory
    double eps2, eta, dt_min, dt_max;
    int halving_mode;
    int passes;                      // k_force_slice: slices per CTA, taken one after the other (1 where n / grid records fit)
    int ext;                         // != 0 (k_force_slice): the sinks are named by ext_idx in the predicted planes
    const int32_t *ext_idx;          //   (NULL: sink k = particle k); 0 (k_block_loop): they are the published records
};

__device__ __forceinline__ int gd_slice_begin(int c, int n, int G) { return (int)((long long)c * n / G); }

#define GD_INF __longlong_as_double(0x7ff0000000000000LL)
#define GD_FULL 0xffffffffu

// ---- grid barrier: monotonic 64-bit arrival counter, one arrival per CTA ------------------------------------------
__device__ __forceinline__ void gd_bar_arrive(unsigned long long *bar)
{
    __syncthreads();                                         // every thread's stores precede thread 0's release
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(bar, 1ull);
    }
}
__device__ __forceinline__ void gd_bar_wait(unsigned long long *bar, unsigned long long target)
{
    if (threadIdx.x == 0) {
        unsigned long long v;
        do {
            asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(bar) : "memory");
        } while (v < target);
    }
    __syncthreads();
}

// device global timer, read by thread 0 of CTA 0 of the instantiation with timers only (the read is slow); 0 elsewhere
template <bool TIMERS>
__device__ __forceinline__ unsigned long long gd_gtime()
{
    unsigned long long t = 0;
#if GD_LP_PROFILE
    if (TIMERS && blockIdx.x == 0 && threadIdx.x == 0) asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
#endif
    return t;
}

// warp minimum of non-negative doubles (times, +inf): their order is the order of their bit patterns, so two
// integer warp reductions (REDUX) do it -- high words first, then the low words of the lanes that tie
__device__ __forceinline__ double gd_warp_min_d(double v)
{
    const unsigned int hi = (unsigned int)__double2hiint(v), lo = (unsigned int)__double2loint(v);
    const unsigned int mh = __reduce_min_sync(GD_FULL, hi);
    const unsigned int ml = __reduce_min_sync(GD_FULL, hi == mh ? lo : 0xffffffffu);
    return __hiloint2double((int)mh, (int)ml);
}

// ---- fixed-tree warp reduce-scatter ---------------------------------------------------------------------------------
// N values per lane -> after the step, N/2 values per lane, each the sum of the lane pair (lane, lane ^ o); lanes
// with bit o clear keep elements [0, N/2), the others [N/2, N).
template <int N>
__device__ __forceinline__ void gd_rs_step(double *v, int o, int lane)
{
    const bool up = (lane & o) != 0;
#pragma unroll
    for (int k = 0; k < N / 2; ++k) {
        double keep = up ? v[k + N / 2] : v[k];
        double send = up ? v[k] : v[k + N / 2];
        v[k] = keep + __shfl_xor_sync(GD_FULL, send, o);
    }
}

// 24 sums (4 sinks x 6) -> lane holds element gd_rs24_elem(lane) in v[0] (element 24.. = padding)
__device__ __forceinline__ void gd_rs24(double *v, int lane)
{
    gd_rs_step<24>(v, 16, lane);
    gd_rs_step<12>(v, 8, lane);
    gd_rs_step<6>(v, 4, lane);
    v[3] = 0.0;
    gd_rs_step<4>(v, 2, lane);
    gd_rs_step<2>(v, 1, lane);
}
__device__ __forceinline__ int gd_rs24_elem(int lane)
{
    if ((lane & 3) == 3) return -1;
    return ((lane & 16) ? 12 : 0) + ((lane & 8) ? 6 : 0) + ((lane & 4) ? 3 : 0) + ((lane & 2) ? 2 : 0) + (lane & 1);
}
// 6 sums (1 sink) -> lanes with (lane & 3) == 0 hold element gd_rs6_elem(lane)
__device__ __forceinline__ void gd_rs6(double *v, int lane)
{
    gd_rs_step<6>(v, 16, lane);
    v[3] = 0.0;
    gd_rs_step<4>(v, 8, lane);
    gd_rs_step<2>(v, 4, lane);
    v[0] += __shfl_xor_sync(GD_FULL, v[0], 2);
    v[0] += __shfl_xor_sync(GD_FULL, v[0], 1);
}
__device__ __forceinline__ int gd_rs6_elem(int lane)
{
    if ((lane & 3) != 0 || (lane & 12) == 12) return -1;
    return ((lane & 16) ? 3 : 0) + ((lane & 8) ? 2 : 0) + ((lane & 4) ? 1 : 0);
}

// ---- shared memory of one CTA ----------------------------------------------------------------------------------------
struct gd_lsm {
    double2 *pxy, *pzm, *vxy;        // [S] predicted records of the own slice (at t+ during [force] / [correct]);
    double *vz;                      // [S]   entries beyond the slice are zero-mass padding up to a multiple of 32
    double *ts;                      // [S] t_i + dt_i of the own slice
    int *lact;                       // [S] local indices of the own candidates, ascending
    int *smap;                       // [GD_LP_MAX_SMALL] active list position -> row of `rec` (small mode)
    double2 *sink;                   // [GD_LP_MAX_SMALL][4] the sink records of the step (small mode)
    int *spre;                       // [GD_LP_MAX_GRID + 1] exclusive prefix of the contributing candidate counts
    int *p0t;                        // [GD_LP_MAX_GRID + 1] first particle of every CTA's slice (k_block_loop fills it once)
    double *red;                     // [GD_LP_WARPS][4][6][32] warp partial sums of a split evaluation
    double *wmin;                    // [GD_LP_WARPS]
    int *wcnt;                       // [GD_LP_WARPS + 1]
    unsigned int *hist;              // [64] particle steps per level, [64..65] diagnostics
    double4 *xm, *vt, *ad, *jk;      // [S] own state (only when it fits: `state` != 0; global memory is written through)
};

__host__ __device__ inline size_t gd_lsm_bytes(int S, int state)
{
    return (size_t)S * (16 * 3 + 8 + 8 + 4 + (state ? 128 : 0)) + GD_LP_WARPS * 4 * 6 * 32 * 8 + GD_LP_WARPS * 8 + GD_LP_MAX_SMALL * (4 + 64) +
           2 * (GD_LP_MAX_GRID + 1) * 4 + (GD_LP_WARPS + 1) * 4 + 66 * 4 + 64;
}

__device__ __forceinline__ gd_lsm gd_lsm_carve(unsigned char *base, int S, int state)
{
    gd_lsm s;
    unsigned char *p = base;
    s.xm = s.vt = s.ad = s.jk = nullptr;
    if (state) {
        s.xm = (double4 *)p; p += (size_t)S * 32;
        s.vt = (double4 *)p; p += (size_t)S * 32;
        s.ad = (double4 *)p; p += (size_t)S * 32;
        s.jk = (double4 *)p; p += (size_t)S * 32;
    }
    s.pxy = (double2 *)p; p += (size_t)S * 16;
    s.pzm = (double2 *)p; p += (size_t)S * 16;
    s.vxy = (double2 *)p; p += (size_t)S * 16;
    s.vz = (double *)p; p += (size_t)S * 8;
    s.ts = (double *)p; p += (size_t)S * 8;
    s.red = (double *)p; p += GD_LP_WARPS * 4 * 6 * 32 * 8;
    s.wmin = (double *)p; p += GD_LP_WARPS * 8;
    s.sink = (double2 *)p; p += GD_LP_MAX_SMALL * 64;
    s.lact = (int *)p; p += (size_t)S * 4;
    s.smap = (int *)p; p += GD_LP_MAX_SMALL * 4;
    s.spre = (int *)p; p += (GD_LP_MAX_GRID + 1) * 4;
    s.p0t = (int *)p; p += (GD_LP_MAX_GRID + 1) * 4;
    s.wcnt = (int *)p; p += (GD_LP_WARPS + 1) * 4;
    s.hist = (unsigned int *)p;
    return s;
}

// own state of local particle p (global index i): shared memory when resident, else global memory (owner-only data)
#define GD_LP_XM(p, i) (sm.xm ? sm.xm[p] : d.xm[i])
#define GD_LP_VT(p, i) (sm.xm ? sm.vt[p] : d.vt[i])
#define GD_LP_AD(p, i) (sm.xm ? sm.ad[p] : d.ad[i])
#define GD_LP_JK(p, i) (sm.xm ? sm.jk[p] : d.jk[i])

// ---- [publish]: L_c, the candidates of this CTA (ascending), their records predicted to L_c ------------------------------
// rec row r = two double4: {xp, yp, zp, particle index (as an integer in a double)}, {vxp, vyp, vzp, 0}
__device__ __forceinline__ int gd_publish(const gd_dev &d, const gd_lsm &sm, int me, int p0, int cnt_own, double *L_out)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double m = GD_INF;
    for (int p = tid; p < cnt_own; p += GD_LP_THREADS) m = fmin(m, sm.ts[p]);
    m = gd_warp_min_d(m);
    if (lane == 0) sm.wmin[warp] = m;
    __syncthreads();
    m = lane < GD_LP_WARPS ? sm.wmin[lane] : GD_INF;
    m = gd_warp_min_d(m);
    const double L = m;
    int base = 0;
    if (L < GD_INF) {
        for (int r0 = 0; r0 < cnt_own; r0 += GD_LP_THREADS) {
            const int p = r0 + tid;
            const bool f = p < cnt_own && sm.ts[p] == L;
            const unsigned int bal = __ballot_sync(GD_FULL, f);
            if (lane == 0) sm.wcnt[warp] = __popc(bal);
            __syncthreads();
            int before = 0, total = 0;
#pragma unroll
            for (int w = 0; w < GD_LP_WARPS; ++w) {
                int c = sm.wcnt[w];
                before += (w < warp) ? c : 0;
                total += c;
            }
            if (f) sm.lact[base + before + __popc(bal & ((1u << lane) - 1u))] = p;
            base += total;
            __syncthreads();
        }
    }
    const int cnt = base;
    for (int k = tid; k < cnt; k += GD_LP_THREADS) {
        const int p = sm.lact[k], i = p0 + p;
        const double4 xm = GD_LP_XM(p, i), vt = GD_LP_VT(p, i), ad = GD_LP_AD(p, i), jk = GD_LP_JK(p, i);
        const gd_pred q = gd_predict_record(xm, vt, ad, jk, L);
        double4 *row = d.lp_rec + 2 * (size_t)(p0 + k);
        row[0] = make_double4(q.x, q.y, q.z, (double)i);
        row[1] = make_double4(q.vx, q.vy, q.vz, 0.0);
    }
    if (tid == 0) {
        d.lp_L[me] = L;
        d.lp_cnt[me] = cnt;
    }
    *L_out = L;
    __syncthreads();                                         // wmin / wcnt / lact are reused by the caller
    return cnt;
}

__device__ __forceinline__ gd_src gd_lp_load_sink(const gd_dev &d, int row_index)
{
    const double2 *row = reinterpret_cast<const double2 *>(d.lp_rec + 2 * (size_t)row_index);
    const double2 xy = __ldcg(row), zi = __ldcg(row + 1), wxy = __ldcg(row + 2), wz = __ldcg(row + 3);
    return gd_src{xy.x, xy.y, zi.x, 0.0, wxy.x, wxy.y, wz.x};
}

// ---- [force], small mode: lanes stride over the own sources ------------------------------------------------------------
// BI sinks (active-list positions pos0 .. pos0 + BI - 1) against the source rounds [r_begin, r_end) of the own
// slice; lane l takes source 32 r + l.  Returns the 6 BI per-lane sums in v[b * 6 + {ax, ay, az, jx, jy, jz}].
template <int BI, bool EPS0, int UNR = GD_LP_ITEM_UNROLL>
__device__ __forceinline__ void gd_lp_item(const gd_dev &d, const gd_lsm &sm, int pos0, int r_begin, int r_end, int lane,
                                           double eps2, double *v)
{
    gd_src si[BI];
    gd_acc acc[BI];
#pragma unroll
    for (int b = 0; b < BI; ++b) {
        const double2 *row = sm.sink + 4 * (pos0 + b);
        const double2 xy = row[0], zi = row[1], wxy = row[2], wz = row[3];
        si[b] = gd_src{xy.x, xy.y, zi.x, 0.0, wxy.x, wxy.y, wz.x};
        acc[b] = gd_acc{0, 0, 0, 0, 0, 0};
    }
    GD_LP_PRAGMA_UNROLL(UNR)
    for (int r = r_begin; r < r_end; ++r) {
        const int j = r * 32 + lane;
        const double2 xy = sm.pxy[j], zm = sm.pzm[j], vxy = sm.vxy[j];
        const gd_src sj{xy.x, xy.y, zm.x, zm.y, vxy.x, vxy.y, sm.vz[j]};
#pragma unroll
        for (int b = 0; b < BI; ++b) gd_pair<EPS0>(si[b], sj, eps2, acc[b]);
    }
#pragma unroll
    for (int b = 0; b < BI; ++b) {
        v[b * 6 + 0] = acc[b].ax; v[b * 6 + 1] = acc[b].ay; v[b * 6 + 2] = acc[b].az;
        v[b * 6 + 3] = acc[b].jx; v[b * 6 + 4] = acc[b].jy; v[b * 6 + 5] = acc[b].jz;
    }
}

// Partial sums: partial[position][CTA][6], so that the G rows of one active particle are contiguous for its owner.
// `out` points at this CTA's row of position 0, rs = 6 G doubles is the distance between positions.
// element e = b * 6 + comp of the block starting at position pos -> row of position pos + b
__device__ __forceinline__ void gd_lp_put(double *out, int rs, int pos, int e, double val)
{
    const int b = e / 6;
    out[(size_t)(pos + b) * rs + (e - 6 * b)] = val;
}

// One work item = a register block of sinks: items 0 .. n4 - 1 hold 4 sinks, the n_act % 4 last ones hold 1.
// items >= warps: warp w takes items w, w + 8, ... over all source rounds and writes its sums itself.
// items <  warps: the rounds of every item are split over nsplit = 8 / items warps; the warp sums meet in shared
//                 memory and are added in chunk order.
template <bool EPS0>
__device__ __forceinline__ void gd_lp_force_small(const gd_dev &d, const gd_lsm &sm, const gd_largs &la, double *out, int rs, int n_act, int rounds)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (n_act <= GD_LP_WARPS && rounds <= 8) {               // a handful of sinks against a short slice: a warp per sink, no hand-off
        if (warp < n_act) {
            double v[6];
            gd_lp_item<1, EPS0, 4>(d, sm, warp, 0, rounds, lane, la.eps2, v);
            gd_rs6(v, lane);
            const int e = gd_rs6_elem(lane);
            if (e >= 0) gd_lp_put(out, rs, warp, e, v[0]);
        }
        return;
    }
    const int n4 = n_act >> 2, items = n4 + (n_act & 3);
    if (items >= GD_LP_WARPS) {
        for (int it = warp; it < items; it += GD_LP_WARPS) {
            if (it < n4) {
                double v[24];
                gd_lp_item<4, EPS0>(d, sm, 4 * it, 0, rounds, lane, la.eps2, v);
                gd_rs24(v, lane);
                const int e = gd_rs24_elem(lane);
                if (e >= 0) gd_lp_put(out, rs, 4 * it, e, v[0]);
            } else {
                double v[6];
                const int pos = 4 * n4 + (it - n4);
                gd_lp_item<1, EPS0>(d, sm, pos, 0, rounds, lane, la.eps2, v);
                gd_rs6(v, lane);
                const int e = gd_rs6_elem(lane);
                if (e >= 0) gd_lp_put(out, rs, pos, e, v[0]);
            }
        }
        return;
    }
    const int nsplit = GD_LP_WARPS / items;                  // >= 1; warps beyond items * nsplit idle
    const int it = warp / nsplit, chunk = warp - it * nsplit;
    const bool work = it < items;
    const bool four = it < n4;
    const int pos = four ? 4 * it : 4 * n4 + (it - n4);
    if (work) {
        const int rb = rounds * chunk / nsplit, re = rounds * (chunk + 1) / nsplit;
        if (four) {
            double v[24];
            gd_lp_item<4, EPS0>(d, sm, pos, rb, re, lane, la.eps2, v);
            gd_rs24(v, lane);
            const int e = gd_rs24_elem(lane);
            if (e >= 0) sm.red[warp * 32 + e] = v[0];
        } else {
            double v[6];
            gd_lp_item<1, EPS0>(d, sm, pos, rb, re, lane, la.eps2, v);
            gd_rs6(v, lane);
            const int e = gd_rs6_elem(lane);
            if (e >= 0) sm.red[warp * 32 + e] = v[0];
        }
    }
    __syncthreads();
    if (work && chunk == 0 && lane < (four ? 24 : 6)) {
        double s = sm.red[warp * 32 + lane];
        for (int c = 1; c < nsplit; ++c) s += sm.red[(warp + c) * 32 + lane];
        gd_lp_put(out, rs, pos, lane, s);
    }
}

// ---- [force], big mode: lanes hold sinks, the own sources are read by broadcast --------------------------------------
// narrow tiles: one sink per lane, two independent accumulator sets (even / odd sources)
template <bool EPS0>
__device__ __forceinline__ gd_acc gd_lp_tile(const gd_lsm &sm, const gd_src &si, int jb, int je, double eps2)
{
    gd_acc a0 = gd_acc{0, 0, 0, 0, 0, 0}, a1 = gd_acc{0, 0, 0, 0, 0, 0};
    int j = jb;
#pragma unroll 2
    for (; j + 1 < je; j += 2) {
        const double2 xy0 = sm.pxy[j], zm0 = sm.pzm[j], vxy0 = sm.vxy[j];
        const double2 xy1 = sm.pxy[j + 1], zm1 = sm.pzm[j + 1], vxy1 = sm.vxy[j + 1];
        const gd_src s0{xy0.x, xy0.y, zm0.x, zm0.y, vxy0.x, vxy0.y, sm.vz[j]};
        const gd_src s1{xy1.x, xy1.y, zm1.x, zm1.y, vxy1.x, vxy1.y, sm.vz[j + 1]};
        gd_pair<EPS0>(si, s0, eps2, a0);
        gd_pair<EPS0>(si, s1, eps2, a1);
    }
    if (j < je) {
        const double2 xy0 = sm.pxy[j], zm0 = sm.pzm[j], vxy0 = sm.vxy[j];
        const gd_src s0{xy0.x, xy0.y, zm0.x, zm0.y, vxy0.x, vxy0.y, sm.vz[j]};
        gd_pair<EPS0>(si, s0, eps2, a0);
    }
    a0.ax += a1.ax; a0.ay += a1.ay; a0.az += a1.az;
    a0.jx += a1.jx; a0.jy += a1.jy; a0.jz += a1.jz;
    return a0;
}

// wide tiles: BI sinks per lane (positions pos0 + 32 b + lane) against the sources [jb, je), one accumulator set per sink
template <int BI, bool EPS0>
__device__ __forceinline__ void gd_lp_tile_wide(const gd_lsm &sm, const gd_src (&si)[BI], int jb, int je, double eps2, gd_acc (&acc)[BI])
{
#pragma unroll
    for (int b = 0; b < BI; ++b) acc[b] = gd_acc{0, 0, 0, 0, 0, 0};
    GD_LP_PRAGMA_UNROLL(GD_LP_WIDE_UNROLL)
    for (int j = jb; j < je; ++j) {
        const double2 xy = sm.pxy[j], zm = sm.pzm[j], vxy = sm.vxy[j];
        const gd_src sj{xy.x, xy.y, zm.x, zm.y, vxy.x, vxy.y, sm.vz[j]};
#pragma unroll
        for (int b = 0; b < BI; ++b) gd_pair<EPS0>(si[b], sj, eps2, acc[b]);
    }
}

// position in the active list -> row of rec: CTA c with spre[c] <= pos < spre[c + 1] (segments of empty CTAs have
// zero width), row = first row of c's segment + offset
__device__ __forceinline__ int gd_lp_row_of(const gd_lsm &sm, int pos, int n, int G)
{
    int lo = 0, hi = G;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (sm.spre[mid] <= pos) lo = mid; else hi = mid;
    }
    return sm.p0t[lo] + (pos - sm.spre[lo]);
}

// sink at a position of the active list
__device__ __forceinline__ gd_src gd_lp_sink_at(const gd_dev &d, const gd_lsm &sm, const gd_largs &la, int pos, int G)
{
    if (la.ext) {
        const int i = la.ext_idx ? __ldg(la.ext_idx + pos) : pos;
        const double2 xy = __ldg(d.pxy + i), zm = __ldg(d.pzm + i), vxy = __ldg(d.vxy + i);
        return gd_src{xy.x, xy.y, zm.x, 0.0, vxy.x, vxy.y, __ldg(d.vz + i)};
    }
    return gd_lp_load_sink(d, gd_lp_row_of(sm, pos, la.n, G));
}

// Tiles of 32 BI consecutive positions, BI sinks per lane: BI independent pair chains per warp (the FP64 pipe needs
// ~8 per scheduler to stay busy) and one shared-memory read of a source per BI pairs.  tiles >= warps: warp w takes
// tiles w, w + 8, ... against the whole slice.  Fewer tiles: see below.
template <int BI, bool EPS0>
__device__ __forceinline__ void gd_lp_force_wide(const gd_dev &d, const gd_lsm &sm, const gd_largs &la, double *out, int rs, int G, int n_act, int cnt_own)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int tiles = (n_act + 32 * BI - 1) / (32 * BI);
    if (tiles >= GD_LP_WARPS) {
        for (int tile = warp; tile < tiles; tile += GD_LP_WARPS) {
            gd_src si[BI];
            gd_acc acc[BI];
#pragma unroll
            for (int b = 0; b < BI; ++b) si[b] = gd_lp_sink_at(d, sm, la, min(tile * 32 * BI + 32 * b + lane, n_act - 1), G);
            gd_lp_tile_wide<BI, EPS0>(sm, si, 0, cnt_own, la.eps2, acc);
#pragma unroll
            for (int b = 0; b < BI; ++b) {
                const int pos = tile * 32 * BI + 32 * b + lane;
                if (pos < n_act) {
                    double2 *o = reinterpret_cast<double2 *>(out + (size_t)pos * rs);
                    o[0] = make_double2(acc[b].ax, acc[b].ay); o[1] = make_double2(acc[b].az, acc[b].jx); o[2] = make_double2(acc[b].jy, acc[b].jz);
                }
            }
        }
        return;
    }
    // fewer tiles than warps: the slice is split over nsplit = 8 / tiles warps per tile; the warp sums meet in shared
    // memory and are added in chunk order
    const int nsplit = GD_LP_WARPS / tiles;
    const int tile = warp / nsplit, chunk = warp - tile * nsplit;
    const bool work = tile < tiles;
    if (work) {
        gd_src si[BI];
        gd_acc acc[BI];
#pragma unroll
        for (int b = 0; b < BI; ++b) si[b] = gd_lp_sink_at(d, sm, la, min(tile * 32 * BI + 32 * b + lane, n_act - 1), G);
        const int jb = (int)((long long)cnt_own * chunk / nsplit), je = (int)((long long)cnt_own * (chunk + 1) / nsplit);
        gd_lp_tile_wide<BI, EPS0>(sm, si, jb, je, la.eps2, acc);
#pragma unroll
        for (int b = 0; b < BI; ++b) {
            double *r = sm.red + (warp * 4 + b) * 192 + lane;
            r[0] = acc[b].ax; r[32] = acc[b].ay; r[64] = acc[b].az; r[96] = acc[b].jx; r[128] = acc[b].jy; r[160] = acc[b].jz;
        }
    }
    __syncthreads();
    if (work && chunk == 0) {
#pragma unroll
        for (int b = 0; b < BI; ++b) {
            const int pos = tile * 32 * BI + 32 * b + lane;
            if (pos < n_act) {
#pragma unroll
                for (int comp = 0; comp < 6; ++comp) {
                    double sum = sm.red[(warp * 4 + b) * 192 + comp * 32 + lane];
                    for (int c = 1; c < nsplit; ++c) sum += sm.red[((warp + c) * 4 + b) * 192 + comp * 32 + lane];
                    out[(size_t)pos * rs + comp] = sum;
                }
            }
        }
    }
}

// share of the warps that work when `tiles` tiles are dealt to 8 warps (tiles < 8: the sources are split instead)
__device__ __forceinline__ int gd_lp_balance(int tiles)
{
    if (tiles < GD_LP_WARPS) return 100 * (tiles * (GD_LP_WARPS / tiles)) / GD_LP_WARPS;
    return 100 * tiles / (GD_LP_WARPS * ((tiles + GD_LP_WARPS - 1) / GD_LP_WARPS));
}

template <bool EPS0>
__device__ __forceinline__ void gd_lp_force_big(const gd_dev &d, const gd_lsm &sm, const gd_largs &la, double *out, int rs, int G, int n_act, int cnt_own)
{
    // Wide tiles (2 or 4 sinks per lane: more independent pair chains per warp, fewer shared-memory reads per pair)
    // wherever they still deal the work evenly: always from 1024 sinks on, and below that when the slice is long
    // enough to be split over the warps of a tile (measured: N = 65536, 256 sinks: 44 us against 76 us with narrow
    // tiles; N = 16384 the other way round).
    if (n_act >= 2 * 64 * GD_LP_WARPS || cnt_own >= 256) {
        if (GD_LP_THREADS <= 256 && gd_lp_balance((n_act + 127) >> 7) + 5 >= gd_lp_balance((n_act + 63) >> 6))
            gd_lp_force_wide<4, EPS0>(d, sm, la, out, rs, G, n_act, cnt_own);
        else
            gd_lp_force_wide<2, EPS0>(d, sm, la, out, rs, G, n_act, cnt_own);
        return;
    }
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tiles = (n_act + 31) >> 5;
    if (tiles >= GD_LP_WARPS) {
        for (int tile = warp; tile < tiles; tile += GD_LP_WARPS) {
            const int pos = tile * 32 + lane;
            const gd_src si = gd_lp_sink_at(d, sm, la, min(pos, n_act - 1), G);
            const gd_acc a = gd_lp_tile<EPS0>(sm, si, 0, cnt_own, la.eps2);
            if (pos < n_act) {
                double2 *o = reinterpret_cast<double2 *>(out + (size_t)pos * rs);
                o[0] = make_double2(a.ax, a.ay); o[1] = make_double2(a.az, a.jx); o[2] = make_double2(a.jy, a.jz);
            }
        }
        return;
    }
    const int nsplit = GD_LP_WARPS / tiles;
    const int tile = warp / nsplit, chunk = warp - tile * nsplit;
    const bool work = tile < tiles;
    const int pos = tile * 32 + lane;
    if (work) {
        const gd_src si = gd_lp_sink_at(d, sm, la, min(pos, n_act - 1), G);
        const int jb = (int)((long long)cnt_own * chunk / nsplit), je = (int)((long long)cnt_own * (chunk + 1) / nsplit);
        const gd_acc a = gd_lp_tile<EPS0>(sm, si, jb, je, la.eps2);
        double *r = sm.red + warp * 192 + lane;
        r[0] = a.ax; r[32] = a.ay; r[64] = a.az; r[96] = a.jx; r[128] = a.jy; r[160] = a.jz;
    }
    __syncthreads();
    if (work && chunk == 0 && pos < n_act) {
#pragma unroll
        for (int comp = 0; comp < 6; ++comp) {
            double s = sm.red[warp * 192 + comp * 32 + lane];
            for (int c = 1; c < nsplit; ++c) s += sm.red[(warp + c) * 192 + comp * 32 + lane];
            out[(size_t)pos * rs + comp] = s;
        }
    }
}


// fine-grained phase stamps of a debug build (-DGD_LP_FINE=1): per CTA, thread 0's clock64 deltas of the steps with
// n_act <= GD_LP_FINE_MAX, summed into d.staging as [CTA][16] {cycles x 12, -, -, steps, owner steps}
#ifndef GD_LP_FINE_MAX
#define GD_LP_FINE_MAX 8
#endif
#if GD_LP_FINE
#define GD_STAMP(k) do { if (tid == 0) { const long long c_ = clock64(); if (fine_on) fine[k] += c_ - fine_last; fine_last = c_; } } while (0)
#else
#define GD_STAMP(k) do { } while (0)
#endif

// ---- [correct] -----------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void gd_lp_commit(const gd_dev &d, const gd_lsm &sm, int i, int p, double m, const gd_corrected &r,
                                             const double (&a1)[3], const double (&j1)[3], double h, double t_next)
{
    if (r.flags & 1) atomicAdd(&sm.hist[64], 1u);
    if (r.flags & 2) atomicAdd(&sm.hist[65], 1u);
    const int lvl = gd_step_level(h);
    if (lvl >= 0 && lvl < 64) atomicAdd(&sm.hist[lvl], 1u);
    const double4 xm = make_double4(r.x, r.y, r.z, m), vt = make_double4(r.vx, r.vy, r.vz, t_next);
    const double4 ad = make_double4(a1[0], a1[1], a1[2], r.dt), jk = make_double4(j1[0], j1[1], j1[2], 0.0);
    d.xm[i] = xm; d.vt[i] = vt; d.ad[i] = ad; d.jk[i] = jk;
    if (sm.xm) { sm.xm[p] = xm; sm.vt[p] = vt; sm.ad[p] = ad; sm.jk[p] = jk; }
    const double tn = t_next + r.dt;                         // exact (dyadic)
    d.tnext[i] = tn;
    sm.ts[p] = tn;
}

// small mode: one warp per own active particle.  Lanes stride over the CTAs' partial sums (ascending c within a lane,
// fixed butterfly across lanes); lanes 0..2 then run one Cartesian component of the corrector each; the criterion and
// the block rule are evaluated by every lane on the same values; lane 0 commits.
__device__ __forceinline__ void gd_lp_correct_warp(const gd_dev &d, const gd_lsm &sm, const gd_largs &la, int G, int p0, int pos, int p,
                                                   double t_next, int lane)
{
    const int i = p0 + p;
    const double4 ad = GD_LP_AD(p, i), jk = GD_LP_JK(p, i);
    double s[6] = {0, 0, 0, 0, 0, 0};
    {   // the G rows of this position are contiguous; lane l takes rows l, l + 32, ... (48 bytes each).  Every load in
        // flight at once (branch-free: rows beyond G are re-reads of the lane's first row with weight 0), then added in
        // ascending c
        const double2 *base = reinterpret_cast<const double2 *>(d.partial + (size_t)pos * 6 * G);
        double2 v[GD_LP_MAX_GRID / 32][3];
#pragma unroll
        for (int u = 0; u < GD_LP_MAX_GRID / 32; ++u) {
            const int c = lane + 32 * u;
            const double2 *row = base + 3 * (c < G ? c : lane);
            v[u][0] = __ldcg(row); v[u][1] = __ldcg(row + 1); v[u][2] = __ldcg(row + 2);
        }
#pragma unroll
        for (int u = 0; u < GD_LP_MAX_GRID / 32; ++u) {
            const double wgt = (lane + 32 * u < G) ? 1.0 : 0.0;
            s[0] += wgt * v[u][0].x; s[1] += wgt * v[u][0].y; s[2] += wgt * v[u][1].x;
            s[3] += wgt * v[u][1].y; s[4] += wgt * v[u][2].x; s[5] += wgt * v[u][2].y;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int k = 0; k < 6; ++k) s[k] += __shfl_xor_sync(GD_FULL, s[k], o);
    }
    const double2 pxy = sm.pxy[p], pzm = sm.pzm[p], pvxy = sm.vxy[p];
    const double pvz = sm.vz[p];
    const int comp = lane < 2 ? lane : 2;
    const double xp = comp == 0 ? pxy.x : (comp == 1 ? pxy.y : pzm.x);
    const double vp = comp == 0 ? pvxy.x : (comp == 1 ? pvxy.y : pvz);
    const double a0 = comp == 0 ? ad.x : (comp == 1 ? ad.y : ad.z);
    const double j0 = comp == 0 ? jk.x : (comp == 1 ? jk.y : jk.z);
    const double a1 = comp == 0 ? s[0] : (comp == 1 ? s[1] : s[2]);
    const double j1 = comp == 0 ? s[3] : (comp == 1 ? s[4] : s[5]);
    const double h = ad.w;
    const gd_hpow hp = gd_step_powers(h);
    const gd_corr1 cr = gd_correct_component(xp, vp, a0, j0, a1, j1, hp);
    const double a2x = __shfl_sync(GD_FULL, cr.a2e, 0), a2y = __shfl_sync(GD_FULL, cr.a2e, 1), a2z = __shfl_sync(GD_FULL, cr.a2e, 2);
    const double a3x = __shfl_sync(GD_FULL, cr.a3, 0), a3y = __shfl_sync(GD_FULL, cr.a3, 1), a3z = __shfl_sync(GD_FULL, cr.a3, 2);
    gd_corrected r;
    r.x = __shfl_sync(GD_FULL, cr.xnew, 0); r.y = __shfl_sync(GD_FULL, cr.xnew, 1); r.z = __shfl_sync(GD_FULL, cr.xnew, 2);
    r.vx = __shfl_sync(GD_FULL, cr.vnew, 0); r.vy = __shfl_sync(GD_FULL, cr.vnew, 1); r.vz = __shfl_sync(GD_FULL, cr.vnew, 2);
    const double na1 = gd_norm3(s[0], s[1], s[2]), nj1 = gd_norm3(s[3], s[4], s[5]);
    const double na2 = gd_norm3(a2x, a2y, a2z), na3 = gd_norm3(a3x, a3y, a3z);
    r.dt = gd_new_step(na1, nj1, na2, na3, h, t_next, la.eta, la.dt_min, la.dt_max, la.halving_mode, r.flags);
    if (lane == 0) {
        const double a1v[3] = {s[0], s[1], s[2]}, j1v[3] = {s[3], s[4], s[5]};
        gd_lp_commit(d, sm, i, p, pzm.y, r, a1v, j1v, h, t_next);
    }
}

// big mode: one thread per own active particle; the CTAs' partial sums are added in ascending c
__device__ __forceinline__ void gd_lp_correct_thread(const gd_dev &d, const gd_lsm &sm, const gd_largs &la, int G, int p0, int pos, int p,
                                                     double t_next)
{
    const int i = p0 + p;
    const double4 ad = GD_LP_AD(p, i), jk = GD_LP_JK(p, i);
    double s[6] = {0, 0, 0, 0, 0, 0};
    const double2 *row = reinterpret_cast<const double2 *>(d.partial + (size_t)pos * 6 * G);
    // batches of 16 CTAs: 48 loads in flight, then added in ascending c
    for (int c0 = 0; c0 < G; c0 += 16) {
        double2 v[16][3];
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            const int c = min(c0 + u, G - 1);
#pragma unroll
            for (int k = 0; k < 3; ++k) v[u][k] = __ldcg(row + 3 * c + k);
        }
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            if (c0 + u < G) {
                s[0] += v[u][0].x; s[1] += v[u][0].y; s[2] += v[u][1].x; s[3] += v[u][1].y; s[4] += v[u][2].x; s[5] += v[u][2].y;
            }
        }
    }
    const double2 pxy = sm.pxy[p], pzm = sm.pzm[p], pvxy = sm.vxy[p];
    const double pvz = sm.vz[p];
    const double a1v[3] = {s[0], s[1], s[2]}, j1v[3] = {s[3], s[4], s[5]};
    const gd_corrected r = gd_correct_particle(pxy.x, pxy.y, pzm.x, pvxy.x, pvxy.y, pvz, ad, jk, a1v, j1v, t_next, la.eta, la.dt_min,
                                               la.dt_max, la.halving_mode);
    gd_lp_commit(d, sm, i, p, pzm.y, r, a1v, j1v, ad.w, t_next);
}

// ---------------------------------------------------------------------------------------------------------------------------
// lp_ctl (layout in gd_common.cuh): word GD_LP_CTL_BAR = arrivals at the first hand-off, word GD_LP_CTL_BAR2 = arrivals at
// the second (both monotonic over the life of the context, a 128-byte line each), words GD_LP_CTL_BASE + 1 / + 13 = their
// counts when this launch began, words GD_LP_CTL_BASE + 2 .. + 12 = the counters of gd_get_loop_profile.
// TIMERS: CTA 0 reads %globaltimer around every phase and adds the step to the per-size bins of gd_get_loop_histogram
// (six atomics per block step); without, the loop has no timer reads and no atomics besides the two hand-offs.
template <bool EPS0, bool TIMERS>
__global__ void __launch_bounds__(GD_LP_THREADS, 1)
k_block_loop(gd_dev d, gd_largs la)
{
    extern __shared__ __align__(16) unsigned char gd_lp_smem[];
    gd_ctrl *ct = d.ctrl;
    if (ct->finished) return;                                // nobody writes ct before the first barrier
    const gd_lsm sm = gd_lsm_carve(gd_lp_smem, la.S, la.state);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = gridDim.x, me = blockIdx.x;
    const int p0 = gd_slice_begin(me, la.n, G);
    const int cnt_own = gd_slice_begin(me + 1, la.n, G) - p0;
    const int rounds = (cnt_own + 31) / 32;
    const double t_end = ct->t_end;
    const long long max_steps = ct->max_steps;
    double t_cur = ct->t;
    long long steps = ct->steps, psteps = 0;
    const long long ct_steps0 = steps;
    unsigned long long *bar = d.lp_ctl + GD_LP_CTL_BAR;
    unsigned long long target = d.lp_ctl[GD_LP_CTL_BASE + 1];
    unsigned long long *bar2 = d.lp_ctl + GD_LP_CTL_BAR2, target2 = d.lp_ctl[GD_LP_CTL_BASE + 13];   // second hand-off: only the owners of a step arrive
    double *out = d.partial + (size_t)me * 6;
    const int rs = 6 * G;
    const int r0_tid = gd_slice_begin(tid < G ? tid : 0, la.n, G);   // first row of the segment of CTA `tid` (a 64-bit division: once)

    for (int p = tid; p < rounds * 32; p += GD_LP_THREADS) {
        if (p < cnt_own) {
            sm.ts[p] = d.tnext[p0 + p];
            if (sm.xm) { sm.xm[p] = d.xm[p0 + p]; sm.vt[p] = d.vt[p0 + p]; sm.ad[p] = d.ad[p0 + p]; sm.jk[p] = d.jk[p0 + p]; }
        } else {                                             // zero-mass padding of the last source round
            sm.pxy[p] = make_double2(0.0, 0.0);
            sm.pzm[p] = make_double2(0.0, 0.0);
            sm.vxy[p] = make_double2(0.0, 0.0);
            sm.vz[p] = 0.0;
        }
    }
    if (tid < 66) sm.hist[tid] = 0u;
    for (int k = tid; k <= G; k += GD_LP_THREADS) sm.p0t[k] = gd_slice_begin(k, la.n, G);   // G + 1 entries: G may equal GD_LP_THREADS
    __syncthreads();
    double L_me;
    int cnt_me = gd_publish(d, sm, me, p0, cnt_own, &L_me);
    gd_bar_arrive(bar);
    target += G;
    gd_bar_wait(bar, target);

    bool fin = false;
    unsigned long long tr[4] = {0, 0, 0, 0}, own[3] = {0, 0, 0}, g0 = gd_gtime<TIMERS>(), g1;   // CTA 0's view: ns in [force], barrier, [correct], barrier
    const unsigned long long g_begin = g0;
#if GD_LP_FINE
    long long fine[16] = {0}, fine_last = clock64();
    bool fine_on = false;
#endif
    for (;;) {
        if (t_cur >= t_end || (max_steps >= 0 && steps >= max_steps)) { fin = true; break; }
        // ---- [force] ----
        double Lc = GD_INF;
        int cc = 0;
        if (tid < G) { Lc = __ldcg(d.lp_L + tid); cc = __ldcg(d.lp_cnt + tid); }
        double m = gd_warp_min_d(Lc);
        if (lane == 0) sm.wmin[warp] = m;
        __syncthreads();
        m = gd_warp_min_d(lane < GD_LP_WARPS ? sm.wmin[lane] : GD_INF);
        const double t_next = m;
        GD_STAMP(0);
        const int mine = (tid < G && Lc == t_next) ? cc : 0;
        int incl = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(GD_FULL, incl, o); if (lane >= o) incl += u; }
        if (lane == 31) sm.wcnt[warp] = incl;
        // n_con = CTAs that contribute active particles = the owners of this step.  It must equal the number of CTAs whose
        // `contributing` below is true (they are the arrivals the second hand-off waits for): CTA c publishes lp_cnt[c] > 0
        // exactly when it has candidates at its own minimum L, so (Lc == t_next && cc > 0) here is (L_me == t_next && cnt_me > 0) there.
        const int n_con = __syncthreads_count(mine > 0);
        int wbase = 0, n_act = 0;
#pragma unroll
        for (int w = 0; w < GD_LP_WARPS; ++w) { int c = sm.wcnt[w]; wbase += (w < warp) ? c : 0; n_act += c; }
        if (n_act > la.hi) break;                            // uniform: the stage kernels take this step
#if GD_LP_FINE
        fine_on = n_act <= GD_LP_FINE_MAX;
#endif
        const bool small = n_act <= la.small_hi;
        const int excl = wbase + incl - mine;
        if (tid < G) sm.spre[tid] = excl;
        if (tid == 0) sm.spre[G] = n_act;
        if (small && mine > 0) {
            for (int k = 0; k < mine; ++k) sm.smap[excl + k] = r0_tid + k;
        }
        // small mode: the sink records are fetched (L2) while the own slice is predicted
        constexpr int NPF = (GD_LP_MAX_SMALL * 4 + GD_LP_THREADS - 1) / GD_LP_THREADS;
        double2 pf[NPF];
        if (small) {
            __syncthreads();                                 // smap is complete
#pragma unroll
            for (int u = 0; u < NPF; ++u) {
                const int e = tid + GD_LP_THREADS * u;
                if (e < 4 * n_act) pf[u] = __ldcg(reinterpret_cast<const double2 *>(d.lp_rec) + 4 * (size_t)sm.smap[e >> 2] + (e & 3));
            }
        }
        GD_STAMP(1);
        // own slice predicted to t+
        for (int p = tid; p < cnt_own; p += GD_LP_THREADS) {
            const int i = p0 + p;
            const double4 xm = GD_LP_XM(p, i), vt = GD_LP_VT(p, i), ad = GD_LP_AD(p, i), jk = GD_LP_JK(p, i);
            const gd_pred q = gd_predict_record(xm, vt, ad, jk, t_next);
            sm.pxy[p] = make_double2(q.x, q.y);
            sm.pzm[p] = make_double2(q.z, xm.w);
            sm.vxy[p] = make_double2(q.vx, q.vy);
            sm.vz[p] = q.vz;
        }
        if (small) {
#pragma unroll
            for (int u = 0; u < NPF; ++u) {
                const int e = tid + GD_LP_THREADS * u;
                if (e < 4 * n_act) sm.sink[e] = pf[u];
            }
        }
        __syncthreads();
        GD_STAMP(2);
        if (small) gd_lp_force_small<EPS0>(d, sm, la, out, rs, n_act, rounds);
        else gd_lp_force_big<EPS0>(d, sm, la, out, rs, G, n_act, cnt_own);
        GD_STAMP(3);
        g1 = gd_gtime<TIMERS>(); const unsigned long long d0 = g1 - g0; tr[0] += d0; g0 = g1;
        // first hand-off (all -> owners): every CTA arrives, only the owners of the step have something to wait for
        gd_bar_arrive(bar);
        GD_STAMP(4);
        target += G;
        if ((L_me == t_next) && cnt_me > 0) gd_bar_wait(bar, target);
        GD_STAMP(5);
        g1 = gd_gtime<TIMERS>(); const unsigned long long d1 = g1 - g0; tr[1] += d1; g0 = g1;
        // ---- [correct] + [publish] ----
        const bool contributing = (L_me == t_next) && cnt_me > 0;
        if (contributing) {
            const unsigned long long o0 = gd_gtime<TIMERS>();
            const int pre = sm.spre[me];
            // few own active particles: a warp each (lanes over the CTAs' partial sums); many: a thread each
            if (cnt_me <= la.wc_hi) {
                for (int k = warp; k < cnt_me; k += GD_LP_WARPS) gd_lp_correct_warp(d, sm, la, G, p0, pre + k, sm.lact[k], t_next, lane);
            } else {
                for (int k = tid; k < cnt_me; k += GD_LP_THREADS) gd_lp_correct_thread(d, sm, la, G, p0, pre + k, sm.lact[k], t_next);
            }
            __syncthreads();
            GD_STAMP(6);
            const unsigned long long o1 = gd_gtime<TIMERS>();
            cnt_me = gd_publish(d, sm, me, p0, cnt_own, &L_me);
            GD_STAMP(7);
#if GD_LP_FINE
            if (tid == 0 && fine_on) fine[15] += 1;
#endif
            own[0] += 1; own[1] += o1 - o0; own[2] += gd_gtime<TIMERS>() - o1;
        }
        t_cur = t_next;
        steps += 1;
        psteps += n_act;
        g1 = gd_gtime<TIMERS>(); const unsigned long long d2 = g1 - g0; tr[2] += d2; g0 = g1;
        GD_STAMP(8);
        // second hand-off (owners -> all): only the owners arrive, everybody waits for as many arrivals as the step had
        // owners.  (No CTA is still reading what an owner overwrites: the owner waited for every CTA's first arrival.)
        if (contributing) gd_bar_arrive(bar2);
        GD_STAMP(9);
        target2 += (unsigned long long)n_con;
        gd_bar_wait(bar2, target2);
        GD_STAMP(10);
#if GD_LP_FINE
        if (tid == 0 && fine_on) fine[14] += 1;
#endif
        g1 = gd_gtime<TIMERS>(); const unsigned long long d3 = g1 - g0; tr[3] += d3; g0 = g1;
#if GD_LP_PROFILE
        if (TIMERS && me == 0 && tid == 0) {                            // per-size bins of gd_get_loop_histogram (fire-and-forget REDs)
            unsigned long long *hb = d.lp_prof + 6 * (32 - __clz(n_act));
            atomicAdd(hb, 1ull); atomicAdd(hb + 1, (unsigned long long)n_act);
            atomicAdd(hb + 2, d0); atomicAdd(hb + 3, d1); atomicAdd(hb + 4, d2); atomicAdd(hb + 5, d3);
        }
#endif
    }

#if GD_LP_FINE
    if (tid == 0) for (int k = 0; k < 16; ++k) ((long long *)d.staging)[me * 16 + k] = fine[k];
#endif
    // ---- leave: flush the counters; CTA 0 hands the run state back ----
    if (tid < 64 && sm.hist[tid]) atomicAdd((unsigned long long *)&d.hist[tid], (unsigned long long)sm.hist[tid]);
    if (tid < 2 && sm.hist[64 + tid]) atomicAdd((unsigned long long *)&d.diag[tid], (unsigned long long)sm.hist[64 + tid]);
    if (me == 0 && tid == 0) {
        unsigned long long *const ctl = d.lp_ctl + GD_LP_CTL_BASE;
        ct->t = t_cur;
        ct->steps = steps;
        ct->psteps += psteps;
        if (fin) ct->finished = 1;
        ctl[1] = target;
        ctl[13] = target2;
        // profiling counters: particle steps and block steps taken inside the loop, ns inside it, ns per phase
        ctl[2] += (unsigned long long)psteps;
        ctl[3] += (unsigned long long)(steps - ct_steps0);
        ctl[4] += gd_gtime<TIMERS>() - g_begin;
        for (int k = 0; k < 4; ++k) ctl[5 + k] += tr[k];
        ctl[9] += 1ull;
        for (int k = 0; k < 3; ++k) ctl[10 + k] += own[k];   // CTA 0 as an owner: steps, ns correcting, ns publishing
    }
}

// ---------------------------------------------------------------------------------------------------------------------------
// k_force_slice: the loop's force phase as a stage kernel for gd_force_jerk (steps a3 / a4 with an explicit or the
// internal active list): one CTA per SM takes a slice of the np predicted source records into shared memory and
// evaluates the partial sums of EVERY listed sink against it, with the mappings above.  The partial rows are folded
//   n_act <= 16:  by the last CTA to finish (ticket), a warp per sink over the G contiguous rows of its position;
//   larger:       by k_fold_slice_warp, the same with a warp per sink over the whole machine (one coalesced read each).
// Systems whose 1/G of the source records does not fit in shared memory (C5: 7085 records per SM) are cut into
// T = P G slices instead and CTA c takes the slices c, G + c, ... one after the other (P passes, T partial rows per
// sink): the sinks stay in place, only the slice is reloaded.
// Device-count form (n_act_dev != NULL: the captured block-step graph of systems too large for the persistent loop):
// the active count is read from device memory and the kernel runs only for lo < n_act <= hi.
#define GD_SL_TICKET_MAX 16
#define GD_SL_MAX_PASSES 16
struct gd_sargs {
    int n_act;
    double *a_out, *j_out;           // [n_act,3]
    unsigned int *ticket;
    const long long *n_act_dev;
    int lo, hi;
};

__device__ __forceinline__ bool gd_slice_count(const gd_sargs &sa, int &n_act)
{
    n_act = sa.n_act;
    if (!sa.n_act_dev) return true;
    n_act = (int)__ldcg(sa.n_act_dev);
    return n_act > sa.lo && n_act <= sa.hi;
}

template <bool EPS0>
__global__ void __launch_bounds__(GD_LP_THREADS, 1)
k_force_slice(gd_dev d, gd_largs la, gd_sargs sa)
{
    extern __shared__ __align__(16) unsigned char gd_lp_smem[];
    __shared__ bool s_last;
    const gd_lsm sm = gd_lsm_carve(gd_lp_smem, la.S, 0);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = gridDim.x, me = blockIdx.x, T = G * la.passes;
    int n_act;
    if (!gd_slice_count(sa, n_act)) return;
    const bool small = n_act <= la.small_hi;
    if (small) {
        for (int e = tid; e < 4 * n_act; e += GD_LP_THREADS) {
            const int pos = e >> 2, part = e & 3;
            const int i = la.ext_idx ? __ldg(la.ext_idx + pos) : pos;
            double2 v;
            if (part == 0) v = __ldg(d.pxy + i);
            else if (part == 1) v = __ldg(d.pzm + i);
            else if (part == 2) v = __ldg(d.vxy + i);
            else v = make_double2(__ldg(d.vz + i), 0.0);
            sm.sink[e] = v;
        }
    }
    const size_t ps = (size_t)6 * T;
    for (int pass = 0; pass < la.passes; ++pass) {
        const int sl = pass * G + me;
        const int p0 = gd_slice_begin(sl, la.n, T);
        const int cnt_own = gd_slice_begin(sl + 1, la.n, T) - p0;
        const int rounds = (cnt_own + 31) / 32;
        if (pass) __syncthreads();                           // every warp is done with the previous slice
        for (int p = tid; p < rounds * 32; p += GD_LP_THREADS) {
            const bool in = p < cnt_own;
            sm.pxy[p] = in ? d.pxy[p0 + p] : make_double2(0.0, 0.0);
            sm.pzm[p] = in ? d.pzm[p0 + p] : make_double2(0.0, 0.0);
            sm.vxy[p] = in ? d.vxy[p0 + p] : make_double2(0.0, 0.0);
            sm.vz[p] = in ? d.vz[p0 + p] : 0.0;
        }
        __syncthreads();
        double *out = d.partial + (size_t)sl * 6;
        if (small) gd_lp_force_small<EPS0>(d, sm, la, out, (int)ps, n_act, rounds);
        else gd_lp_force_big<EPS0>(d, sm, la, out, (int)ps, T, n_act, cnt_own);
    }
    if (n_act > GD_SL_TICKET_MAX) return;

    // a handful of sinks: the last CTA to arrive folds; a warp per sink, lanes over the G contiguous rows of its position
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        const unsigned int tk = atomicAdd(sa.ticket, 1u);
        s_last = (tk == (unsigned int)G - 1u);
        if (s_last) *sa.ticket = 0u;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    for (int pos = warp; pos < n_act; pos += GD_LP_WARPS) {
        const double *base = d.partial + (size_t)pos * ps;
        double s[6] = {0, 0, 0, 0, 0, 0};
        for (int c = lane; c < T; c += 32) {
            const double2 *row = reinterpret_cast<const double2 *>(base + (size_t)c * 6);
            const double2 u0 = __ldcg(row), u1 = __ldcg(row + 1), u2 = __ldcg(row + 2);
            s[0] += u0.x; s[1] += u0.y; s[2] += u1.x; s[3] += u1.y; s[4] += u2.x; s[5] += u2.y;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
            for (int k = 0; k < 6; ++k) s[k] += __shfl_xor_sync(GD_FULL, s[k], o);
        }
        if (lane == 0) {
            sa.a_out[3 * (size_t)pos] = s[0]; sa.a_out[3 * (size_t)pos + 1] = s[1]; sa.a_out[3 * (size_t)pos + 2] = s[2];
            sa.j_out[3 * (size_t)pos] = s[3]; sa.j_out[3 * (size_t)pos + 1] = s[4]; sa.j_out[3 * (size_t)pos + 2] = s[5];
        }
    }
}

// partial[pos][c][6] -> a_out, j_out; one warp per sink: lanes stride over the G contiguous rows (G = slices: CTAs x
// passes), GD_LP_MAX_GRID rows in flight at a time, fixed butterfly
__global__ void __launch_bounds__(GD_LP_THREADS)
k_fold_slice_warp(gd_dev d, int G, gd_sargs sa)
{
    const int lane = threadIdx.x & 31, pos = blockIdx.x * GD_LP_WARPS + (threadIdx.x >> 5);
    int n_act;
    if (!gd_slice_count(sa, n_act)) return;
    if (sa.n_act_dev && n_act <= GD_SL_TICKET_MAX) return;   // folded inside k_force_slice
    if (pos >= n_act) return;
    const double2 *base = reinterpret_cast<const double2 *>(d.partial + (size_t)pos * 6 * G);
    double s[6] = {0, 0, 0, 0, 0, 0};
    for (int c0 = 0; c0 < G; c0 += GD_LP_MAX_GRID) {
        double2 v[GD_LP_MAX_GRID / 32][3];
#pragma unroll
        for (int u = 0; u < GD_LP_MAX_GRID / 32; ++u) {
            const int c = c0 + lane + 32 * u;
            const double2 *row = base + 3 * (c < G ? c : lane);
            v[u][0] = __ldcg(row); v[u][1] = __ldcg(row + 1); v[u][2] = __ldcg(row + 2);
        }
#pragma unroll
        for (int u = 0; u < GD_LP_MAX_GRID / 32; ++u) {
            const double wgt = (c0 + lane + 32 * u < G) ? 1.0 : 0.0;
            s[0] += wgt * v[u][0].x; s[1] += wgt * v[u][0].y; s[2] += wgt * v[u][1].x;
            s[3] += wgt * v[u][1].y; s[4] += wgt * v[u][2].x; s[5] += wgt * v[u][2].y;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int k = 0; k < 6; ++k) s[k] += __shfl_xor_sync(GD_FULL, s[k], o);
    }
    if (lane == 0) {
        sa.a_out[3 * (size_t)pos] = s[0]; sa.a_out[3 * (size_t)pos + 1] = s[1]; sa.a_out[3 * (size_t)pos + 2] = s[2];
        sa.j_out[3 * (size_t)pos] = s[3]; sa.j_out[3 * (size_t)pos + 1] = s[4]; sa.j_out[3 * (size_t)pos + 2] = s[5];
    }
}

// ---- host side ------------------------------------------------------------------------------------------------------------
// Geometry: one CTA per SM; S = slice capacity (multiple of 32); hi = largest active set taken, bounded by the option
// `loop_max_nact` and by the partial-sum scratch (grid x 6 x cap doubles).  loop_grid = 0: the loop is not usable
// (slice does not fit in shared memory, or the device cannot co-schedule the grid) and the stage kernels run alone.
// dynamic shared memory a kernel may use: the device's opt-in maximum minus the kernel's static shared memory.  The limit
// is a property of the function, not of a context, so it is raised to that maximum once for every instantiation:
// contexts of different sizes can then coexist.
template <typename K>
static int gd_raise_smem_limit(gd_ctx *c, K kernel, int max_optin, size_t *avail)
{
    cudaFuncAttributes fa;
    GD_CUDA(c, cudaFuncGetAttributes(&fa, kernel));
    const int lim = max_optin - (int)fa.sharedSizeBytes;
    if (lim <= 0) { *avail = 0; return 0; }
    GD_CUDA(c, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, lim));
    if ((size_t)lim < *avail) *avail = (size_t)lim;
    return 0;
}

int gdk_loop_setup(gd_ctx *c)
{
    c->loop_grid = 0;
    int grid = c->sm_count < GD_LP_MAX_GRID ? c->sm_count : GD_LP_MAX_GRID;
    if (grid < 1 || c->loop_max_nact < 1 || c->n > INT_MAX / 2) return 0;
    int64_t S = (c->n + grid - 1) / grid;
    S = (S + 31) / 32 * 32;
    int64_t hi = c->loop_max_nact < c->n ? c->loop_max_nact : c->n;
    int64_t cap = (hi + 31) / 32 * 32;
    if (cap > c->pcap / grid) { cap = c->pcap / grid / 32 * 32; hi = cap; }
    if (hi < 1) return 0;
    int dev = 0, max_smem = 0, coop = 0;
    GD_CUDA(c, cudaGetDevice(&dev));
    GD_CUDA(c, cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    GD_CUDA(c, cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
    size_t avail = (size_t)max_smem;
    if (gd_raise_smem_limit(c, k_block_loop<false, false>, max_smem, &avail) || gd_raise_smem_limit(c, k_block_loop<true, false>, max_smem, &avail) ||
        gd_raise_smem_limit(c, k_block_loop<false, true>, max_smem, &avail) || gd_raise_smem_limit(c, k_block_loop<true, true>, max_smem, &avail))
        return -3;                                           // GD_ECUDA; text already in c->err
    int state = c->loop_state_opt ? 1 : 0;
    size_t bytes = gd_lsm_bytes((int)S, state);
    if (bytes > avail) { state = 0; bytes = gd_lsm_bytes((int)S, 0); }
    if (!coop || bytes > avail) return 0;
    int resident = 0;
    GD_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&resident, k_block_loop<false, true>, GD_LP_THREADS, bytes));
    if (resident < 1) return 0;
    c->loop_grid = grid;
    c->loop_S = (int)S;
    c->loop_hi = (int)hi;
    c->loop_cap = (int)cap;
    c->loop_smem = bytes;
    c->loop_state = state;
    return 0;
}

// enqueue one run of the loop (reads and updates d.ctrl like the dev forms of the stage kernels)
int gdk_loop(gd_ctx *c)
{
    if (c->loop_grid < 1) return 0;
    gd_largs la;
    la.n = (int)c->n;
    la.S = c->loop_S;
    la.hi = c->loop_hi;
    la.cap = c->loop_cap;
    la.state = c->loop_state;
    int64_t sh = c->loop_small_nact < GD_LP_MAX_SMALL ? c->loop_small_nact : GD_LP_MAX_SMALL;
    la.small_hi = (int)(sh < 0 ? 0 : sh);
    la.wc_hi = (int)(c->loop_warp_correct < 0 ? 0 : (c->loop_warp_correct > 4096 ? 4096 : c->loop_warp_correct));
    la.eps2 = c->eps2;
    la.eta = c->eta;
    la.dt_min = c->dt_min;
    la.dt_max = c->dt_max;
    la.halving_mode = c->halving_mode;
    la.passes = 1;
    la.ext = 0;
    la.ext_idx = nullptr;
    void *args[] = {(void *)&c->d, (void *)&la};
    const bool eps0 = c->eps2 < 2.3e-308, timers = GD_LP_PROFILE && c->loop_timers;
    const void *fn = eps0 ? (timers ? (const void *)k_block_loop<true, true> : (const void *)k_block_loop<true, false>)
                          : (timers ? (const void *)k_block_loop<false, true> : (const void *)k_block_loop<false, false>);
    cudaError_t e = cudaLaunchCooperativeKernel(fn, dim3((unsigned)c->loop_grid), dim3(GD_LP_THREADS), args, c->loop_smem, c->stream);
    if (e != cudaSuccess) return gd_fail_cuda(c, e, "k_block_loop");
    c->launches += 1;
    return 0;
}

// ---- k_force_slice: host side -------------------------------------------------------------------------------------------
int gdk_slice_setup(gd_ctx *c)
{
    c->slice_grid = 0;
    int grid = c->sm_count < GD_LP_MAX_GRID ? c->sm_count : GD_LP_MAX_GRID;
    if (grid < 1 || c->n > INT_MAX / 2) return 0;
    int dev = 0, max_smem = 0;
    GD_CUDA(c, cudaGetDevice(&dev));
    GD_CUDA(c, cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    // passes: the fewest slices per CTA whose records fit in shared memory (option `slice_passes` forces a count)
    size_t avail = (size_t)max_smem;
    if (gd_raise_smem_limit(c, k_force_slice<false>, max_smem, &avail) || gd_raise_smem_limit(c, k_force_slice<true>, max_smem, &avail))
        return -3;                                           // GD_ECUDA; text already in c->err
    int64_t S = 0;
    size_t bytes = 0;
    int passes = c->slice_passes_opt > 0 ? (int)c->slice_passes_opt : 1;
    for (;; ++passes) {
        S = (c->n + (int64_t)grid * passes - 1) / ((int64_t)grid * passes);
        S = (S + 31) / 32 * 32;
        bytes = gd_lsm_bytes((int)S, 0);
        if (bytes <= avail) break;
        if (c->slice_passes_opt > 0 || passes >= GD_SL_MAX_PASSES) return 0;
    }
    c->slice_grid = grid;
    c->slice_passes = passes;
    c->slice_S = (int)S;
    c->slice_smem = bytes;
    return 0;
}

// largest active set k_force_slice can take: option `slice_max_nact`, one partial row per (CTA, sink)
int64_t gdk_slice_hi(const gd_ctx *c)
{
    if (c->slice_grid < 1) return 0;
    int64_t hi = c->slice_max_nact < c->np ? c->slice_max_nact : c->np;
    const int64_t cap = c->pcap / ((int64_t)c->slice_grid * c->slice_passes) / 32 * 32;
    return hi < cap ? hi : cap;
}

// dev = false: the host knows n_act (explicit call).  dev = true (captured graph): the count is read from device memory
// (cell[1]) and the kernels run only for 0 < n_act <= n_act (the argument is then the largest set they take).
int gdk_force_slice(gd_ctx *c, const int32_t *idx, int64_t n_act, double *a_out, double *j_out, bool dev)
{
    gd_largs la;
    la.n = (int)c->n;
    la.S = c->slice_S;
    la.passes = c->slice_passes;
    la.hi = (int)n_act;
    la.cap = (int)((n_act + 31) / 32 * 32);
    int64_t sh = c->loop_small_nact < GD_LP_MAX_SMALL ? c->loop_small_nact : GD_LP_MAX_SMALL;
    la.small_hi = (int)(sh < 0 ? 0 : sh);
    la.wc_hi = (int)(c->loop_warp_correct < 0 ? 0 : (c->loop_warp_correct > 4096 ? 4096 : c->loop_warp_correct));
    la.state = 0;
    la.eps2 = c->eps2;
    la.eta = c->eta;
    la.dt_min = c->dt_min;
    la.dt_max = c->dt_max;
    la.halving_mode = c->halving_mode;
    la.ext = 1;
    la.ext_idx = idx;
    gd_sargs sa;
    sa.n_act = (int)n_act;
    sa.a_out = a_out;
    sa.j_out = j_out;
    sa.ticket = c->d.work + 2;
    sa.n_act_dev = dev ? (const long long *)c->d.cell + 1 : nullptr;
    sa.lo = 0;
    sa.hi = (int)n_act;
    if (c->eps2 < 2.3e-308)
        k_force_slice<true><<<c->slice_grid, GD_LP_THREADS, c->slice_smem, c->stream>>>(c->d, la, sa);
    else
        k_force_slice<false><<<c->slice_grid, GD_LP_THREADS, c->slice_smem, c->stream>>>(c->d, la, sa);
    GD_LAUNCH_CHECK(c, "k_force_slice");
    if (n_act > GD_SL_TICKET_MAX) {
        k_fold_slice_warp<<<(unsigned)((n_act + GD_LP_WARPS - 1) / GD_LP_WARPS), GD_LP_THREADS, 0, c->stream>>>(c->d, c->slice_grid * c->slice_passes, sa);
        GD_LAUNCH_CHECK(c, "k_fold_slice_warp");
    }
    return 0;
}
