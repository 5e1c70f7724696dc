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

#define GD_LP_THREADS 256
#define GD_LP_WARPS (GD_LP_THREADS / 32)
#define GD_LP_MAX_GRID 256          // CTAs (one per SM); bounds the shared tables
#define GD_LP_MAX_HI 1024           // largest active set the loop takes

struct gd_largs {
    int np, S, hi;
    double eps2, eta, dt_min, dt_max;
    int halving_mode;
};

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

__device__ __forceinline__ double gd_warp_min_d(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(GD_FULL, v, o));
    return v;
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
    double2 *pxy, *pzm, *vxy;        // [S] predicted records of the own slice (at t+ during [force] / [correct])
    double *vz;                      // [S]
    double *ts;                      // [S] t_i + dt_i of the own slice (+inf beyond np and in the padding)
    int *lact;                       // [S] local indices of the own candidates, ascending
    int *smap;                       // [hi] active list position -> row of `rec`
    double *sL;                      // [GD_LP_MAX_GRID] L_c of every CTA
    int *spre;                       // [GD_LP_MAX_GRID + 1] exclusive prefix of the contributing candidate counts
    double *red;                     // [GD_LP_WARPS][32] warp partial sums of a split evaluation
    double *wmin;                    // [GD_LP_WARPS]
    int *wcnt;                       // [GD_LP_WARPS + 1]
    unsigned int *hist;              // [64] particle steps per level, [64..65] diagnostics
};

__host__ __device__ inline size_t gd_lsm_bytes(int S, int hi)
{
    return (size_t)S * (16 * 3 + 8 + 8 + 4) + (size_t)hi * 4 + GD_LP_MAX_GRID * 8 + (GD_LP_MAX_GRID + 1) * 4 + 4 +
           GD_LP_WARPS * 32 * 8 + GD_LP_WARPS * 8 + (GD_LP_WARPS + 1) * 4 + 4 + 66 * 4 + 64;
}

__device__ __forceinline__ gd_lsm gd_lsm_carve(unsigned char *base, int S, int hi)
{
    gd_lsm s;
    unsigned char *p = base;
    s.pxy = (double2 *)p; p += (size_t)S * 16;
    s.pzm = (double2 *)p; p += (size_t)S * 16;
    s.vxy = (double2 *)p; p += (size_t)S * 16;
    s.vz = (double *)p; p += (size_t)S * 8;
    s.ts = (double *)p; p += (size_t)S * 8;
    s.sL = (double *)p; p += GD_LP_MAX_GRID * 8;
    s.red = (double *)p; p += GD_LP_WARPS * 32 * 8;
    s.wmin = (double *)p; p += GD_LP_WARPS * 8;
    s.lact = (int *)p; p += (size_t)S * 4;
    s.smap = (int *)p; p += (size_t)hi * 4;
    s.spre = (int *)p; p += (GD_LP_MAX_GRID + 1) * 4;
    s.wcnt = (int *)p; p += (GD_LP_WARPS + 1) * 4;
    s.hist = (unsigned int *)p;
    return s;
}

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
    m = sm.wmin[lane & (GD_LP_WARPS - 1)];
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
        const int i = p0 + sm.lact[k];
        const double4 xm = d.xm[i], vt = d.vt[i], ad = d.ad[i], jk = d.jk[i];
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

// ---- [force]: BI sinks (active-list positions pos0 .. pos0 + BI - 1) against the source rounds [r_begin, r_end) -------
// of the own slice; lane l takes source 32 r + l.  Returns the 6 BI per-lane sums in v[b * 6 + {ax, ay, az, jx, jy, jz}].
template <int BI, bool EPS0>
__device__ __forceinline__ void gd_lp_item(const gd_dev &d, const gd_lsm &sm, int pos0, int r_begin, int r_end, int lane,
                                           double eps2, double *v)
{
    gd_src si[BI];
    gd_acc acc[BI];
#pragma unroll
    for (int b = 0; b < BI; ++b) {
        const double2 *row = reinterpret_cast<const double2 *>(d.lp_rec + 2 * (size_t)sm.smap[pos0 + b]);
        const double2 xy = __ldcg(row), zi = __ldcg(row + 1), wxy = __ldcg(row + 2), wz = __ldcg(row + 3);
        si[b] = gd_src{xy.x, xy.y, zi.x, 0.0, wxy.x, wxy.y, wz.x};
        acc[b] = gd_acc{0, 0, 0, 0, 0, 0};
    }
#pragma unroll 2
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

// One work item = a register block of sinks: items 0 .. n4 - 1 hold 4 sinks, the n_act % 4 last ones hold 1.
// items >= warps: warp w takes items w, w + 8, ... over all source rounds and writes partial[me][pos][6] itself.
// items <  warps: the rounds of every item are split over nsplit = 8 / items warps; the warp sums meet in shared
//                 memory and are added in chunk order.
template <bool EPS0>
__device__ __forceinline__ void gd_lp_force(const gd_dev &d, const gd_lsm &sm, const gd_largs &la, int me, int n_act, int rounds)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n4 = n_act >> 2, items = n4 + (n_act & 3);
    double *out = d.partial + (size_t)me * la.hi * 6;
    if (items >= GD_LP_WARPS) {
        for (int it = warp; it < items; it += GD_LP_WARPS) {
            if (it < n4) {
                double v[24];
                gd_lp_item<4, EPS0>(d, sm, 4 * it, 0, rounds, lane, la.eps2, v);
                gd_rs24(v, lane);
                const int e = gd_rs24_elem(lane);
                if (e >= 0) out[(size_t)(4 * it) * 6 + e] = v[0];
            } else {
                double v[6];
                const int pos = 4 * n4 + (it - n4);
                gd_lp_item<1, EPS0>(d, sm, pos, 0, rounds, lane, la.eps2, v);
                gd_rs6(v, lane);
                const int e = gd_rs6_elem(lane);
                if (e >= 0) out[(size_t)pos * 6 + e] = v[0];
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
        const int rb = (int)((long long)rounds * chunk / nsplit), re = (int)((long long)rounds * (chunk + 1) / nsplit);
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
        out[(size_t)pos * 6 + lane] = s;
    }
}

// ---- [correct]: one warp per own active particle -------------------------------------------------------------------------
// Lanes stride over the CTAs' partial rows (ascending c within a lane, fixed butterfly across lanes); lanes 0..2
// then run one Cartesian component of the corrector each; the criterion and the block rule are evaluated by every
// lane on the same values; lane 0 commits.
__device__ __forceinline__ void gd_lp_correct(const gd_dev &d, const gd_lsm &sm, const gd_largs &la, int G, int p0, int pos, int p,
                                              double t_next, int lane)
{
    double s[6] = {0, 0, 0, 0, 0, 0};
    for (int c = lane; c < G; c += 32) {
        const double2 *row = reinterpret_cast<const double2 *>(d.partial + ((size_t)c * la.hi + pos) * 6);
        const double2 u0 = __ldcg(row), u1 = __ldcg(row + 1), u2 = __ldcg(row + 2);
        s[0] += u0.x; s[1] += u0.y; s[2] += u1.x; s[3] += u1.y; s[4] += u2.x; s[5] += u2.y;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int k = 0; k < 6; ++k) s[k] += __shfl_xor_sync(GD_FULL, s[k], o);
    }
    const int i = p0 + p;
    const double4 ad = d.ad[i], jk = d.jk[i];
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
    const double xn = __shfl_sync(GD_FULL, cr.xnew, 0), yn = __shfl_sync(GD_FULL, cr.xnew, 1), zn = __shfl_sync(GD_FULL, cr.xnew, 2);
    const double vxn = __shfl_sync(GD_FULL, cr.vnew, 0), vyn = __shfl_sync(GD_FULL, cr.vnew, 1), vzn = __shfl_sync(GD_FULL, cr.vnew, 2);
    const double na1 = gd_norm3(s[0], s[1], s[2]), nj1 = gd_norm3(s[3], s[4], s[5]);
    const double na2 = gd_norm3(a2x, a2y, a2z), na3 = gd_norm3(a3x, a3y, a3z);
    int flags;
    const double dnew = gd_new_step(na1, nj1, na2, na3, h, t_next, la.eta, la.dt_min, la.dt_max, la.halving_mode, flags);
    if (lane == 0) {
        if (flags & 1) atomicAdd(&sm.hist[64], 1u);
        if (flags & 2) atomicAdd(&sm.hist[65], 1u);
        const int lvl = gd_step_level(h);
        if (lvl >= 0 && lvl < 64) atomicAdd(&sm.hist[lvl], 1u);
        d.xm[i] = make_double4(xn, yn, zn, pzm.y);
        d.vt[i] = make_double4(vxn, vyn, vzn, t_next);
        d.ad[i] = make_double4(s[0], s[1], s[2], dnew);
        d.jk[i] = make_double4(s[3], s[4], s[5], 0.0);
        const double tn = t_next + dnew;                     // exact (dyadic)
        d.tnext[i] = tn;
        sm.ts[p] = tn;
    }
}

// ---------------------------------------------------------------------------------------------------------------------------
// lp_ctl[0] = barrier arrivals (monotonic over the life of the context), lp_ctl[1] = arrivals when this launch began.
template <bool EPS0>
__global__ void __launch_bounds__(GD_LP_THREADS, 1)
k_block_loop(gd_dev d, gd_largs la)
{
    extern __shared__ __align__(16) unsigned char gd_lp_smem[];
    gd_ctrl *ct = d.ctrl;
    if (ct->finished) return;                                // nobody writes ct before the first barrier
    const gd_lsm sm = gd_lsm_carve(gd_lp_smem, la.S, la.hi);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = gridDim.x, me = blockIdx.x;
    const int p0 = me * la.S;
    const int cnt_own = max(0, min(la.S, la.np - p0));       // multiple of 32
    const int rounds = cnt_own / 32;
    const double t_end = ct->t_end;
    const long long max_steps = ct->max_steps;
    double t_cur = ct->t;
    long long steps = ct->steps, psteps = 0;
    unsigned long long *bar = d.lp_ctl;
    unsigned long long target = d.lp_ctl[1];

    for (int p = tid; p < cnt_own; p += GD_LP_THREADS) sm.ts[p] = d.tnext[p0 + p];
    if (tid < 66) sm.hist[tid] = 0u;
    __syncthreads();
    double L_me;
    int cnt_me = gd_publish(d, sm, me, p0, cnt_own, &L_me);
    gd_bar_arrive(bar);
    target += G;
    gd_bar_wait(bar, target);

    bool fin = false;
    for (;;) {
        if (t_cur >= t_end || (max_steps >= 0 && steps >= max_steps)) { fin = true; break; }
        // ---- [force] ----
        double Lc = GD_INF;
        int cc = 0;
        if (tid < G) { Lc = __ldcg(d.lp_L + tid); cc = __ldcg(d.lp_cnt + tid); }
        double m = gd_warp_min_d(Lc);
        if (lane == 0) sm.wmin[warp] = m;
        __syncthreads();
        m = gd_warp_min_d(sm.wmin[lane & (GD_LP_WARPS - 1)]);
        const double t_next = m;
        const int mine = (tid < G && Lc == t_next) ? cc : 0;
        int incl = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(GD_FULL, incl, o); if (lane >= o) incl += u; }
        if (lane == 31) sm.wcnt[warp] = incl;
        __syncthreads();
        int wbase = 0, n_act = 0;
#pragma unroll
        for (int w = 0; w < GD_LP_WARPS; ++w) { int c = sm.wcnt[w]; wbase += (w < warp) ? c : 0; n_act += c; }
        if (n_act > la.hi) break;                            // uniform: the stage kernels take this step
        const int excl = wbase + incl - mine;
        if (tid < G) sm.spre[tid] = excl;
        for (int k = 0; k < mine; ++k) sm.smap[excl + k] = tid * la.S + k;
        // own slice predicted to t+
        for (int p = tid; p < cnt_own; p += GD_LP_THREADS) {
            const int i = p0 + p;
            const double4 xm = d.xm[i], vt = d.vt[i], ad = d.ad[i], jk = d.jk[i];
            const gd_pred q = gd_predict_record(xm, vt, ad, jk, t_next);
            sm.pxy[p] = make_double2(q.x, q.y);
            sm.pzm[p] = make_double2(q.z, xm.w);
            sm.vxy[p] = make_double2(q.vx, q.vy);
            sm.vz[p] = q.vz;
        }
        __syncthreads();
        gd_lp_force<EPS0>(d, sm, la, me, n_act, rounds);
        gd_bar_arrive(bar);
        target += G;
        gd_bar_wait(bar, target);
        // ---- [correct] + [publish] ----
        const bool contributing = (L_me == t_next) && cnt_me > 0;
        if (contributing) {
            const int pre = sm.spre[me];
            for (int k = warp; k < cnt_me; k += GD_LP_WARPS) gd_lp_correct(d, sm, la, G, p0, pre + k, sm.lact[k], t_next, lane);
            __syncthreads();
            cnt_me = gd_publish(d, sm, me, p0, cnt_own, &L_me);
        }
        t_cur = t_next;
        steps += 1;
        psteps += n_act;
        gd_bar_arrive(bar);
        target += G;
        gd_bar_wait(bar, target);
    }

    // ---- leave: flush the counters; CTA 0 hands the run state back ----
    if (tid < 64 && sm.hist[tid]) atomicAdd((unsigned long long *)&d.hist[tid], (unsigned long long)sm.hist[tid]);
    if (tid < 2 && sm.hist[64 + tid]) atomicAdd((unsigned long long *)&d.diag[tid], (unsigned long long)sm.hist[64 + tid]);
    if (me == 0 && tid == 0) {
        ct->t = t_cur;
        ct->steps = steps;
        ct->psteps += psteps;
        if (fin) ct->finished = 1;
        d.lp_ctl[1] = target;
        d.lp_ctl[2] += (unsigned long long)psteps;           // particle steps taken inside the loop (profiling)
    }
}

// ---- host side ------------------------------------------------------------------------------------------------------------
// Geometry: one CTA per SM; S = slice length (multiple of 32); hi = largest active set taken, bounded by the option
// `loop_max_nact`, the partial-sum scratch (grid x hi rows) and GD_LP_MAX_HI.  loop_grid = 0: the loop is not usable
// (slice does not fit in shared memory, or the device cannot co-schedule the grid) and the stage kernels run alone.
int gdk_loop_setup(gd_ctx *c)
{
    c->loop_grid = 0;
    int grid = c->sm_count < GD_LP_MAX_GRID ? c->sm_count : GD_LP_MAX_GRID;
    if (grid < 1 || c->loop_max_nact < 1) return 0;
    int64_t S = (c->np + grid - 1) / grid;
    S = (S + 31) / 32 * 32;
    if (S * grid > c->np + GD_LP_REC_SLACK) return 0;
    int64_t hi = c->loop_max_nact;
    if (hi > GD_LP_MAX_HI) hi = GD_LP_MAX_HI;
    if (hi > c->pcap / grid) hi = c->pcap / grid;
    if (hi < 1) return 0;
    int dev = 0, max_smem = 0, coop = 0;
    GD_CUDA(c, cudaGetDevice(&dev));
    GD_CUDA(c, cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    GD_CUDA(c, cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
    const size_t bytes = gd_lsm_bytes((int)S, (int)hi);
    if (!coop || bytes > (size_t)max_smem) return 0;
    GD_CUDA(c, cudaFuncSetAttribute(k_block_loop<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    GD_CUDA(c, cudaFuncSetAttribute(k_block_loop<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    int resident = 0;
    GD_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&resident, k_block_loop<false>, GD_LP_THREADS, bytes));
    if (resident < 1) return 0;
    c->loop_grid = grid;
    c->loop_S = (int)S;
    c->loop_hi = (int)hi;
    c->loop_smem = bytes;
    return 0;
}

// enqueue one run of the loop (reads and updates d.ctrl like the dev forms of the stage kernels)
int gdk_loop(gd_ctx *c)
{
    if (c->loop_grid < 1) return 0;
    gd_largs la;
    la.np = (int)c->np;
    la.S = c->loop_S;
    la.hi = c->loop_hi;
    la.eps2 = c->eps2;
    la.eta = c->eta;
    la.dt_min = c->dt_min;
    la.dt_max = c->dt_max;
    la.halving_mode = c->halving_mode;
    void *args[] = {(void *)&c->d, (void *)&la};
    const void *fn = (c->eps2 < 2.3e-308) ? (const void *)k_block_loop<true> : (const void *)k_block_loop<false>;
    cudaError_t e = cudaLaunchCooperativeKernel(fn, dim3((unsigned)c->loop_grid), dim3(GD_LP_THREADS), args, c->loop_smem, c->stream);
    if (e != cudaSuccess) return gd_fail_cuda(c, e, "k_block_loop");
    c->launches += 1;
    return 0;
}
