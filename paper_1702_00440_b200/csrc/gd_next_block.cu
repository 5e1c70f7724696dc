// gd_next_block.cu -- active-set selection (step v; Fig. 2):
//   t_next = min_i (t_i + dt_i) ;  active = { i ascending : t_i + dt_i == t_next }
// Times are exact dyadic doubles, so the comparison is exact and the result is unique (R13, R20).
//
// Large systems: two kernels, both bandwidth/latency bound at 8 B per particle each (small systems: the
// single-CTA k_block_select below):
//   k_block_min      grid-wide minimum of tnext[]; the last block to finish (ticket) folds the per-block minima
//   k_block_compact  stream compaction by warp ballot + prefix sums: each block counts its flags, publishes
//                    the count, sums the counts of all lower-numbered blocks, and writes its indices in order.
// Block numbers are handed out by an atomic ticket, so a block only ever waits for blocks that already run.
// Tickets are re-armed by the last block to take one; aggregates carry a launch epoch that k_block_min advances
// in device memory, so that both kernels can be replayed from a captured graph with frozen arguments.
// dev != 0 (block-step graph): k_block_min also decides whether the run is over (gd_ctrl) and, if it is, marks it
// finished and publishes an empty active list; every later kernel of the graph then does nothing.
#include "gd_common.cuh"
#include <stdio.h>

__device__ __forceinline__ double gd_warp_min(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

__global__ void __launch_bounds__(GD_SCAN_THREADS)
k_block_min(gd_dev d, int64_t np, int per_block, int dev)
{
    if (dev && d.ctrl->finished) return;
    __shared__ double s_min[GD_SCAN_THREADS / 32];
    __shared__ bool s_last;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t begin = (int64_t)blockIdx.x * per_block;
    const int64_t end = min(np, begin + per_block);
    double m = __longlong_as_double(0x7ff0000000000000LL);
    for (int64_t i = begin + tid; i < end; i += GD_SCAN_THREADS) m = fmin(m, d.tnext[i]);
    m = gd_warp_min(m);
    if (lane == 0) s_min[warp] = m;
    __syncthreads();
    if (warp == 0) {
        m = s_min[lane];
        m = gd_warp_min(m);
        if (lane == 0) {
            d.blockmin[blockIdx.x] = m;
            __threadfence();
            unsigned int tk = atomicAdd(&d.ticket[0], 1u);
            s_last = (tk == gridDim.x - 1);
            if (s_last) d.ticket[0] = 0u;                        // every block has arrived: re-arm
        }
    }
    __syncthreads();
    if (s_last) {
        __threadfence();
        m = __longlong_as_double(0x7ff0000000000000LL);
        for (int b = tid; b < (int)gridDim.x; b += GD_SCAN_THREADS) m = fmin(m, __ldcg(d.blockmin + b));
        m = gd_warp_min(m);
        if (lane == 0) s_min[warp] = m;
        __syncthreads();
        if (warp == 0) {
            m = gd_warp_min(s_min[lane]);
            if (lane == 0) {
                unsigned int ep = d.ticket[2] + 1u;
                d.ticket[2] = ep ? ep : 1u;                      // epoch of this scan; 0 = freshly cleared scratch
                gd_ctrl *ct = d.ctrl;
                if (dev && (ct->t >= ct->t_end || (ct->max_steps >= 0 && ct->steps >= ct->max_steps))) {
                    ct->finished = 1;
                    ((long long *)d.cell)[1] = 0;                // empty active list: the force and corrector kernels fall through
                } else {
                    d.cell[0] = m;
                }
            }
        }
    }
}

// per_block <= 32 * GD_SCAN_THREADS: every thread keeps its flags in one 32-bit mask
__global__ void __launch_bounds__(GD_SCAN_THREADS)
k_block_compact(gd_dev d, int64_t np, int per_block, int dev)
{
    if (dev && d.ctrl->finished) return;
    __shared__ unsigned int s_bid;
    __shared__ int s_warp[GD_SCAN_THREADS / 32];
    __shared__ int s_round_base[33];
    __shared__ int s_prefix;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) {
        s_bid = atomicAdd(&d.ticket[1], 1u);
        if (s_bid == gridDim.x - 1) d.ticket[1] = 0u;            // every block has its number: re-arm
    }
    __syncthreads();
    const unsigned int bid = s_bid;
    const unsigned int epoch = d.ticket[2];
    const double t_next = d.cell[0];
    const int64_t begin = (int64_t)bid * per_block;
    const int64_t end = min(np, begin + per_block);
    // k_block_min left the minimum of this very range in blockmin[bid] (same geometry): a range whose minimum is not
    // t_next holds no active particle and is not read again -- under block time steps that is almost every range
    const bool any = __ldcg(d.blockmin + bid) == t_next;
    const int rounds = any ? (int)((end - begin + GD_SCAN_THREADS - 1) / GD_SCAN_THREADS) : 0;

    // pass 1: flags and per-round counts
    unsigned int mask = 0;
    int total = 0;
    for (int r = 0; r < rounds; ++r) {
        int64_t i = begin + (int64_t)r * GD_SCAN_THREADS + tid;
        bool f = (i < end) && (d.tnext[i] == t_next);
        mask |= (f ? 1u : 0u) << r;
        unsigned int bal = __ballot_sync(0xffffffffu, f);
        if (lane == 0) s_warp[warp] = __popc(bal);
        __syncthreads();
        if (warp == 0) {
            int v = s_warp[lane];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) s_round_base[r] = v;
        }
        __syncthreads();
    }
    if (tid == 0) {
        int run = 0;
        for (int r = 0; r < rounds; ++r) { int v = s_round_base[r]; s_round_base[r] = run; run += v; }
        s_round_base[32] = run;
        // publish this block's count, tagged with the epoch (one 64-bit store: never torn)
        atomicExch(&d.agg[bid], ((unsigned long long)epoch << 32) | (unsigned int)run);
    }
    __syncthreads();
    total = s_round_base[32];

    // exclusive prefix over the lower-numbered blocks: wait for their aggregates (they are already running)
    if (warp == 0) {
        int sum = 0;
        for (unsigned int p = lane; p < bid; p += 32) {
            unsigned long long v;
            do { v = *((volatile unsigned long long *)&d.agg[p]); } while ((unsigned int)(v >> 32) != epoch);
            sum += (int)(unsigned int)v;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
        if (lane == 0) s_prefix = sum;
    }
    __syncthreads();
    const int prefix = s_prefix;

    // pass 2: ordered scatter
    for (int r = 0; r < rounds; ++r) {
        bool f = (mask >> r) & 1u;
        unsigned int bal = __ballot_sync(0xffffffffu, f);
        if (lane == 0) s_warp[warp] = __popc(bal);
        __syncthreads();
        if (warp == 0) {
            int v = s_warp[lane], incl = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += u; }
            s_warp[lane] = incl - v;
        }
        __syncthreads();
        if (f) {
            int pos = prefix + s_round_base[r] + s_warp[warp] + __popc(bal & ((1u << lane) - 1u));
            d.idx[pos] = (int32_t)(begin + (int64_t)r * GD_SCAN_THREADS + tid);
        }
        __syncthreads();
    }
    if (bid == gridDim.x - 1 && tid == 0) ((long long *)d.cell)[1] = (long long)(prefix + total);
}

// ---------------------------------------------------------------------------------------------------------
// Small systems (np <= 1024 * 64): one CTA does both passes -- no tickets, no fences, one launch.  Thread t owns the
// contiguous chunk [t * R, (t + 1) * R) of tnext (vector loads of whole lines), so the ascending order of the
// active list is the thread order: block minimum, per-thread match counts, one block-wide exclusive scan, ordered
// writes.  KEEP holds the chunk in registers between the passes; otherwise the second pass re-reads it from L2.
template <int R, bool KEEP>
__global__ void __launch_bounds__(GD_SCAN_THREADS)
k_block_select(gd_dev d, int64_t np, int dev)
{
    __shared__ double s_min[32];
    __shared__ int s_cnt[32];
    if (dev && d.ctrl->finished) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t base = (int64_t)tid * R;
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    double v[KEEP ? R : 1];
    double m = inf;
#pragma unroll
    for (int k = 0; k < R; k += 2) {
        double2 x = (base + k < np) ? __ldcg(reinterpret_cast<const double2 *>(d.tnext + base + k)) : make_double2(inf, inf);
        if (KEEP) { v[k] = x.x; v[k + 1] = x.y; }
        m = fmin(m, fmin(x.x, x.y));
    }
    m = gd_warp_min(m);
    if (lane == 0) s_min[warp] = m;
    __syncthreads();
    m = gd_warp_min(s_min[lane]);                                // every warp folds the 32 warp minima itself

    unsigned long long mask = 0ull;                              // R <= 64 match flags of this thread's chunk
#pragma unroll
    for (int k = 0; k < R; k += 2) {
        double2 x;
        if (KEEP) x = make_double2(v[k], v[k + 1]);
        else x = (base + k < np) ? __ldcg(reinterpret_cast<const double2 *>(d.tnext + base + k)) : make_double2(inf, inf);
        mask |= (unsigned long long)(x.x == m) << k;
        mask |= (unsigned long long)(x.y == m) << (k + 1);
    }
    const int cnt = __popcll(mask);
    int incl = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += u; }
    if (lane == 31) s_cnt[warp] = incl;
    __syncthreads();
    int wsum = s_cnt[lane], wincl = wsum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(0xffffffffu, wincl, o); if (lane >= o) wincl += u; }
    const int total = __shfl_sync(0xffffffffu, wincl, 31);
    int pos = __shfl_sync(0xffffffffu, wincl - wsum, warp) + incl - cnt;     // exclusive prefix of this thread

    bool stop = false;
    if (dev) {
        const gd_ctrl *ct = d.ctrl;
        stop = ct->t >= ct->t_end || (ct->max_steps >= 0 && ct->steps >= ct->max_steps);
    }
    if (!stop) {
        while (mask) {
            int k = __ffsll((long long)mask) - 1;
            mask &= mask - 1;
            d.idx[pos++] = (int32_t)(base + k);
        }
    }
    if (tid == 0) {
        if (stop) {
            d.ctrl->finished = 1;
            ((long long *)d.cell)[1] = 0;
        } else {
            d.cell[0] = m;
            ((long long *)d.cell)[1] = (long long)total;
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// Mid-size systems (up to sm_count x 1024 x 16 particles: C4, C5): ONE cooperative kernel, one CTA per SM, tnext read
// once.  Thread t of block b owns the contiguous chunk [(b 1024 + t) R, +R) and keeps it in registers:
//   block minimum -> one 64-bit atomic per block on the grid minimum (non-negative doubles order like their bit patterns; the
//   word holds the COMPLEMENT under atomicMax, so that its rest state is the zero the scratch is cleared to) -> grid
//   barrier (arrival counter: the launch is cooperative, every block is resident) -> match flags from the registers ->
//   block-wide exclusive scan -> the block's count goes to agg[b] with the epoch, the counts of the lower blocks are
//   waited for -> ordered writes.  The last block to finish re-arms the counters.
// The result {t_next, n_act} also goes straight to the caller's pinned host words (host_cell, mapped): gd_next_block
// then needs one launch and one stream synchronisation, no copy.
template <int R>
__global__ void __launch_bounds__(GD_SCAN_THREADS, 1)
k_block_one(gd_dev d, int64_t np, int dev, double *host_cell)
{
    __shared__ double s_min[32];
    __shared__ int s_cnt[32];
    __shared__ int s_prefix;
    __shared__ double s_t;
    if (dev && d.ctrl->finished) return;                         // set only behind the grid barrier below: uniform
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned int bid = blockIdx.x, G = gridDim.x;
    const int64_t base = ((int64_t)bid * GD_SCAN_THREADS + tid) * R;
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    unsigned long long *gmax = reinterpret_cast<unsigned long long *>(d.blockmin + GD_SCAN_MAX_BLOCKS - 1);
    const unsigned int epoch = d.ticket[2] + 1u ? d.ticket[2] + 1u : 1u;     // read before the barrier, advanced behind it
    bool stop = false;
    if (dev) {
        const gd_ctrl *ct = d.ctrl;
        stop = ct->t >= ct->t_end || (ct->max_steps >= 0 && ct->steps >= ct->max_steps);
    }
    double v[R];
    double m = inf;
#pragma unroll
    for (int k = 0; k < R; k += 2) {
        const double2 x = (base + k < np) ? __ldcg(reinterpret_cast<const double2 *>(d.tnext + base + k)) : make_double2(inf, inf);
        v[k] = x.x; v[k + 1] = x.y;
        m = fmin(m, fmin(x.x, x.y));
    }
    m = gd_warp_min(m);
    if (lane == 0) s_min[warp] = m;
    __syncthreads();
    if (warp == 0) {
        m = gd_warp_min(s_min[lane]);
        if (lane == 0) {
            atomicMax(gmax, ~(unsigned long long)__double_as_longlong(m));
            __threadfence();
            atomicAdd(&d.ticket[0], 1u);
            unsigned int seen;
            do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(d.ticket) : "memory"); } while (seen < G);
            s_t = __longlong_as_double((long long)~__ldcg(gmax));
        }
    }
    __syncthreads();
    const double t_next = s_t;

    unsigned int mask = 0u;                                      // R <= 16 match flags of this thread's chunk
#pragma unroll
    for (int k = 0; k < R; ++k) mask |= (unsigned int)(v[k] == t_next) << k;
    const int cnt = stop ? 0 : __popc(mask);
    int incl = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += u; }
    if (lane == 31) s_cnt[warp] = incl;
    __syncthreads();
    int wsum = s_cnt[lane], wincl = wsum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(0xffffffffu, wincl, o); if (lane >= o) wincl += u; }
    const int total = __shfl_sync(0xffffffffu, wincl, 31);
    int pos = __shfl_sync(0xffffffffu, wincl - wsum, warp) + incl - cnt;     // exclusive prefix of this thread inside the block
    if (tid == 0) atomicExch(&d.agg[bid], ((unsigned long long)epoch << 32) | (unsigned int)total);
    if (warp == 0) {                                             // counts of the lower-numbered blocks (all resident)
        int sum = 0;
        for (unsigned int p = lane; p < bid; p += 32) {
            unsigned long long a;
            do { a = *((volatile unsigned long long *)&d.agg[p]); } while ((unsigned int)(a >> 32) != epoch);
            sum += (int)(unsigned int)a;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
        if (lane == 0) s_prefix = sum;
    }
    __syncthreads();
    pos += s_prefix;
    if (!stop) {
        while (mask) {
            const int k = __ffs((int)mask) - 1;
            mask &= mask - 1;
            d.idx[pos++] = (int32_t)(base + k);
        }
    }
    if (tid == 0) {
        if (bid == G - 1) {                                      // the highest block knows the whole count
            if (stop) {
                d.ctrl->finished = 1;
                ((long long *)d.cell)[1] = 0;
            } else {
                const long long n_act = (long long)(s_prefix + total);
                d.cell[0] = t_next;
                ((long long *)d.cell)[1] = n_act;
                if (host_cell) { host_cell[0] = t_next; ((long long *)host_cell)[1] = n_act; }
            }
        }
        __threadfence();
        if (atomicAdd(&d.ticket[1], 1u) == G - 1) {              // every block is through: re-arm for the next launch
            d.ticket[0] = 0u;
            d.ticket[1] = 0u;
            d.ticket[2] = epoch;
            *gmax = 0ull;
        }
    }
}

template <int R>
static int gd_launch_block_one(gd_ctx *c, int blocks, bool dev, double *host_cell)
{
    int dv = dev ? 1 : 0;
    int64_t np = c->np;
    void *args[] = {(void *)&c->d, (void *)&np, (void *)&dv, (void *)&host_cell};
    cudaError_t e = cudaLaunchCooperativeKernel((const void *)k_block_one<R>, dim3((unsigned)blocks), dim3(GD_SCAN_THREADS), args, 0, c->stream);
    if (e != cudaSuccess) return gd_fail_cuda(c, e, "k_block_one");
    c->launches += 1;
    return 0;
}

// host_cell: device-side address of the caller's pinned {t_next, n_act} words, or NULL (graph path; kernels that cannot write it)
int gdk_next_block(gd_ctx *c, bool dev, double *host_cell, bool *wrote_host)
{
    if (wrote_host) *wrote_host = false;
    if (c->np > 64 * GD_SCAN_THREADS && c->coop && c->np <= (int64_t)c->sm_count * GD_SCAN_THREADS * 16) {
        const int64_t per_sm = (c->np + (int64_t)c->sm_count * GD_SCAN_THREADS - 1) / ((int64_t)c->sm_count * GD_SCAN_THREADS);
        const int R = per_sm <= 4 ? 4 : (per_sm <= 8 ? 8 : 16);
        const int blocks = (int)((c->np + (int64_t)GD_SCAN_THREADS * R - 1) / ((int64_t)GD_SCAN_THREADS * R));
        if (wrote_host) *wrote_host = host_cell != nullptr;
        if (R == 4) return gd_launch_block_one<4>(c, blocks, dev, host_cell);
        if (R == 8) return gd_launch_block_one<8>(c, blocks, dev, host_cell);
        return gd_launch_block_one<16>(c, blocks, dev, host_cell);
    }
    if (c->np <= 64 * GD_SCAN_THREADS) {
        const int dv = dev ? 1 : 0;
        if (c->np <= 4 * GD_SCAN_THREADS) k_block_select<4, true><<<1, GD_SCAN_THREADS, 0, c->stream>>>(c->d, c->np, dv);
        else if (c->np <= 16 * GD_SCAN_THREADS) k_block_select<16, true><<<1, GD_SCAN_THREADS, 0, c->stream>>>(c->d, c->np, dv);
        else k_block_select<64, false><<<1, GD_SCAN_THREADS, 0, c->stream>>>(c->d, c->np, dv);
        GD_LAUNCH_CHECK(c, "k_block_select");
        return 0;
    }
    // contiguous ranges of whole 1024-element rounds; at most 32 rounds per block
    int64_t rounds_total = (c->np + GD_SCAN_THREADS - 1) / GD_SCAN_THREADS;
    int64_t blocks = rounds_total < 2 * c->sm_count ? rounds_total : 2 * c->sm_count;
    if (blocks > GD_SCAN_MAX_BLOCKS) blocks = GD_SCAN_MAX_BLOCKS;
    int64_t rounds_per_block = (rounds_total + blocks - 1) / blocks;
    if (rounds_per_block > 32) {
        rounds_per_block = 32;
        blocks = (rounds_total + 31) / 32;
        if (blocks > GD_SCAN_MAX_BLOCKS) {
            snprintf(c->err, sizeof c->err, "next_block: n too large for the scan scratch");
            return -1;
        }
    }
    blocks = (rounds_total + rounds_per_block - 1) / rounds_per_block;
    int per_block = (int)(rounds_per_block * GD_SCAN_THREADS);

    k_block_min<<<(unsigned)blocks, GD_SCAN_THREADS, 0, c->stream>>>(c->d, c->np, per_block, dev ? 1 : 0);
    GD_LAUNCH_CHECK(c, "k_block_min");
    k_block_compact<<<(unsigned)blocks, GD_SCAN_THREADS, 0, c->stream>>>(c->d, c->np, per_block, dev ? 1 : 0);
    GD_LAUNCH_CHECK(c, "k_block_compact");
    return 0;
}
