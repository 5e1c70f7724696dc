// gd_next_block.cu -- active-set selection (step v; Fig. 2):
//   t_next = min_i (t_i + dt_i) ;  active = { i ascending : t_i + dt_i == t_next }
// Times are exact dyadic doubles, so the comparison is exact and the result is unique (R13, R20).
//
// Two kernels, both bandwidth/latency bound at 8 B per particle each:
//   k_block_min      grid-wide minimum of tnext[]; the last block to finish (ticket) folds the per-block minima
//   k_block_compact  stream compaction by warp ballot + prefix sums: each block counts its flags, publishes
//                    the count, sums the counts of all lower-numbered blocks, and writes its indices in order.
// Block numbers are handed out by an atomic ticket, so a block only ever waits for blocks that already run;
// tickets and aggregates carry the launch epoch and are never reset.
#include "gd_common.cuh"
#include <stdio.h>

__device__ __forceinline__ double gd_warp_min(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

__global__ void __launch_bounds__(GD_SCAN_THREADS)
k_block_min(gd_dev d, int64_t np, int per_block, unsigned int ticket_base)
{
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
            unsigned int tk = atomicAdd(&d.ticket[0], 1u) - ticket_base;
            s_last = (tk == gridDim.x - 1);
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
            if (lane == 0) d.cell[0] = m;
        }
    }
}

// per_block <= 32 * GD_SCAN_THREADS: every thread keeps its flags in one 32-bit mask
__global__ void __launch_bounds__(GD_SCAN_THREADS)
k_block_compact(gd_dev d, int64_t np, int per_block, unsigned int ticket_base, unsigned int epoch)
{
    __shared__ unsigned int s_bid;
    __shared__ int s_warp[GD_SCAN_THREADS / 32];
    __shared__ int s_round_base[33];
    __shared__ int s_prefix;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_bid = atomicAdd(&d.ticket[1], 1u) - ticket_base;
    __syncthreads();
    const unsigned int bid = s_bid;
    const double t_next = d.cell[0];
    const int64_t begin = (int64_t)bid * per_block;
    const int64_t end = min(np, begin + per_block);
    const int rounds = (int)((end - begin + GD_SCAN_THREADS - 1) / GD_SCAN_THREADS);

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

int gdk_next_block(gd_ctx *c)
{
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

    k_block_min<<<(unsigned)blocks, GD_SCAN_THREADS, 0, c->stream>>>(c->d, c->np, per_block, c->ticket_min_base);
    GD_LAUNCH_CHECK(c, "k_block_min");
    c->ticket_min_base += (unsigned int)blocks;
    c->epoch += 1;
    if (c->epoch == 0) c->epoch = 1;     // 0 is the value of freshly cleared scratch
    k_block_compact<<<(unsigned)blocks, GD_SCAN_THREADS, 0, c->stream>>>(c->d, c->np, per_block, c->ticket_cmp_base, c->epoch);
    GD_LAUNCH_CHECK(c, "k_block_compact");
    c->ticket_cmp_base += (unsigned int)blocks;
    return 0;
}
