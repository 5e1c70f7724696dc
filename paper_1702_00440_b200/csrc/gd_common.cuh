// gd_common.cuh -- shared declarations of the CUDA path (sm_100a only).  Not shared with oracle/.
//
// Device-resident state (all in the caller's workspace, every array 256-byte aligned; np = n rounded up to
// GD_TILE_J, records n..np-1 are zero-mass padding):
//   xm[np]  double4 {x, y, z, m}          vt[np] double4 {vx, vy, vz, t_i}
//   ad[np]  double4 {ax, ay, az, dt_i}    jk[np] double4 {jx, jy, jz, 0}
//   tnext[np] double  t_i + dt_i (exact dyadic; +inf in the padding)
// Predicted records written by the predictor and read by the force kernels, as four coalesced SoA planes:
//   pxy[np] double2 {xp, yp}   pzm[np] double2 {zp, m}   vxy[np] double2 {vxp, vyp}   vz[np] double {vzp}
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

#define GD_TILE_J 256            // sources per shared-memory stage of the force kernels; np is a multiple
#define GD_UNIT_J 64             // granularity of a CTA's source range (TMA copies stay 16-byte aligned)

// Device-resident run control of the captured block-step graph (gd_step / gd_run_until): the host writes the
// limits, the kernels keep the counters, and once `finished` is set every later kernel of the graph does nothing.
struct gd_ctrl {
    double t_end;                // stop once t >= t_end
    double t;                    // time reached (k_correct_timestep)
    long long max_steps;         // stop after this many block steps of the current run (< 0: no limit)
    long long steps, psteps;     // block steps / particle steps taken in the current run
    long long finished;          // set by k_block_min
};

struct gd_dev {
    double4 *xm, *vt, *ad, *jk;
    double *tnext;
    double2 *pxy, *pzm, *vxy;
    double *vz;
    int32_t *idx;                // active list (ascending)
    double *a1, *j1;             // [np,3] force results of the internal active list
    double *partial;             // [pcap,6] partial sums of split force evaluations
    double *blockmin;            // [GD_SCAN_MAX_BLOCKS] per-block minima of tnext
    unsigned long long *agg;     // [GD_SCAN_MAX_BLOCKS] {epoch:32 | count:32} per-block aggregates of the compaction
    unsigned int *ticket;        // [4] {k_block_min arrivals, k_block_compact block numbers, scan epoch, -}: re-armed by the last block
    gd_ctrl *ctrl;
    unsigned int *tile_ticket;   // [np / 32] arrivals per i-tile of a split force evaluation (re-armed to 0 by the last CTA)
    unsigned int *work;          // [4] {next unit ticket, CTAs finished} of the persistent force grid (re-armed by the last CTA)
    int2 *geom_s, *geom_l;       // [np / 32 + 2], [np / 256 + 2]: i-tiles -> {source splits, units per split}
    double *cell;                // [4] {t_next, n_act (as int64 bits), K, U}
    long long *hist;             // [64] particle steps per level
    long long *diag;             // [2]  NaN criteria, dt_min clamps
    double *phi;                 // [np] per-particle potential sums  (energy)
    double *kin;                 // [np] per-particle kinetic terms   (energy)
    void *staging;               // [7 np] doubles: staging for host<->device copies of m, x, v
    unsigned long long *diag_scratch;    // [4352] centre, scale, targets, prefixes and histograms of the Lagrange-radius select
    // persistent block-step loop (gd_loop.cu)
    double4 *lp_rec;             // [np + GD_LP_REC_SLACK][2] candidate records, one segment of S rows per CTA
    double *lp_L;                // [256] smallest t_i + dt_i of every CTA's slice
    int *lp_cnt;                 // [256] candidates per CTA
    unsigned long long *lp_ctl;  // [GD_LP_CTL_WORDS] hand-off counters and run counters of k_block_loop, three 128-byte lines:
                                 //  word GD_LP_CTL_BAR   arrivals at the first hand-off (every CTA, once per block step; monotonic)
                                 //  word GD_LP_CTL_BAR2  arrivals at the second hand-off (the owners of a step; monotonic)
                                 //  words GD_LP_CTL_BASE + k, written by CTA 0 when a launch ends and read when the next begins:
                                 //   k = 1 first hand-off's count at the start of the next launch, 13 the second's;
                                 //   k = 2 particle steps, 3 block steps inside the loop (always kept);
                                 //   k = 4 ns in the loop, 5..8 ns per phase, 9 launches that ran, 10..12 CTA 0 as an owner
                                 //   (steps, ns correcting, ns publishing) -- the ns words stay 0 unless the timers are on.
                                 //  The two polled counters have a line each so that the spinning loads of one hand-off do not
                                 //  share a line with the arrivals of the other; anything new goes behind GD_LP_CTL_BASE + 13.
    unsigned long long *lp_prof; // [GD_LP_PROF_BUCKETS][6] per bucket b = bit length of n_act: {block steps, particle steps,
                                 //  ns in [force], in the barrier after it, in [correct], in the barrier after it} (CTA 0's view)
};
#define GD_LP_PROF_BUCKETS 32
#define GD_LP_CTL_BAR 0
#define GD_LP_CTL_BAR2 16
#define GD_LP_CTL_BASE 32
#define GD_LP_CTL_WORDS 48
#ifndef GD_LP_FINE
#define GD_LP_FINE 0               // 1: debug build with fine-grained phase stamps of the loop (gd_loop.cu)
#endif

#define GD_SCAN_MAX_BLOCKS 1024
#define GD_LP_REC_SLACK (32 * 256)   // rows of lp_rec beyond np: slices are rounded up to 32 for up to 256 CTAs
#define GD_PROF_POOL 64
#define GD_SCAN_THREADS 1024

struct gd_ctx {
    int64_t n, np, pcap;
    double eps, eps2, eta;
    int lvl_min, lvl_max, halving_mode;
    double dt_min, dt_max;
    int64_t jsplit_max_nact;
    cudaStream_t stream;
    gd_dev d;
    double *h_cell;              // pinned host mirror of d.cell (mapped: h_cell_dev is its address on the device)
    double *h_cell_dev;
    int coop;                    // the device can launch cooperative kernels
    // host-side step state
    double t, t_next;
    int64_t n_act;
    bool have_block, have_pred, have_force;
    double t_pred;
    int64_t block_steps, particle_steps, launches;
    int last_force_kernel;
    int64_t ipar_small_max_nact;         // js_hi < n_act <= this: i-parallel kernel with 32-sink tiles
    int grid_s, grid_l, js_clusters;     // launch shapes (gdk_force_setup)
    int *h_geom_s, *h_geom_l;            // host copies of the geometry tables ({splits, units per split} pairs)
    int last_geom[4];                    // geometry of the last force launch: variant, i-tiles (or groups), splits, units per split
    cudaGraphExec_t step_graph;          // GD_GRAPH_STEPS block steps captured from the stream (built on first use)
    gd_ctrl *h_ctrl;                     // pinned host mirror of d.ctrl
    int use_graph;
    int64_t loop_max_nact;               // option: largest active set the persistent loop takes (0 = loop off)
    int loop_state_opt;                  // option: keep the own state resident in shared memory when it fits
    int64_t loop_warp_correct;           // option: a CTA owning up to this many active particles corrects them a warp each
    int64_t loop_small_nact;             // option: active sets up to this size use the lanes-over-sources mapping
    int loop_timers;                     // option: CTA 0 of k_block_loop reads the device timer per phase and fills the per-size bins
    int loop_grid, loop_S, loop_hi, loop_cap, loop_state;   // geometry of k_block_loop (loop_grid = 0: not usable)
    size_t loop_smem;
    int64_t slice_max_nact;              // option: largest active set gd_force_jerk gives to k_force_slice (0 = off)
    int slice_grid, slice_S, slice_passes;   // geometry of k_force_slice (slice_grid = 0: not usable)
    int64_t slice_passes_opt;            // option: slices per CTA (0 = the fewest that fit shared memory)
    size_t slice_smem;
    int64_t graph_nodes;                 // kernel nodes in step_graph
    int sm_count;
    // optional CUDA-event timing of the force launches ("profile" option; see gd_get_profile)
    int profile;
    cudaEvent_t ev0[GD_PROF_POOL], ev1[GD_PROF_POOL];
    double ev_pairs[GD_PROF_POOL];
    int ev_kind[GD_PROF_POOL];
    int ev_pending;
    bool ev_created;
    double prof[20];             // per kind k = 0 (i-parallel L), 1 (j-split), 2 (i-parallel S), 3 (block-step loop), 4 (slice): {launches, ms, pairs, ms^2}
    char err[512];
};

int gd_prof_begin(gd_ctx *c);                               // gd_api.cu: record the start event (returns slot or -1)
void gd_prof_end(gd_ctx *c, int slot, int kind, double pairs);
int gd_prof_drain(gd_ctx *c);

// ---- launch wrappers (one per kernel file); all enqueue on c->stream and bump c->launches -------------
int gdk_pack_state(gd_ctx *c, const double *m, const double *x, const double *v);           // gd_predict.cu
int gdk_predict(gd_ctx *c, double t, bool dev = false);
int gdk_initial_dt(gd_ctx *c);
int gdk_unpack_state(gd_ctx *c, double *x, double *v, double *a, double *j, double *t, double *dt);
int gdk_unpack_predicted(gd_ctx *c, double *xp, double *vp);
int gdk_pack_sources(gd_ctx *c, const double *m, const double *x, const double *v);
int gdk_iota(gd_ctx *c, int32_t *idx, int64_t n);

int gdk_force(gd_ctx *c, const int32_t *idx, int64_t n_act, double *a_out, double *j_out);   // gd_force.cu
int gdk_force_dev(gd_ctx *c);
int gdk_force_setup(gd_ctx *c);

int gdk_correct(gd_ctx *c, double t_next, bool dev = false);                                 // gd_correct.cu
int gdk_next_block(gd_ctx *c, bool dev = false, double *host_cell = nullptr, bool *wrote_host = nullptr);   // gd_next_block.cu
int gdk_loop_setup(gd_ctx *c);                                                               // gd_loop.cu
int gdk_loop(gd_ctx *c);
int gdk_slice_setup(gd_ctx *c);
int64_t gdk_slice_hi(const gd_ctx *c);
int gdk_force_slice(gd_ctx *c, const int32_t *idx, int64_t n_act, double *a_out, double *j_out, bool dev);
int gdk_energy(gd_ctx *c);
int gdk_lagrange(gd_ctx *c, const double *center_host, const double *frac_dev, int n_frac, double *radii_dev);   // gd_diag.cu                                                                   // gd_energy.cu
int gdk_census(gd_ctx *c, unsigned long long *counts_dev);
int gdk_core_radius(gd_ctx *c, int K, double *rho_dev, double *out_dev);
int gdk_selftest_div_const(long long n, unsigned long long seed, long long *mismatches);          // gd_probe.cu
int gdk_fp64_probe(int iters, double *flops, double *ms);                                    // gd_probe.cu

int gd_fail_cuda(gd_ctx *c, cudaError_t e, const char *what);

#define GD_CUDA(c, call)                                                     \
    do {                                                                     \
        cudaError_t e_ = (call);                                             \
        if (e_ != cudaSuccess) return gd_fail_cuda((c), e_, #call);          \
    } while (0)
#define GD_LAUNCH_CHECK(c, name)                                             \
    do {                                                                     \
        cudaError_t e_ = cudaGetLastError();                                 \
        if (e_ != cudaSuccess) return gd_fail_cuda((c), e_, name);           \
        (c)->launches += 1;                                                  \
    } while (0)

// ---- small device helpers ---------------------------------------------------------------------------
__device__ __forceinline__ double gd_norm3(double x, double y, double z)
{
    // sqrt((x*x + y*y) + z*z) with separately rounded operations (no contraction): the time-step decisions
    // downstream are discrete, so the memory-bound kernels keep every rounding explicit.
    return __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(x, x), __dmul_rn(y, y)), __dmul_rn(z, z)));
}
