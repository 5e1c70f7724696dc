/*
 * gravidy_b200.h -- C-ABI boundary of the B200-native Hermite force/jerk hot path.
 *
 * The calls follow the paper's statement of the integration scheme (GraviDy, arXiv 1702.00440;
 * "P:<n>" = line n of the paper text): steps (i)-(vii) of section 2.4.
 *
 *   gd_init                  steps (i)-(iv)  P:123-126   allocate/initialise, initial a and jerk (O(N^2)), initial dt
 *   gd_next_block            step  (v)       P:127       find the particles to move at the next integration time
 *   gd_predict               step  (vii-a)   P:130       predict x, v of ALL N particles to time t
 *   gd_force_jerk            step  (vii-c)   P:132-136   a and jerk of the active particles from all N (Eq. 3, fn. 11 P:188)
 *   gd_correct_and_timestep  steps (vi),(vii-d,e) P:128, P:137-138, P:241   corrector + Aarseth time-step update
 *   gd_energy                Eq. 2           P:71, P:125 kinetic + (softened) potential energy
 *
 * Conventions
 *   - All floating point is IEEE binary64.  Indices are int32.  G = 1 (N-body units).
 *   - Pointers named *_dev are DEVICE pointers, *_host are HOST pointers.  The library never allocates
 *     device memory: the caller hands one workspace of gd_workspace_bytes(n) bytes (256-byte aligned) to
 *     gd_init and keeps it alive until gd_destroy.  Inputs are copied at init: HOST inputs (gd_init_host) may be
 *     reused or freed as soon as the call returns (it synchronises once the copies are done); DEVICE inputs (gd_init)
 *     are read by a kernel enqueued on the stream and must stay untouched until the stream has passed it (any
 *     synchronising call, or stream order).  (The two self-tests gd_fp64_peak_probe / gd_selftest_div_const, which
 *     take no ctx, allocate and free 8 bytes of their own.)
 *   - [n,3] arrays are row-major (x0 y0 z0 x1 y1 z1 ...).
 *   - All work is enqueued on the CUDA stream given at init (a cudaStream_t passed as void*; NULL = the
 *     legacy default stream).  Calls are asynchronous unless stated; the ones that return values to the
 *     host (gd_next_block, gd_energy, gd_get_*_host, gd_*_host) synchronise that stream.
 *   - Every call returns GD_OK (0) or a negative error code; the text of the last error is available from
 *     gd_last_error().  After an error the only guaranteed-safe call is gd_destroy.
 *   - Call order inside one block step: gd_next_block -> gd_predict(t_next) -> gd_force_jerk(NULL list)
 *     -> gd_correct_and_timestep.  gd_step / gd_run_until replay exactly that sequence.
 *   - There is no CPU fallback: without a CUDA device every compute call fails with GD_ECUDA.
 */
#ifndef GRAVIDY_B200_H
#define GRAVIDY_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define GD_API __attribute__((visibility("default")))
#else
#define GD_API
#endif

#define GD_OK        0
#define GD_EINVAL   -1   /* bad argument: n < 1, NaN or <= 0 eta, eps < 0, NULL pointer, workspace too small/misaligned */
#define GD_ESTATE   -2   /* call order violated (e.g. correct before force) */
#define GD_ECUDA    -3   /* CUDA runtime error (sticky); text via gd_last_error */

/* Block-time-step limits (powers of two; the paper does not print them -- DESIGN.md reading R6). */
#define GD_LEVEL_MIN 3    /* dt_max = 2^-3  */
#define GD_LEVEL_MAX 23   /* dt_min = 2^-23 */

typedef struct gd_ctx gd_ctx;   /* opaque; created by gd_init, destroyed by gd_destroy */

/* Library / build identification: "gravidy_b200 <version> sm_100a". Never fails. */
GD_API const char *gd_version(void);

/* Bytes of device memory gd_init needs for n particles (state, predicted records, active list, force
 * outputs, partial sums, scan scratch).  Returns 0 for n < 1. */
GD_API size_t gd_workspace_bytes(int64_t n);

/* Steps (i)-(iv).  Copies m [n], x [n,3], v [n,3] (device pointers) into the workspace, sets
 * t = 0 and t_i = 0, evaluates a_i and jerk_i of every particle from the unpredicted state (one all-active
 * gd_force_jerk, O(N^2)), and sets the initial block step dt_i = largest 2^-k <= eta |a_i| / |jerk_i|,
 * clamped to [2^-GD_LEVEL_MAX, 2^-GD_LEVEL_MIN] (|jerk| = 0 -> dt_max).  eps is the softening length
 * (>= 0; Eq. 3), eta the accuracy parameter of the time-step criterion (> 0).
 * On success *out owns a small host struct; release it with gd_destroy.  Asynchronous. */
GD_API int gd_init(gd_ctx **out, int64_t n, const double *m_dev, const double *x_dev, const double *v_dev,
            double eps, double eta, void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* Same as gd_init with HOST input arrays (pageable or pinned): the host->device copies are part of the
 * call, and the call waits for them (and for the kernel that repacks them) before it returns, so the arrays may be
 * reused at once; the all-active force evaluation behind them stays asynchronous.  Used for end-to-end timing. */
GD_API int gd_init_host(gd_ctx **out, int64_t n, const double *m_host, const double *x_host, const double *v_host,
                 double eps, double eta, void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* Releases the host struct (not the workspace).  NULL is allowed. */
GD_API void gd_destroy(gd_ctx *ctx);

/* Text of the last error recorded on ctx (ctx == NULL: last error of a failed gd_init). Never NULL. */
GD_API const char *gd_last_error(const gd_ctx *ctx);

/* Tunables.  Which kernel gd_force_jerk (and the force stage of gd_step behind the persistent loop) launches is
 * decided by the size of the active set, first match wins:
 *   n_act <= "slice_max_nact" (default 8192; 0 = off)   k_force_slice: one CTA per SM over a shared-memory slice of
 *                                                        the sources, every sink against it, partial rows folded per sink
 *   n_act <= "jsplit_max_nact" (default 512, capped at 32 x the clusters of its grid)
 *                                                        k_force_jsplit: clusters of 8 CTAs split the sources, DSMEM fold
 *   n_act <= "ipar_small_max_nact" (default 2048)        k_force_ipar<1,4>: i-parallel, 32-sink tiles, sources split
 *   larger                                               k_force_ipar<2,1>: i-parallel, 256-sink tiles (the all-active kernel)
 * With the defaults the second and third rows are never reached (the slice kernel measured faster over their whole
 * range); they run only when "slice_max_nact" is lowered, which the parity tests do.
 * Other keys: "slice_passes" (slices per CTA of k_force_slice: 0 = the fewest whose records fit in shared memory
 * [default: 1 up to N ~ 3.5e5, 3 at C5's size], 1..16 forces a count),
 * "dt_level_min", "dt_level_max" (override GD_LEVEL_MIN/MAX before the first step; 0 <= min <= max <= 52),
 * "halving_mode" (1: halve until dt <= dt_req [default]; 0: a single halving per step),
 * "loop_max_nact", "loop_small_nact", "loop_state_smem", "loop_warp_correct" (the persistent block-step loop behind
 * gd_step / gd_run_until: largest active set it takes [default: all], size up to which lanes stride over sources
 * [96], own state resident in shared memory [1], number of own active particles up to which a CTA corrects them a
 * warp each instead of a thread each [48]),
 * "loop_timers" (0/1, default 0: launch the loop's instantiation whose CTA 0 reads the device timer around every phase
 * and fills the bins of gd_get_loop_histogram; costs about 1 % on runs of small block steps),
 * "use_graph" (0/1, default 1: gd_step / gd_run_until replay a captured graph),
 * "profile" (0/1: time every force launch with CUDA events, see gd_get_profile).
 * GD_EINVAL on unknown keys. */
GD_API int gd_set_option(gd_ctx *ctx, const char *key, double value);

/* Step (v).  t_next = min_i (t_i + dt_i); the active list becomes { i ascending : t_i + dt_i == t_next }
 * (exact comparison of dyadic doubles).  Writes t_next and the active count to the host pointers (either may
 * be NULL).  Synchronises the stream. */
GD_API int gd_next_block(gd_ctx *ctx, double *t_next_host, int64_t *n_act_host);

/* Step (vii-a).  For ALL n particles, D = t - t_i:
 *   xp = x + v D + a D^2/2 + jerk D^3/6 ;  vp = v + a D + jerk D^2/2
 * written to the packed predicted records the force kernels read.  Sets the context's current time to t. */
GD_API int gd_predict(gd_ctx *ctx, double t);

/* Step (vii-c); Eq. 3 P:145 and its time derivative (sign per fn. 11 P:188).  For each listed i:
 *   a_i    = sum_{j != i} m_j r_ij / (r_ij^2 + eps^2)^(3/2)
 *   jerk_i = sum_{j != i} m_j [ v_ij / (r_ij^2 + eps^2)^(3/2) - 3 (r_ij . v_ij) r_ij / (r_ij^2 + eps^2)^(5/2) ]
 * with r_ij = xp_j - xp_i, v_ij = vp_j - vp_i over the predicted records of all n particles (a prior gd_predict
 * is required).  idx_dev: n_act int32 particle indices in [0, n) (device), or NULL for the internal active list
 * of the last gd_next_block (then n_act is ignored).  a_out_dev / j_out_dev: [n_act,3] device arrays, or NULL
 * to keep the results in the internal buffers that gd_correct_and_timestep consumes.  With an explicit
 * idx_dev the call does not touch integrator state.  Indices are not range-checked.  n_act == 0 is a no-op.
 * The kernel is chosen by n_act as the table at gd_set_option says (by default: the source-slice kernel up to 8192
 * sinks, the i-parallel kernel with 256-sink tiles above). */
GD_API int gd_force_jerk(gd_ctx *ctx, const int32_t *idx_dev, int64_t n_act, double *a_out_dev, double *j_out_dev);

/* One-shot form of gd_force_jerk on HOST arrays: x, v are taken as the (already predicted) state of n sources,
 * idx_host (or NULL = all n) lists the sinks, results go to host arrays [n_act,3].  All copies are inside the call. */
GD_API int gd_force_jerk_host(int64_t n, const double *m_host, const double *x_host, const double *v_host, double eps,
                       const int32_t *idx_host, int64_t n_act, double *a_out_host, double *j_out_host,
                       void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* Steps (vi), (vii-d), (vii-e).  For every particle of the internal active list, with
 * h = dt_i, (a0, j0) the stored values and (a1, j1) the results of the last gd_force_jerk(NULL list):
 *   a2 = (-6 (a0 - a1) - h (4 j0 + 2 j1)) / h^2 ;  a3 = (12 (a0 - a1) + 6 h (j0 + j1)) / h^3
 *   x = xp + a2 h^4/24 + a3 h^5/120 ;  v = vp + a2 h^3/6 + a3 h^4/24 ;  a2e = a2 + h a3
 *   dt_req = sqrt( eta (|a1||a2e| + |j1|^2) / (|j1||a3| + |a2e|^2) )          (denominator 0 -> +inf)
 *   dt_i <- h/2, h/4, ... (largest 2^-k h <= dt_req) if dt_req < h ; 2h if dt_req >= 2h and t_next is a multiple of 2h ; else h ; clamped
 *   a_i <- a1, jerk_i <- j1, t_i <- t_next.
 * GD_ESTATE unless preceded by next_block, predict(t_next) and force_jerk(NULL). */
GD_API int gd_correct_and_timestep(gd_ctx *ctx);

/* Eq. 2, P:71 (potential softened consistently with Eq. 3 -- DESIGN.md reading R8):
 *   K = 1/2 sum m_i |v_i|^2 ;  U = - sum_{i<j} m_i m_j / sqrt(|r_ij|^2 + eps^2)
 * evaluated on all particles predicted to the current time (identical to the stored state when every particle
 * is synchronised).  Overwrites the predicted records.  Synchronises. */
GD_API int gd_energy(gd_ctx *ctx, double *kinetic_host, double *potential_host);

/* gd_energy for callers that cannot allocate device memory -- Eq. 2, with the softened potential of gd_energy:
 *   out_dev[0] = K = 1/2 sum m_i |v_i|^2 ;  out_dev[1] = U = - sum_{i<j} m_i m_j / sqrt(|r_ij|^2 + eps^2)
 * of the n particles m_dev [n], x_dev [n,3], v_dev [n,3] exactly as given (no ctx, no prediction).
 * Why it exists: all other calls need a workspace the caller obtained from cudaMalloc, and gd_init pins host memory.
 * A program that gave all free HBM to its own pool at start-up (a later cudaMalloc fails), a loop that must not
 * stall (cudaMalloc / cudaFree make the whole device wait), or a plug-in whose host application forbids driver
 * allocations after start-up cannot satisfy that.  This call allocates nothing, on the device or the host: its scratch
 * (one {K, U} pair per 256 particles) is a fixed array inside the library's device image, 128 KiB on every GPU that
 * loads the library, held until the process exits.
 *   - Limit: 1 <= n <= GD_ENERGY_STATIC_MAX_N; anything larger returns GD_EINVAL (nothing is truncated).
 *   - Pointers: m_dev, x_dev, v_dev, out_dev (two doubles) are DEVICE pointers owned by the caller, on the GPU that is
 *     current in the calling thread; cuda_stream (cudaStream_t as void*, NULL = legacy default stream) belongs to it too.
 *   - Asynchronous: two kernels are enqueued on cuda_stream, nothing is synchronised; read out_dev in stream order.
 *   - First call on each GPU: looks up the device address of the built-in array (and may make the CUDA runtime load
 *     the library's device code).  Make that first call outside any stream capture.
 *   - The array is shared by every call on that GPU and keeps the last call's contents.  No slot has to start at zero
 *     (a call reads only what it wrote itself), and calls in one stream are ordered and safe; calls that may run
 *     CONCURRENTLY on one GPU (different streams without an event between them) race on it -- serialise them.
 *   - Errors: GD_EINVAL (n out of range, NULL pointer, eps negative or not finite: checked before any CUDA call),
 *     GD_ECUDA; text from gd_energy_static_last_error() (per calling thread; never NULL). */
#define GD_ENERGY_STATIC_MAX_N 2097152   /* 2^21 particles */
GD_API int gd_energy_static(int64_t n, const double *m_dev, const double *x_dev, const double *v_dev, double eps,
                            double *out_dev, void *cuda_stream);
GD_API const char *gd_energy_static_last_error(void);

/* Convenience: n_steps block steps (next_block, predict, force_jerk, correct) / block steps until t >= t_end.
 * Optional outputs (NULL to skip): steps taken, sum of active counts (particle steps).  Synchronises. */
GD_API int gd_step(gd_ctx *ctx, int64_t n_steps, int64_t *particle_steps_host);
GD_API int gd_run_until(gd_ctx *ctx, double t_end, int64_t max_steps, int64_t *steps_host, int64_t *particle_steps_host);

/* Current time / counters.  Never fail on a valid ctx. */
GD_API double  gd_time(const gd_ctx *ctx);
GD_API int64_t gd_n(const gd_ctx *ctx);
GD_API int64_t gd_n_active(const gd_ctx *ctx);          /* size of the current internal active list */
GD_API int64_t gd_block_steps(const gd_ctx *ctx);       /* "Iter"   of Listing 1 */
GD_API int64_t gd_particle_steps(const gd_ctx *ctx);    /* "Nsteps" of Listing 1 */
GD_API int     gd_last_force_kernel(const gd_ctx *ctx); /* 0 none, 1 i-parallel (256-sink tiles), 2 j-split, 3 i-parallel (32-sink tiles), 4 source-slice kernel */
GD_API int64_t gd_kernel_launches(const gd_ctx *ctx);   /* kernels launched on behalf of this ctx so far */
/* Launch geometry of the last explicit force evaluation -> geom_host[4] = { kernel (as above, 0 = 256-sink tiles),
 * i-tiles, source splits (i-parallel) or clusters per i-tile (j-split), units of 64 sources per split }.  Diagnostics only. */
GD_API int gd_last_force_geometry(const gd_ctx *ctx, int *geom_host);

/* Copies of the state into DEVICE arrays ([n,3] or [n]); any pointer may be NULL.  Asynchronous. */
GD_API int gd_get_state(gd_ctx *ctx, double *x_dev, double *v_dev, double *a_dev, double *j_dev, double *t_dev, double *dt_dev);
/* Same into HOST arrays; synchronises. */
GD_API int gd_get_state_host(gd_ctx *ctx, double *x_host, double *v_host, double *a_host, double *j_host, double *t_host, double *dt_host);
/* Predicted positions / velocities of the last gd_predict into DEVICE arrays [n,3]. */
GD_API int gd_get_predicted(gd_ctx *ctx, double *xp_dev, double *vp_dev);
/* Current internal active list into a device array of capacity cap (>= gd_n_active). */
GD_API int gd_get_active(gd_ctx *ctx, int32_t *idx_dev, int64_t cap);
/* Particle steps taken per level k (dt = 2^-k) since init -> counts_host[64]; and diagnostic counters
 * diag_host[2] = { time-step criteria that evaluated to NaN, clamps at dt_min }.  Synchronises. */
GD_API int gd_get_level_histogram(gd_ctx *ctx, int64_t *counts_host, int64_t *diag_host);
/* Lagrange radii, "the radii of spheres containing a certain mass fraction of the system" (Fig. 9, Fig. 11
 * P:347): for each fraction f_k in (0, 1] (n_frac <= 16, HOST array) the radius, about the centre, of the smallest
 * sphere that holds at least that fraction of the total mass, taken on the positions predicted to the current time
 * -> radii_host[n_frac].  center_host: HOST {x, y, z}, or NULL = the centre of mass.  center_out_host: NULL or HOST
 * [4] <- {centre x, y, z, total mass}.  Masses are counted in fixed point so that the result does not depend on the
 * order of summation (R24).  On-device 8-pass radix select, no sort.  Synchronises. */
GD_API int gd_lagrange_radii(gd_ctx *ctx, const double *center_host, const double *fractions_host, int n_frac,
                             double *radii_host, double *center_out_host);
/* Time-step census, "the distribution of the time steps" (Fig. 13 P:363 shows it at four times): counts_host[64]
 * <- the number of particles whose CURRENT block step is 2^-k, k = 0 .. 63 (gd_get_level_histogram counts the particle
 * steps TAKEN per level since init instead).  Synchronises. */
GD_API int gd_get_level_census(gd_ctx *ctx, int64_t *counts_host);
/* Density centre and core radius, "the core radius as calculated at T=0" (Fig. 12).  The paper prints no
 * definition; reading R25 takes Casertano & Hut (1985) as the direct-summation codes use it: with r_iK the
 * distance from particle i to its K-th nearest neighbour (K = k_neighbours, 2 .. 8; 6 is the usual choice),
 *   rho_i = (sum of the masses of the K - 1 nearest neighbours) / (4 pi / 3 r_iK^3)
 *   x_d = sum rho_i x_i / sum rho_i ;   r_c = sqrt( sum rho_i^2 |x_i - x_d|^2 / sum rho_i^2 )
 * on the positions predicted to the current time.  *core_radius_host <- r_c; density_centre_host: NULL or HOST [3] <- x_d;
 * rho_dev: NULL or a DEVICE array [n] that receives rho_i.  O(n^2) distance evaluations on the device (every particle
 * keeps its K nearest in registers): a diagnostic for snapshots, about as long as one all-active force evaluation
 * (~0.1 s at n = 262144, ~2 s at n = 2^20; there is no size limit besides that).  If some particle has its K-th neighbour
 * at distance 0 (K others on its own point) the density is not finite: the outputs are written as computed (NaN / inf) and
 * the call returns GD_EINVAL with a text saying so.  Overwrites the predicted records like gd_energy.  Synchronises. */
GD_API int gd_core_radius(gd_ctx *ctx, int k_neighbours, double *core_radius_host, double *density_centre_host, double *rho_dev);
/* Counters of the persistent block-step loop (k_block_loop, the kernel behind gd_step / gd_run_until that takes the
 * block steps) since init -> out_host[11] = { particle steps, block steps taken inside
 * the loop, ns spent inside it (device global timer, CTA 0), ns in its force phase, in the barrier after it, in its
 * corrector phase, in the barrier after it, launches that did work, and for CTA 0 as an owner of active particles:
 * steps, ns summing partials + correcting, ns publishing } (11 values).  The step counts are always kept; the ns
 * values only grow while the "loop_timers" option is on.  Synchronises. */
GD_API int gd_get_loop_profile(gd_ctx *ctx, int64_t *out_host);
/* The same loop's block steps binned by the size of their active set ("N_act << N": where the step count and the
 * time of a block-step run go) -> out_host[32][6]: bucket b holds the steps with bit_length(n_act) == b, i.e.
 * 2^(b-1) <= n_act < 2^b, as { block steps, particle steps, ns in the force phase, ns in the barrier after it, ns in
 * the corrector phase, ns in the barrier after it } (device global timer, CTA 0's view), since init; only the steps
 * taken while the "loop_timers" option was on are binned.  Synchronises. */
GD_API int gd_get_loop_histogram(gd_ctx *ctx, int64_t *out_host);

/* Optional CUDA-event timing of the force launches, switched on with gd_set_option(ctx, "profile", 1): every
 * gd_force_jerk issued afterwards is bracketed by two events on the context's stream (the all-active evaluation
 * inside gd_init runs before the option can be set and is not timed); gd_step / gd_run_until then launch the
 * persistent block-step loop directly instead of replaying the graph, each launch bracketed the same way.
 * prof_host[20] receives, for kind k = 0 (i-parallel kernel, 256-sink tiles), 1 (j-split kernel), 2 (i-parallel
 * kernel, 32-sink tiles), 3 (k_block_loop: pairs = particle steps taken inside the loop x n), 4 (k_force_slice,
 * with its fold kernel):
 *   prof[4k] launches timed, prof[4k+1] sum of durations in ms, prof[4k+2] sum of pair interactions (n_act * n),
 *   prof[4k+3] sum of squared durations (ms^2).  Synchronises on the last recorded event. */
GD_API int gd_get_profile(gd_ctx *ctx, double *prof_host);

/* Register-only DFMA loop on every SM: measures the FP64 peak the force kernels are bounded by.  Returns the
 * achieved rate in flop/s (2 flop per FMA per lane) in *flops_host; ms_host receives the elapsed milliseconds.
 * Needs no ctx (it allocates and frees 8 bytes of device memory itself).  Synchronises the device. */
GD_API int gd_fp64_peak_probe(int iters, double *flops_host, double *ms_host);

/* Self-test of the device arithmetic: the predictor and corrector divide by the constants 6, 24, 120
 * with a multiply and two FMAs instead of the division routine; the two must agree bit for bit.  Evaluates both on n
 * random operands of the stream `seed` (all signs, binary exponents -960 .. 959, random significands) for each of
 * the three constants and returns the number of differing results in *mismatches_host (0 = identical).  Needs no
 * ctx; allocates and frees 8 bytes of device memory; synchronises the device. */
GD_API int gd_selftest_div_const(int64_t n, uint64_t seed, int64_t *mismatches_host);

#ifdef __cplusplus
}
#endif
#endif /* GRAVIDY_B200_H */
