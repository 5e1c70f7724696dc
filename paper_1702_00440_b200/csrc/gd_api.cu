// gd_api.cu -- the C-ABI of include/gravidy_b200.h: argument checks, workspace carving, call-order state and
// the sequencing of the kernels.  No arithmetic of the method lives here.
#include "gd_common.cuh"
#include "../../include/gravidy_b200.h"
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <cmath>

static char g_init_err[512] = "";

int gd_fail_cuda(gd_ctx *c, cudaError_t e, const char *what)
{
    char *dst = c ? c->err : g_init_err;
    snprintf(dst, 512, "CUDA error %d (%s) at %s", (int)e, cudaGetErrorString(e), what);
    return GD_ECUDA;
}

static int gd_fail(gd_ctx *c, int code, const char *msg)
{
    char *dst = c ? c->err : g_init_err;
    snprintf(dst, 512, "%s", msg);
    return code;
}

// ---- optional event timing of the force launches ---------------------------------------------------------
int gd_prof_drain(gd_ctx *c)
{
    if (c->ev_pending == 0) return 0;
    GD_CUDA(c, cudaEventSynchronize(c->ev1[c->ev_pending - 1]));
    for (int k = 0; k < c->ev_pending; ++k) {
        float ms = 0.f;
        GD_CUDA(c, cudaEventElapsedTime(&ms, c->ev0[k], c->ev1[k]));
        double *p = c->prof + 4 * c->ev_kind[k];
        p[0] += 1.0;
        p[1] += ms;
        p[2] += c->ev_pairs[k];
        p[3] += (double)ms * ms;
    }
    c->ev_pending = 0;
    return 0;
}

int gd_prof_begin(gd_ctx *c)
{
    if (!c->profile) return -1;
    if (!c->ev_created) {
        for (int k = 0; k < GD_PROF_POOL; ++k) {
            if (cudaEventCreate(&c->ev0[k]) != cudaSuccess || cudaEventCreate(&c->ev1[k]) != cudaSuccess) return -1;
        }
        c->ev_created = true;
    }
    if (c->ev_pending == GD_PROF_POOL && gd_prof_drain(c)) return -1;
    int slot = c->ev_pending;
    if (cudaEventRecord(c->ev0[slot], c->stream) != cudaSuccess) return -1;
    return slot;
}

void gd_prof_end(gd_ctx *c, int slot, int kind, double pairs)
{
    if (slot < 0) return;
    cudaEventRecord(c->ev1[slot], c->stream);
    c->ev_kind[slot] = kind;
    c->ev_pairs[slot] = pairs;
    c->ev_pending = slot + 1;
}

// ---- workspace -------------------------------------------------------------------------------------------
static inline int64_t gd_pad(int64_t n) { return ((n + GD_TILE_J - 1) / GD_TILE_J) * GD_TILE_J; }
// rows of 6 partial sums: the split force kernels need up to 4 np; the persistent loop (systems up to
// GD_LP_MAX_NP particles) keeps one row per (CTA, active particle), for up to GD_LP_GRID_BOUND CTAs
#define GD_LP_MAX_NP (1 << 19)
#define GD_LP_GRID_BOUND 160
// largest active set the loop's scratch is sized for.  The whole system: measured on C4 (N = 262144, t = 0 .. 2^-5), with
// the steps above 32768 sinks handed to the stage kernels behind the loop the run took 10.5 s instead of 2.9 s (the 33
// largest steps cost 280 ms each outside the loop, 51 ms inside), so every step stays inside.
#ifndef GD_LP_MAX_HI
#define GD_LP_MAX_HI GD_LP_MAX_NP
#endif
static inline int64_t gd_pcap(int64_t np)
{
    int64_t r = (4 * np > (1 << 20)) ? 4 * np : (1 << 20);
    const int64_t hi = np < GD_LP_MAX_HI ? np : GD_LP_MAX_HI;
    if (np <= GD_LP_MAX_NP && GD_LP_GRID_BOUND * hi > r) r = GD_LP_GRID_BOUND * hi;
    return r;
}
static inline size_t gd_up(size_t b) { return (b + 255) & ~(size_t)255; }

struct gd_carver {
    char *base;
    size_t off;
    template <typename T> T *take(size_t count)
    {
        T *p = base ? reinterpret_cast<T *>(base + off) : nullptr;
        off += gd_up(count * sizeof(T));
        return p;
    }
};

static size_t gd_carve(gd_dev *d, void *base, int64_t np, int64_t pcap)
{
    gd_carver w{(char *)base, 0};
    gd_dev t;
    t.xm = w.take<double4>(np);
    t.vt = w.take<double4>(np);
    t.ad = w.take<double4>(np);
    t.jk = w.take<double4>(np);
    t.tnext = w.take<double>(np);
    t.pxy = w.take<double2>(np);
    t.pzm = w.take<double2>(np);
    t.vxy = w.take<double2>(np);
    t.vz = w.take<double>(np);
    t.idx = w.take<int32_t>(np);
    t.a1 = w.take<double>(3 * np);
    t.j1 = w.take<double>(3 * np);
    t.partial = w.take<double>(6 * pcap);
    t.blockmin = w.take<double>(GD_SCAN_MAX_BLOCKS);
    t.agg = w.take<unsigned long long>(GD_SCAN_MAX_BLOCKS);
    t.ticket = w.take<unsigned int>(4);
    t.ctrl = w.take<gd_ctrl>(1);
    t.tile_ticket = w.take<unsigned int>(np / 32);
    t.work = w.take<unsigned int>(4);
    t.geom_s = w.take<int2>(np / 32 + 2);
    t.geom_l = w.take<int2>(np / 256 + 2);
    t.lp_L = w.take<double>(256);
    t.lp_cnt = w.take<int>(256);
    t.lp_ctl = w.take<unsigned long long>(GD_LP_CTL_WORDS);
    t.lp_prof = w.take<unsigned long long>(GD_LP_PROF_BUCKETS * 6);
    t.diag_scratch = w.take<unsigned long long>(4352);
    t.cell = w.take<double>(4);
    t.hist = w.take<long long>(64);
    t.diag = w.take<long long>(2);
    t.phi = w.take<double>(np);
    t.kin = w.take<double>(np);
    t.staging = w.take<double>(7 * np);
    t.lp_rec = w.take<double4>(2 * (np + GD_LP_REC_SLACK));
    if (d) *d = t;
    return w.off;
}

extern "C" const char *gd_version(void) { return "gravidy_b200 0.1 sm_100a"; }

extern "C" size_t gd_workspace_bytes(int64_t n)
{
    if (n < 1) return 0;
    int64_t np = gd_pad(n);
    return gd_carve(nullptr, nullptr, np, gd_pcap(np));
}

extern "C" const char *gd_last_error(const gd_ctx *ctx) { return ctx ? ctx->err : g_init_err; }

extern "C" void gd_destroy(gd_ctx *ctx)
{
    if (!ctx) return;
    if (ctx->h_cell) cudaFreeHost(ctx->h_cell);
    if (ctx->h_ctrl) cudaFreeHost(ctx->h_ctrl);
    if (ctx->step_graph) cudaGraphExecDestroy(ctx->step_graph);
    free(ctx->h_geom_s);
    free(ctx->h_geom_l);
    if (ctx->ev_created)
        for (int k = 0; k < GD_PROF_POOL; ++k) { cudaEventDestroy(ctx->ev0[k]); cudaEventDestroy(ctx->ev1[k]); }
    free(ctx);
}

// ---- init ------------------------------------------------------------------------------------------------
static int gd_create(gd_ctx **out, int64_t n, double eps, double eta, void *ws, size_t ws_bytes, void *stream)
{
    if (!out) return gd_fail(nullptr, GD_EINVAL, "gd_init: out is NULL");
    *out = nullptr;
    // the active-set compaction scans at most GD_SCAN_MAX_BLOCKS x 32 rounds x GD_SCAN_THREADS particles
    if (n < 1 || n > (int64_t)GD_SCAN_MAX_BLOCKS * 32 * GD_SCAN_THREADS) return gd_fail(nullptr, GD_EINVAL, "gd_init: n out of range (1 .. 2^25)");
    if (!(eta > 0.0) || !(eps >= 0.0) || !isfinite(eta) || !isfinite(eps)) return gd_fail(nullptr, GD_EINVAL, "gd_init: need eta > 0 and eps >= 0");
    // eps > 0 keeps the self pair in the sum (m / eps^3 times a zero vector): eps^3 must not underflow the pair term to
    // inf * 0.  Below 1e-100 only eps == 0 (the masked path) is accepted.
    if (eps > 0.0 && eps < 1e-100) return gd_fail(nullptr, GD_EINVAL, "gd_init: eps must be 0 or >= 1e-100");
    if (!ws || ((uintptr_t)ws & 255)) return gd_fail(nullptr, GD_EINVAL, "gd_init: workspace NULL or not 256-byte aligned");
    if (ws_bytes < gd_workspace_bytes(n)) return gd_fail(nullptr, GD_EINVAL, "gd_init: workspace too small (see gd_workspace_bytes)");
    gd_ctx *c = (gd_ctx *)calloc(1, sizeof(gd_ctx));
    if (!c) return gd_fail(nullptr, GD_EINVAL, "gd_init: out of host memory");
    c->n = n;
    c->np = gd_pad(n);
    c->pcap = gd_pcap(c->np);
    c->eps = eps;
    c->eps2 = eps * eps;
    c->eta = eta;
    c->lvl_min = GD_LEVEL_MIN;
    c->lvl_max = GD_LEVEL_MAX;
    c->dt_max = ldexp(1.0, -GD_LEVEL_MIN);
    c->dt_min = ldexp(1.0, -GD_LEVEL_MAX);
    c->halving_mode = 1;
    c->use_graph = 1;
    c->jsplit_max_nact = 512;
    c->ipar_small_max_nact = 2048;
    c->loop_max_nact = GD_LP_MAX_HI;          // every step the scratch allows (larger active sets: i-parallel stage kernel)
    c->loop_small_nact = 96;
    c->loop_warp_correct = 48;
    c->loop_timers = 0;
    c->slice_max_nact = 8192;
    c->slice_passes_opt = 0;
    c->loop_state_opt = 1;
    c->stream = (cudaStream_t)stream;
    gd_carve(&c->d, ws, c->np, c->pcap);
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->coop, cudaDevAttrCooperativeLaunch, dev);
    if (e == cudaSuccess) e = cudaHostAlloc((void **)&c->h_cell, 64, cudaHostAllocMapped);
    if (e == cudaSuccess) e = cudaHostGetDevicePointer((void **)&c->h_cell_dev, c->h_cell, 0);
    if (e == cudaSuccess) e = cudaHostAlloc((void **)&c->h_ctrl, 2 * sizeof(gd_ctrl), cudaHostAllocDefault);
    if (e != cudaSuccess) {
        gd_fail_cuda(nullptr, e, "gd_init: no usable CUDA device (there is no CPU fallback)");
        free(c);
        return GD_ECUDA;
    }
    *out = c;
    return GD_OK;
}

// scan scratch, tickets, histogram, diagnostics start from zero (epoch 0 = "never written"); then the launch
// shapes and geometry tables of the force kernels
static int gd_prepare(gd_ctx *c)
{
    GD_CUDA(c, cudaMemsetAsync(c->d.blockmin, 0, (char *)c->d.phi - (char *)c->d.blockmin, c->stream));
    int rc = gdk_force_setup(c);
    if (!rc) rc = gdk_loop_setup(c);
    if (!rc) rc = gdk_slice_setup(c);
    return rc;
}

static int gd_init_common(gd_ctx *c, const double *m_dev, const double *x_dev, const double *v_dev, bool wait_inputs)
{
    int rc;
    if ((rc = gd_prepare(c))) return rc;
    if ((rc = gdk_pack_state(c, m_dev, x_dev, v_dev))) return rc;          // also the predicted records at t = 0
    // host inputs: the caller may reuse its arrays when the call returns, so wait here -- before the O(N^2) evaluation is
    // enqueued, not after it -- until the copies and the repacking kernel are done
    if (wait_inputs) GD_CUDA(c, cudaStreamSynchronize(c->stream));
    c->t = 0.0;
    c->t_pred = 0.0;
    c->have_pred = true;
    // steps (iii)-(iv): initial a, jerk of every particle from the unpredicted state, then the initial dt
    if ((rc = gdk_force(c, nullptr, c->n, c->d.a1, c->d.j1))) return rc;
    if ((rc = gdk_initial_dt(c))) return rc;
    c->have_block = c->have_force = false;
    c->n_act = 0;
    return GD_OK;
}

extern "C" int gd_init(gd_ctx **out, int64_t n, const double *m_dev, const double *x_dev, const double *v_dev, double eps,
                       double eta, void *workspace_dev, size_t workspace_bytes, void *cuda_stream)
{
    if (!m_dev || !x_dev || !v_dev) return gd_fail(nullptr, GD_EINVAL, "gd_init: NULL input array");
    int rc = gd_create(out, n, eps, eta, workspace_dev, workspace_bytes, cuda_stream);
    if (rc) return rc;
    rc = gd_init_common(*out, m_dev, x_dev, v_dev, false);
    if (rc) { cudaStreamSynchronize((*out)->stream); snprintf(g_init_err, sizeof g_init_err, "%s", (*out)->err); gd_destroy(*out); *out = nullptr; }
    return rc;
}

extern "C" int gd_init_host(gd_ctx **out, int64_t n, const double *m_host, const double *x_host, const double *v_host,
                            double eps, double eta, void *workspace_dev, size_t workspace_bytes, void *cuda_stream)
{
    if (!m_host || !x_host || !v_host) return gd_fail(nullptr, GD_EINVAL, "gd_init_host: NULL input array");
    int rc = gd_create(out, n, eps, eta, workspace_dev, workspace_bytes, cuda_stream);
    if (rc) return rc;
    gd_ctx *c = *out;
    double *st = (double *)c->d.staging;
    cudaError_t e = cudaMemcpyAsync(st, m_host, n * sizeof(double), cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(st + c->np, x_host, 3 * n * sizeof(double), cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(st + 4 * c->np, v_host, 3 * n * sizeof(double), cudaMemcpyHostToDevice, c->stream);
    rc = (e == cudaSuccess) ? gd_init_common(c, st, st + c->np, st + 4 * c->np, true) : gd_fail_cuda(c, e, "gd_init_host: H2D copy");
    if (rc) { cudaStreamSynchronize(c->stream); snprintf(g_init_err, sizeof g_init_err, "%s", c->err); gd_destroy(c); *out = nullptr; }
    return rc;
}

// the captured graph froze the kernel arguments: options that change them invalidate it
static void gd_graph_drop(gd_ctx *c)
{
    if (c->step_graph) { cudaGraphExecDestroy(c->step_graph); c->step_graph = nullptr; }
}

extern "C" int gd_set_option(gd_ctx *c, const char *key, double value)
{
    if (!c || !key) return GD_EINVAL;
    if (!strcmp(key, "jsplit_max_nact")) { c->jsplit_max_nact = (int64_t)value; gd_graph_drop(c); return GD_OK; }
    if (!strcmp(key, "ipar_small_max_nact")) { c->ipar_small_max_nact = (int64_t)value; gd_graph_drop(c); return GD_OK; }
    if (!strcmp(key, "use_graph")) { c->use_graph = value != 0.0; return GD_OK; }
    if (!strcmp(key, "slice_max_nact")) { c->slice_max_nact = (int64_t)value; gd_graph_drop(c); return GD_OK; }
    if (!strcmp(key, "slice_passes")) {
        if (value < 0 || value > 16) return gd_fail(c, GD_EINVAL, "gd_set_option: slice_passes out of range");
        c->slice_passes_opt = (int64_t)value;
        gd_graph_drop(c);
        return gdk_slice_setup(c);
    }
    if (!strcmp(key, "loop_max_nact") || !strcmp(key, "loop_small_nact") || !strcmp(key, "loop_state_smem")) {
        if (!strcmp(key, "loop_max_nact")) c->loop_max_nact = (int64_t)value;
        else if (!strcmp(key, "loop_small_nact")) c->loop_small_nact = (int64_t)value;
        else c->loop_state_opt = value != 0.0;
        gd_graph_drop(c);
        return gdk_loop_setup(c);
    }
    if (!strcmp(key, "loop_timers")) { c->loop_timers = value != 0.0; gd_graph_drop(c); return GD_OK; }
    if (!strcmp(key, "loop_warp_correct")) { c->loop_warp_correct = (int64_t)value; gd_graph_drop(c); return GD_OK; }
    if (!strcmp(key, "profile")) {
        int rc = gd_prof_drain(c);
        c->profile = (int)value;
        return rc;
    }
    if (!strcmp(key, "halving_mode")) { c->halving_mode = value != 0.0; gd_graph_drop(c); return GD_OK; }
    if (!strcmp(key, "dt_level_min") || !strcmp(key, "dt_level_max")) {
        int lv = (int)value;
        if (lv < 0 || lv > 52) return gd_fail(c, GD_EINVAL, "gd_set_option: level out of range");
        if (c->block_steps > 0) return gd_fail(c, GD_ESTATE, "gd_set_option: levels can only change before the first step");
        int lo = !strcmp(key, "dt_level_min") ? lv : c->lvl_min, hi = !strcmp(key, "dt_level_max") ? lv : c->lvl_max;
        c->lvl_min = lo;
        c->lvl_max = hi;
        c->have_block = c->have_force = c->have_pred = false;   // any active list / force result in flight is void now
        gd_graph_drop(c);
        if (lo > hi) return GD_OK;                 // transient while the caller sets both: every stage call fails with GD_ESTATE until ordered
        c->dt_max = ldexp(1.0, -lo);
        c->dt_min = ldexp(1.0, -hi);
        gd_graph_drop(c);
        // the initial steps depend on the limits: redo them from the stored a, jerk
        int rc = gdk_unpack_state(c, nullptr, nullptr, c->d.a1, c->d.j1, nullptr, nullptr);
        if (!rc) rc = gdk_initial_dt(c);
        return rc;
    }
    return gd_fail(c, GD_EINVAL, "gd_set_option: unknown key");
}

// ---- the five stages ----------------------------------------------------------------------------------------
extern "C" int gd_next_block(gd_ctx *c, double *t_next_host, int64_t *n_act_host)
{
    if (!c) return GD_EINVAL;
    if (c->lvl_min > c->lvl_max) return gd_fail(c, GD_ESTATE, "gd_next_block: dt_level_min > dt_level_max");
    bool wrote_host = false;
    int rc = gdk_next_block(c, false, c->h_cell_dev, &wrote_host);
    if (rc) return rc == GD_ECUDA ? rc : GD_EINVAL;          // text already in c->err
    // the one-kernel form writes {t_next, n_act} into the pinned words itself: no copy to enqueue
    if (!wrote_host) GD_CUDA(c, cudaMemcpyAsync(c->h_cell, c->d.cell, 16, cudaMemcpyDeviceToHost, c->stream));
    GD_CUDA(c, cudaStreamSynchronize(c->stream));
    c->t_next = c->h_cell[0];
    long long na;
    memcpy(&na, &c->h_cell[1], 8);
    c->n_act = na;
    c->have_block = true;
    c->have_force = false;
    if (t_next_host) *t_next_host = c->t_next;
    if (n_act_host) *n_act_host = c->n_act;
    return GD_OK;
}

extern "C" int gd_predict(gd_ctx *c, double t)
{
    if (!c) return GD_EINVAL;
    if (t != t) return gd_fail(c, GD_EINVAL, "gd_predict: t is NaN");
    if (c->lvl_min > c->lvl_max) return gd_fail(c, GD_ESTATE, "gd_predict: dt_level_min > dt_level_max");
    int rc = gdk_predict(c, t);
    if (rc) return rc;
    c->t_pred = t;
    c->have_pred = true;
    c->have_force = false;
    return GD_OK;
}

extern "C" int gd_force_jerk(gd_ctx *c, const int32_t *idx_dev, int64_t n_act, double *a_out_dev, double *j_out_dev)
{
    if (!c) return GD_EINVAL;
    if (c->lvl_min > c->lvl_max) return gd_fail(c, GD_ESTATE, "gd_force_jerk: dt_level_min > dt_level_max");
    if (!c->have_pred) return gd_fail(c, GD_ESTATE, "gd_force_jerk: no predicted records (call gd_predict first)");
    if ((a_out_dev == nullptr) != (j_out_dev == nullptr)) return gd_fail(c, GD_EINVAL, "gd_force_jerk: give both outputs or neither");
    if (!idx_dev) {
        if (!c->have_block) return gd_fail(c, GD_ESTATE, "gd_force_jerk: no internal active list (call gd_next_block first)");
        int rc = gdk_force(c, c->d.idx, c->n_act, a_out_dev ? a_out_dev : c->d.a1, j_out_dev ? j_out_dev : c->d.j1);
        if (rc) return rc;
        if (!a_out_dev) c->have_force = (c->t_pred == c->t_next);
        return GD_OK;
    }
    if (n_act < 0 || n_act > c->np) return gd_fail(c, GD_EINVAL, "gd_force_jerk: n_act out of range");
    if (!a_out_dev) return gd_fail(c, GD_EINVAL, "gd_force_jerk: explicit index list needs explicit outputs");
    return gdk_force(c, idx_dev, n_act, a_out_dev, j_out_dev);
}

extern "C" int gd_correct_and_timestep(gd_ctx *c)
{
    if (!c) return GD_EINVAL;
    if (c->lvl_min > c->lvl_max) return gd_fail(c, GD_ESTATE, "gd_correct_and_timestep: dt_level_min > dt_level_max");
    if (!c->have_block || !c->have_force)
        return gd_fail(c, GD_ESTATE, "gd_correct_and_timestep: needs gd_next_block, gd_predict(t_next), gd_force_jerk(NULL) first");
    int rc = gdk_correct(c, c->t_next);
    if (rc) return rc;
    c->t = c->t_next;
    c->block_steps += 1;
    c->particle_steps += c->n_act;
    c->have_block = c->have_force = false;
    c->have_pred = false;                  // the predicted records of the corrected particles are stale now
    return GD_OK;
}

extern "C" int gd_energy(gd_ctx *c, double *kinetic_host, double *potential_host)
{
    if (!c) return GD_EINVAL;
    int rc = gdk_predict(c, c->t);
    if (rc) return rc;
    c->t_pred = c->t;
    c->have_pred = true;
    c->have_force = false;
    if ((rc = gdk_energy(c))) return rc;
    GD_CUDA(c, cudaMemcpyAsync(c->h_cell + 2, c->d.cell + 2, 16, cudaMemcpyDeviceToHost, c->stream));
    GD_CUDA(c, cudaStreamSynchronize(c->stream));
    if (kinetic_host) *kinetic_host = c->h_cell[2];
    if (potential_host) *potential_host = c->h_cell[3];
    return GD_OK;
}

extern "C" int gd_lagrange_radii(gd_ctx *c, const double *center_host, const double *fractions_host, int n_frac,
                                 double *radii_host, double *center_out_host)
{
    if (!c || !fractions_host || !radii_host) return GD_EINVAL;
    if (n_frac < 1 || n_frac > 16) return gd_fail(c, GD_EINVAL, "gd_lagrange_radii: 1 <= n_frac <= 16");
    for (int k = 0; k < n_frac; ++k)
        if (!(fractions_host[k] > 0.0 && fractions_host[k] <= 1.0)) return gd_fail(c, GD_EINVAL, "gd_lagrange_radii: fractions must lie in (0, 1]");
    int rc = gdk_predict(c, c->t);
    if (rc) return rc;
    c->t_pred = c->t;
    c->have_pred = true;
    c->have_force = false;
    double *st = (double *)c->d.staging;                     // [0, 16) fractions, [16, 32) radii (np >= 256: 7 np doubles)
    GD_CUDA(c, cudaMemcpyAsync(st, fractions_host, n_frac * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    if ((rc = gdk_lagrange(c, center_host, st, n_frac, st + 16))) return rc;
    GD_CUDA(c, cudaMemcpyAsync(radii_host, st + 16, n_frac * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    if (center_out_host)
        GD_CUDA(c, cudaMemcpyAsync(center_out_host, c->d.diag_scratch, 4 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    GD_CUDA(c, cudaStreamSynchronize(c->stream));
    return GD_OK;
}

extern "C" int gd_get_level_census(gd_ctx *c, int64_t *counts_host)
{
    if (!c || !counts_host) return GD_EINVAL;
    unsigned long long *cnt = c->d.diag_scratch + 64;        // the histogram area of the Lagrange-radius select: free between calls
    int rc = gdk_census(c, cnt);
    if (rc) return rc;
    GD_CUDA(c, cudaMemcpyAsync(counts_host, cnt, 64 * sizeof(int64_t), cudaMemcpyDeviceToHost, c->stream));
    GD_CUDA(c, cudaStreamSynchronize(c->stream));
    return GD_OK;
}

extern "C" int gd_core_radius(gd_ctx *c, int k_neighbours, double *core_radius_host, double *density_centre_host, double *rho_dev)
{
    if (!c || !core_radius_host) return GD_EINVAL;
    if (k_neighbours < 2 || k_neighbours > 8) return gd_fail(c, GD_EINVAL, "gd_core_radius: 2 <= k_neighbours <= 8");
    if (c->n <= k_neighbours) return gd_fail(c, GD_EINVAL, "gd_core_radius: needs more than k_neighbours particles");
    int rc = gdk_predict(c, c->t);
    if (rc) return rc;
    c->t_pred = c->t;
    c->have_pred = true;
    c->have_force = false;
    double *st = (double *)c->d.staging;                     // [0, 6) results
    if ((rc = gdk_core_radius(c, k_neighbours, rho_dev, st))) return rc;
    double out[6];
    GD_CUDA(c, cudaMemcpyAsync(out, st, sizeof out, cudaMemcpyDeviceToHost, c->stream));
    GD_CUDA(c, cudaStreamSynchronize(c->stream));
    *core_radius_host = out[3];
    if (density_centre_host) { density_centre_host[0] = out[0]; density_centre_host[1] = out[1]; density_centre_host[2] = out[2]; }
    // a particle with K others on its own point has r_iK = 0 and an infinite (or 0/0) density: the weighted means are then NaN.  The values
    // are handed back as computed, but not as a success.
    if (!std::isfinite(out[5]) || !std::isfinite(out[3]) || !std::isfinite(out[4]))
        return gd_fail(c, GD_EINVAL, "gd_core_radius: a particle has its k-th neighbour at distance 0 (coincident particles): "
                                     "the density estimate is not finite");
    return GD_OK;
}

static int gd_one_step(gd_ctx *c)
{
    int rc = gd_next_block(c, nullptr, nullptr);
    if (!rc) rc = gd_predict(c, c->t_next);
    if (!rc) rc = gd_force_jerk(c, nullptr, 0, nullptr, nullptr);
    if (!rc) rc = gd_correct_and_timestep(c);
    return rc;
}

// ---- the block-step graph -----------------------------------------------------------------------
// GD_GRAPH_STEPS block steps -- next_block, predict, the three force kernels (the device picks one), correct --
// are captured once from an internal stream with every launch shape independent of n_act, and replayed on the
// context's stream.  The host only uploads the limits (gd_ctrl) and reads the counters back once per burst of
// replays; steps enqueued past the end of the run find `finished` set and do nothing.
#define GD_GRAPH_STEPS 32

static int gd_graph_build(gd_ctx *c)
{
    cudaStream_t cap = nullptr, user = c->stream;
    GD_CUDA(c, cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
    const int64_t launches_before = c->launches;
    c->stream = cap;
    cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeRelaxed);
    int rc = 0;
    if (e == cudaSuccess) {
        // with the persistent loop in front, one iteration is a whole run of small steps plus the one step that made the loop
        // leave: a short graph keeps the count of idle nodes behind a finished run low
        const int reps = c->loop_grid > 0 ? GD_GRAPH_STEPS / 4 : GD_GRAPH_STEPS;
        for (int k = 0; k < reps && !rc; ++k) {
            // the persistent loop takes every run of small steps; the stage kernels behind it take the one step
            // that made it leave (active set above loop_hi) and do nothing once the run is finished
            rc = gdk_loop(c);
            if (!rc) rc = gdk_next_block(c, true);
            if (!rc) rc = gdk_predict(c, 0.0, true);
            if (!rc) rc = gdk_force_dev(c);
            if (!rc) rc = gdk_correct(c, 0.0, true);
        }
        cudaGraph_t g = nullptr;
        e = cudaStreamEndCapture(cap, &g);
        if (e == cudaSuccess && !rc) e = cudaGraphInstantiate(&c->step_graph, g, 0);
        if (g) cudaGraphDestroy(g);
    }
    c->stream = user;
    c->graph_nodes = c->launches - launches_before;
    c->launches = launches_before;
    cudaStreamDestroy(cap);
    if (rc) return rc;
    if (e != cudaSuccess) return gd_fail_cuda(c, e, "gd_graph_build");
    return GD_OK;
}

static int gd_run_graph(gd_ctx *c, double t_end, int64_t max_steps, int64_t *steps_out, int64_t *psteps_out)
{
    if (!c->step_graph) {
        int rc = gd_graph_build(c);
        if (rc) return rc;
    }
    gd_ctrl *up = c->h_ctrl, *down = c->h_ctrl + 1;
    up->t_end = t_end;
    up->t = c->t;
    up->max_steps = max_steps;
    up->steps = up->psteps = up->finished = 0;
    GD_CUDA(c, cudaMemcpyAsync(c->d.ctrl, up, sizeof(gd_ctrl), cudaMemcpyHostToDevice, c->stream));
    int burst = 1;
    for (;;) {
        for (int b = 0; b < burst; ++b) GD_CUDA(c, cudaGraphLaunch(c->step_graph, c->stream));
        c->launches += (int64_t)burst * c->graph_nodes;
        GD_CUDA(c, cudaMemcpyAsync(down, c->d.ctrl, sizeof(gd_ctrl), cudaMemcpyDeviceToHost, c->stream));
        GD_CUDA(c, cudaStreamSynchronize(c->stream));
        if (down->finished) break;
        if (burst < 4) burst *= 2;
    }
    c->t = down->t;
    c->block_steps += down->steps;
    c->particle_steps += down->psteps;
    c->have_block = c->have_force = c->have_pred = false;
    if (steps_out) *steps_out = down->steps;
    if (psteps_out) *psteps_out = down->psteps;
    return GD_OK;
}

// "profile" option with the persistent loop available: the same sequence as the graph (loop, then the stage kernels
// for the one step it left), launched directly so that every loop launch is bracketed by two events (kind 3).
static int gd_run_profiled(gd_ctx *c, double t_end, int64_t max_steps, int64_t *steps_out, int64_t *psteps_out)
{
    gd_ctrl *up = c->h_ctrl, *down = c->h_ctrl + 1;
    up->t_end = t_end;
    up->t = c->t;
    up->max_steps = max_steps;
    up->steps = up->psteps = up->finished = 0;
    unsigned long long lp0 = 0, lp1 = 0;
    GD_CUDA(c, cudaMemcpyAsync(c->d.ctrl, up, sizeof(gd_ctrl), cudaMemcpyHostToDevice, c->stream));
    GD_CUDA(c, cudaMemcpyAsync(&lp0, c->d.lp_ctl + GD_LP_CTL_BASE + 2, 8, cudaMemcpyDeviceToHost, c->stream));
    for (;;) {
        const int slot = gd_prof_begin(c);
        int rc = gdk_loop(c);
        gd_prof_end(c, slot, 3, 0.0);
        if (!rc) rc = gdk_next_block(c, true);
        if (!rc) rc = gdk_predict(c, 0.0, true);
        if (!rc) rc = gdk_force_dev(c);
        if (!rc) rc = gdk_correct(c, 0.0, true);
        if (rc) return rc;
        GD_CUDA(c, cudaMemcpyAsync(down, c->d.ctrl, sizeof(gd_ctrl), cudaMemcpyDeviceToHost, c->stream));
        GD_CUDA(c, cudaStreamSynchronize(c->stream));
        if (down->finished) break;
    }
    GD_CUDA(c, cudaMemcpyAsync(&lp1, c->d.lp_ctl + GD_LP_CTL_BASE + 2, 8, cudaMemcpyDeviceToHost, c->stream));
    GD_CUDA(c, cudaStreamSynchronize(c->stream));
    c->prof[4 * 3 + 2] += (double)(lp1 - lp0) * (double)c->n;         // pairs evaluated inside the loop
    c->t = down->t;
    c->block_steps += down->steps;
    c->particle_steps += down->psteps;
    c->have_block = c->have_force = c->have_pred = false;
    if (steps_out) *steps_out = down->steps;
    if (psteps_out) *psteps_out = down->psteps;
    return GD_OK;
}

extern "C" int gd_step(gd_ctx *c, int64_t n_steps, int64_t *particle_steps_host)
{
    if (!c) return GD_EINVAL;
    if (c->lvl_min > c->lvl_max) return gd_fail(c, GD_ESTATE, "gd_step: dt_level_min > dt_level_max");
    if (c->use_graph && !c->profile && n_steps >= GD_GRAPH_STEPS / 2)
        return gd_run_graph(c, INFINITY, n_steps, nullptr, particle_steps_host);
    if (c->use_graph && c->profile && c->loop_grid > 0 && n_steps >= GD_GRAPH_STEPS / 2)
        return gd_run_profiled(c, INFINITY, n_steps, nullptr, particle_steps_host);
    int64_t before = c->particle_steps;
    for (int64_t s = 0; s < n_steps; ++s) {
        int rc = gd_one_step(c);
        if (rc) return rc;
    }
    GD_CUDA(c, cudaStreamSynchronize(c->stream));
    if (particle_steps_host) *particle_steps_host = c->particle_steps - before;
    return GD_OK;
}

extern "C" int gd_run_until(gd_ctx *c, double t_end, int64_t max_steps, int64_t *steps_host, int64_t *particle_steps_host)
{
    if (!c) return GD_EINVAL;
    if (t_end != t_end) return gd_fail(c, GD_EINVAL, "gd_run_until: t_end is NaN");
    if (c->lvl_min > c->lvl_max) return gd_fail(c, GD_ESTATE, "gd_run_until: dt_level_min > dt_level_max");
    if (c->use_graph && !c->profile && c->t < t_end && max_steps != 0)
        return gd_run_graph(c, t_end, max_steps, steps_host, particle_steps_host);
    if (c->use_graph && c->profile && c->loop_grid > 0 && c->t < t_end && max_steps != 0)
        return gd_run_profiled(c, t_end, max_steps, steps_host, particle_steps_host);
    int64_t before = c->particle_steps, steps = 0;
    while (c->t < t_end && (max_steps < 0 || steps < max_steps)) {
        int rc = gd_one_step(c);
        if (rc) return rc;
        ++steps;
    }
    GD_CUDA(c, cudaStreamSynchronize(c->stream));
    if (steps_host) *steps_host = steps;
    if (particle_steps_host) *particle_steps_host = c->particle_steps - before;
    return GD_OK;
}

// ---- getters -----------------------------------------------------------------------------------------------
extern "C" double gd_time(const gd_ctx *c) { return c ? c->t : NAN; }
extern "C" int64_t gd_n(const gd_ctx *c) { return c ? c->n : 0; }
extern "C" int64_t gd_n_active(const gd_ctx *c) { return c && c->have_block ? c->n_act : 0; }
extern "C" int64_t gd_block_steps(const gd_ctx *c) { return c ? c->block_steps : 0; }
extern "C" int64_t gd_particle_steps(const gd_ctx *c) { return c ? c->particle_steps : 0; }
extern "C" int gd_last_force_kernel(const gd_ctx *c) { return c ? c->last_force_kernel : 0; }
extern "C" int64_t gd_kernel_launches(const gd_ctx *c) { return c ? c->launches : 0; }
extern "C" int gd_last_force_geometry(const gd_ctx *c, int *geom_host)
{
    if (!c || !geom_host) return GD_EINVAL;
    memcpy(geom_host, c->last_geom, sizeof c->last_geom);
    return GD_OK;
}

extern "C" int gd_get_state(gd_ctx *c, double *x, double *v, double *a, double *j, double *t, double *dt)
{
    if (!c) return GD_EINVAL;
    return gdk_unpack_state(c, x, v, a, j, t, dt);
}

extern "C" int gd_get_state_host(gd_ctx *c, double *x, double *v, double *a, double *j, double *t, double *dt)
{
    if (!c) return GD_EINVAL;
    // unpack into the staging area ([np,3] x 4 would not fit: two passes of at most 7 np doubles)
    double *st = (double *)c->d.staging;
    const int64_t n = c->n, np = c->np;
    if (x || v) {
        int rc = gdk_unpack_state(c, x ? st : nullptr, v ? st + 3 * np : nullptr, nullptr, nullptr, nullptr, nullptr);
        if (rc) return rc;
        if (x) GD_CUDA(c, cudaMemcpyAsync(x, st, 3 * n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        if (v) GD_CUDA(c, cudaMemcpyAsync(v, st + 3 * np, 3 * n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    }
    if (a || j || t || dt) {
        if (x || v) GD_CUDA(c, cudaStreamSynchronize(c->stream));
        int rc = gdk_unpack_state(c, nullptr, nullptr, a ? st : nullptr, j ? st + 3 * np : nullptr, t ? st + 6 * np : nullptr, nullptr);
        if (rc) return rc;
        if (a) GD_CUDA(c, cudaMemcpyAsync(a, st, 3 * n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        if (j) GD_CUDA(c, cudaMemcpyAsync(j, st + 3 * np, 3 * n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        if (t) GD_CUDA(c, cudaMemcpyAsync(t, st + 6 * np, n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        if (dt) {
            GD_CUDA(c, cudaStreamSynchronize(c->stream));
            rc = gdk_unpack_state(c, nullptr, nullptr, nullptr, nullptr, nullptr, st);
            if (rc) return rc;
            GD_CUDA(c, cudaMemcpyAsync(dt, st, n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        }
    }
    GD_CUDA(c, cudaStreamSynchronize(c->stream));
    return GD_OK;
}

extern "C" int gd_get_predicted(gd_ctx *c, double *xp, double *vp)
{
    if (!c) return GD_EINVAL;
    if (!c->have_pred) return gd_fail(c, GD_ESTATE, "gd_get_predicted: no predicted records");
    return gdk_unpack_predicted(c, xp, vp);
}

extern "C" int gd_get_active(gd_ctx *c, int32_t *idx_dev, int64_t cap)
{
    if (!c || !idx_dev) return GD_EINVAL;
    if (!c->have_block) return gd_fail(c, GD_ESTATE, "gd_get_active: no active list");
    if (cap < c->n_act) return gd_fail(c, GD_EINVAL, "gd_get_active: capacity too small");
    if (c->n_act > 0)
        GD_CUDA(c, cudaMemcpyAsync(idx_dev, c->d.idx, c->n_act * sizeof(int32_t), cudaMemcpyDeviceToDevice, c->stream));
    return GD_OK;
}

extern "C" int gd_get_profile(gd_ctx *c, double *prof_host)
{
    if (!c || !prof_host) return GD_EINVAL;
    int rc = gd_prof_drain(c);
    if (rc) return rc;
    memcpy(prof_host, c->prof, sizeof c->prof);
    return GD_OK;
}

extern "C" int gd_get_loop_profile(gd_ctx *c, int64_t *out_host)
{
    if (!c || !out_host) return GD_EINVAL;
    GD_CUDA(c, cudaMemcpyAsync(out_host, c->d.lp_ctl + GD_LP_CTL_BASE + 2, 11 * sizeof(int64_t), cudaMemcpyDeviceToHost, c->stream));
    GD_CUDA(c, cudaStreamSynchronize(c->stream));
    return GD_OK;
}

#if GD_LP_FINE
extern "C" __attribute__((visibility("default"))) int gd_debug_read_staging(gd_ctx *c, void *host, size_t nbytes)
{
    GD_CUDA(c, cudaMemcpyAsync(host, c->d.staging, nbytes, cudaMemcpyDeviceToHost, c->stream));
    GD_CUDA(c, cudaStreamSynchronize(c->stream));
    return GD_OK;
}
#endif

extern "C" int gd_get_loop_histogram(gd_ctx *c, int64_t *out_host)
{
    if (!c || !out_host) return GD_EINVAL;
    GD_CUDA(c, cudaMemcpyAsync(out_host, c->d.lp_prof, GD_LP_PROF_BUCKETS * 6 * sizeof(int64_t), cudaMemcpyDeviceToHost, c->stream));
    GD_CUDA(c, cudaStreamSynchronize(c->stream));
    return GD_OK;
}

extern "C" int gd_get_level_histogram(gd_ctx *c, int64_t *counts_host, int64_t *diag_host)
{
    if (!c) return GD_EINVAL;
    if (counts_host) GD_CUDA(c, cudaMemcpyAsync(counts_host, c->d.hist, 64 * sizeof(int64_t), cudaMemcpyDeviceToHost, c->stream));
    if (diag_host) GD_CUDA(c, cudaMemcpyAsync(diag_host, c->d.diag, 2 * sizeof(int64_t), cudaMemcpyDeviceToHost, c->stream));
    GD_CUDA(c, cudaStreamSynchronize(c->stream));
    return GD_OK;
}

// ---- one-shot host entry -------------------------------------------------------------------------------------
extern "C" int gd_force_jerk_host(int64_t n, const double *m_host, const double *x_host, const double *v_host, double eps,
                                  const int32_t *idx_host, int64_t n_act, double *a_out_host, double *j_out_host,
                                  void *workspace_dev, size_t workspace_bytes, void *cuda_stream)
{
    if (!m_host || !x_host || !v_host || !a_out_host || !j_out_host) return gd_fail(nullptr, GD_EINVAL, "gd_force_jerk_host: NULL array");
    gd_ctx *c = nullptr;
    int rc = gd_create(&c, n, eps, 1.0, workspace_dev, workspace_bytes, cuda_stream);
    if (rc) return rc;
    if (!idx_host) n_act = n;
    if (n_act < 0 || n_act > n) { gd_destroy(c); return gd_fail(nullptr, GD_EINVAL, "gd_force_jerk_host: n_act out of range"); }
    double *st = (double *)c->d.staging;
    cudaError_t e = cudaMemcpyAsync(st, m_host, n * sizeof(double), cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(st + c->np, x_host, 3 * n * sizeof(double), cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(st + 4 * c->np, v_host, 3 * n * sizeof(double), cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess && idx_host && n_act > 0)
        e = cudaMemcpyAsync(c->d.idx, idx_host, n_act * sizeof(int32_t), cudaMemcpyHostToDevice, c->stream);
    if (e != cudaSuccess) rc = gd_fail_cuda(c, e, "gd_force_jerk_host: H2D copy");
    if (!rc) rc = gd_prepare(c);
    if (!rc) rc = gdk_pack_sources(c, st, st + c->np, st + 4 * c->np);
    if (!rc) rc = gdk_force(c, idx_host ? c->d.idx : nullptr, n_act, c->d.a1, c->d.j1);
    if (!rc && n_act > 0) {
        e = cudaMemcpyAsync(a_out_host, c->d.a1, 3 * n_act * sizeof(double), cudaMemcpyDeviceToHost, c->stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(j_out_host, c->d.j1, 3 * n_act * sizeof(double), cudaMemcpyDeviceToHost, c->stream);
        if (e != cudaSuccess) rc = gd_fail_cuda(c, e, "gd_force_jerk_host: D2H copy");
    }
    if (!rc) {
        e = cudaStreamSynchronize(c->stream);
        if (e != cudaSuccess) rc = gd_fail_cuda(c, e, "gd_force_jerk_host: synchronize");
    }
    if (rc) snprintf(g_init_err, sizeof g_init_err, "%s", c->err);
    gd_destroy(c);
    return rc;
}

extern "C" int gd_fp64_peak_probe(int iters, double *flops_host, double *ms_host)
{
    if (iters < 1) return GD_EINVAL;
    return gdk_fp64_probe(iters, flops_host, ms_host) ? GD_ECUDA : GD_OK;
}

extern "C" int gd_selftest_div_const(int64_t n, uint64_t seed, int64_t *mismatches_host)
{
    if (n < 0 || !mismatches_host) return GD_EINVAL;
    long long bad = 0;
    if (gdk_selftest_div_const((long long)n, (unsigned long long)seed, &bad)) return GD_ECUDA;
    *mismatches_host = (int64_t)bad;
    return GD_OK;
}
