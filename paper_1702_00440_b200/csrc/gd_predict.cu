// gd_predict.cu -- memory-bound per-particle kernels: state packing, predictor (P:130 step vii-a),
// initial time step ("from the initial calculation"), state read-back.
//
// Predictor roofline: HBM/L2 bandwidth.  Algorithmic bytes per particle: 4 x 32 B read (xm, vt, ad, jk)
// + 56 B written (pxy, pzm, vxy, vz) = 184 B.  Thread-per-particle, all accesses 16/32-byte vectors on
// consecutive addresses (fully coalesced).
#include "gd_common.cuh"
#include "gd_hermite.cuh"

#define GD_PB 256   // threads per block of the per-particle kernels

static inline unsigned gd_blocks(int64_t n, int per) { return (unsigned)((n + per - 1) / per); }

// ---------------------------------------------------------------------------------------------------------
// pack: user arrays m[n], x[n,3], v[n,3] -> SoA state; a = jerk = 0, t_i = 0, dt = 0, padding = zero mass.
__global__ void __launch_bounds__(GD_PB) k_pack_state(gd_dev d, int64_t n, int64_t np, const double *__restrict__ m,
                                                      const double *__restrict__ x, const double *__restrict__ v)
{
    int64_t i = (int64_t)blockIdx.x * GD_PB + threadIdx.x;
    if (i >= np) return;
    double4 xm = make_double4(0, 0, 0, 0), vt = make_double4(0, 0, 0, 0);
    double tn = __longlong_as_double(0x7ff0000000000000LL);     // +inf: padding never becomes active
    if (i < n) {
        xm = make_double4(x[3 * i], x[3 * i + 1], x[3 * i + 2], m[i]);
        vt = make_double4(v[3 * i], v[3 * i + 1], v[3 * i + 2], 0.0);
        tn = 0.0;
    }
    d.xm[i] = xm;
    d.vt[i] = vt;
    d.ad[i] = make_double4(0, 0, 0, 0);
    d.jk[i] = make_double4(0, 0, 0, 0);
    d.tnext[i] = tn;
    // padding records of the predicted planes stay zero-mass for the lifetime of the context
    d.pxy[i] = make_double2(xm.x, xm.y);
    d.pzm[i] = make_double2(xm.z, xm.w);
    d.vxy[i] = make_double2(vt.x, vt.y);
    d.vz[i] = vt.z;
}

int gdk_pack_state(gd_ctx *c, const double *m, const double *x, const double *v)
{
    k_pack_state<<<gd_blocks(c->np, GD_PB), GD_PB, 0, c->stream>>>(c->d, c->n, c->np, m, x, v);
    GD_LAUNCH_CHECK(c, "k_pack_state");
    return 0;
}

// sources only (gd_force_jerk_host): x, v are taken as already predicted
__global__ void __launch_bounds__(GD_PB) k_pack_sources(gd_dev d, int64_t n, int64_t np, const double *__restrict__ m,
                                                        const double *__restrict__ x, const double *__restrict__ v)
{
    int64_t i = (int64_t)blockIdx.x * GD_PB + threadIdx.x;
    if (i >= np) return;
    bool in = i < n;
    d.pxy[i] = in ? make_double2(x[3 * i], x[3 * i + 1]) : make_double2(0, 0);
    d.pzm[i] = in ? make_double2(x[3 * i + 2], m[i]) : make_double2(0, 0);
    d.vxy[i] = in ? make_double2(v[3 * i], v[3 * i + 1]) : make_double2(0, 0);
    d.vz[i] = in ? v[3 * i + 2] : 0.0;
}

int gdk_pack_sources(gd_ctx *c, const double *m, const double *x, const double *v)
{
    k_pack_sources<<<gd_blocks(c->np, GD_PB), GD_PB, 0, c->stream>>>(c->d, c->n, c->np, m, x, v);
    GD_LAUNCH_CHECK(c, "k_pack_sources");
    return 0;
}

__global__ void __launch_bounds__(GD_PB) k_iota(int32_t *idx, int64_t n)
{
    int64_t i = (int64_t)blockIdx.x * GD_PB + threadIdx.x;
    if (i < n) idx[i] = (int32_t)i;
}

int gdk_iota(gd_ctx *c, int32_t *idx, int64_t n)
{
    k_iota<<<gd_blocks(n, GD_PB), GD_PB, 0, c->stream>>>(idx, n);
    GD_LAUNCH_CHECK(c, "k_iota");
    return 0;
}

// ---------------------------------------------------------------------------------------------------------
// Predictor, P:130 step (vii-a), all n particles:
//   D = t - t_i ;  xp = x + v D + a D^2/2 + jerk D^3/6 ;  vp = v + a D + jerk D^2/2
// Every product and sum is rounded separately (no FMA contraction), left to right as written, so that the
// predicted records are reproducible bit for bit by any IEEE implementation of the same expression.
// dev != 0 (block-step graph): t is the t_next that k_block_min left in device memory.
__global__ void __launch_bounds__(GD_PB) k_predict(gd_dev d, int64_t n, double t, int dev)
{
    int64_t i = (int64_t)blockIdx.x * GD_PB + threadIdx.x;
    if (i >= n) return;
    if (dev) {
        if (d.ctrl->finished) return;
        t = d.cell[0];
    }
    double4 xm = d.xm[i], vt = d.vt[i], ad = d.ad[i], jk = d.jk[i];
    const gd_pred q = gd_predict_record(xm, vt, ad, jk, t);
    d.pxy[i] = make_double2(q.x, q.y);
    d.pzm[i] = make_double2(q.z, xm.w);
    d.vxy[i] = make_double2(q.vx, q.vy);
    d.vz[i] = q.vz;
}

int gdk_predict(gd_ctx *c, double t, bool dev)
{
    k_predict<<<gd_blocks(c->n, GD_PB), GD_PB, 0, c->stream>>>(c->d, c->n, t, dev ? 1 : 0);
    GD_LAUNCH_CHECK(c, "k_predict");
    return 0;
}

// ---------------------------------------------------------------------------------------------------------
// Initial block step (readings R4-R6): dt_i = largest 2^-k <= eta |a_i| / |jerk_i|, clamped to
// [dt_min, dt_max]; |jerk| = 0 -> dt_max; value not > 0 (or NaN) -> dt_min.  Takes a, jerk of all particles
// from the internal force buffers a1/j1 ([n,3], identity active list) and commits them as the stored a, jerk.
__device__ __forceinline__ double gd_block_floor(double value, double dt_min, double dt_max)
{
    if (!(value > 0.0)) return dt_min;
    if (value >= dt_max) return dt_max;
    if (value <= dt_min) return dt_min;
    // largest power of two <= value: clear the mantissa (value is a normal number here)
    return __longlong_as_double(__double_as_longlong(value) & 0x7ff0000000000000LL);
}

__global__ void __launch_bounds__(GD_PB) k_initial_dt(gd_dev d, int64_t n, double eta, double dt_min, double dt_max)
{
    int64_t i = (int64_t)blockIdx.x * GD_PB + threadIdx.x;
    if (i >= n) return;
    double ax = d.a1[3 * i], ay = d.a1[3 * i + 1], az = d.a1[3 * i + 2];
    double jx = d.j1[3 * i], jy = d.j1[3 * i + 1], jz = d.j1[3 * i + 2];
    double an = gd_norm3(ax, ay, az), jn = gd_norm3(jx, jy, jz);
    double raw = (jn == 0.0) ? __longlong_as_double(0x7ff0000000000000LL) : __ddiv_rn(__dmul_rn(eta, an), jn);
    double dt = gd_block_floor(raw, dt_min, dt_max);
    d.ad[i] = make_double4(ax, ay, az, dt);
    d.jk[i] = make_double4(jx, jy, jz, 0.0);
    double4 vt = d.vt[i];
    vt.w = 0.0;
    d.vt[i] = vt;
    d.tnext[i] = dt;
}

int gdk_initial_dt(gd_ctx *c)
{
    k_initial_dt<<<gd_blocks(c->n, GD_PB), GD_PB, 0, c->stream>>>(c->d, c->n, c->eta, c->dt_min, c->dt_max);
    GD_LAUNCH_CHECK(c, "k_initial_dt");
    return 0;
}

// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(GD_PB) k_unpack_state(gd_dev d, int64_t n, double *x, double *v, double *a, double *j,
                                                        double *t, double *dt)
{
    int64_t i = (int64_t)blockIdx.x * GD_PB + threadIdx.x;
    if (i >= n) return;
    double4 xm = d.xm[i], vt = d.vt[i], ad = d.ad[i], jk = d.jk[i];
    if (x) { x[3 * i] = xm.x; x[3 * i + 1] = xm.y; x[3 * i + 2] = xm.z; }
    if (v) { v[3 * i] = vt.x; v[3 * i + 1] = vt.y; v[3 * i + 2] = vt.z; }
    if (a) { a[3 * i] = ad.x; a[3 * i + 1] = ad.y; a[3 * i + 2] = ad.z; }
    if (j) { j[3 * i] = jk.x; j[3 * i + 1] = jk.y; j[3 * i + 2] = jk.z; }
    if (t) t[i] = vt.w;
    if (dt) dt[i] = ad.w;
}

int gdk_unpack_state(gd_ctx *c, double *x, double *v, double *a, double *j, double *t, double *dt)
{
    k_unpack_state<<<gd_blocks(c->n, GD_PB), GD_PB, 0, c->stream>>>(c->d, c->n, x, v, a, j, t, dt);
    GD_LAUNCH_CHECK(c, "k_unpack_state");
    return 0;
}

__global__ void __launch_bounds__(GD_PB) k_unpack_predicted(gd_dev d, int64_t n, double *xp, double *vp)
{
    int64_t i = (int64_t)blockIdx.x * GD_PB + threadIdx.x;
    if (i >= n) return;
    double2 xy = d.pxy[i], zm = d.pzm[i], vxy = d.vxy[i];
    double vz = d.vz[i];
    if (xp) { xp[3 * i] = xy.x; xp[3 * i + 1] = xy.y; xp[3 * i + 2] = zm.x; }
    if (vp) { vp[3 * i] = vxy.x; vp[3 * i + 1] = vxy.y; vp[3 * i + 2] = vz; }
}

int gdk_unpack_predicted(gd_ctx *c, double *xp, double *vp)
{
    k_unpack_predicted<<<gd_blocks(c->n, GD_PB), GD_PB, 0, c->stream>>>(c->d, c->n, xp, vp);
    GD_LAUNCH_CHECK(c, "k_unpack_predicted");
    return 0;
}
