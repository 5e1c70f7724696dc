/*
 * hermite_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, FP64 CPU statement of the hot path of GraviDy's method (arXiv 1702.00440; cited below as
 * P:<line> of /root/reference/PAPER.md): softened direct-summation acceleration + jerk for the active
 * particles of a 4th-order Hermite block-time-step integrator, with predictor, corrector, Aarseth
 * time-step update, active-set selection and energy.  It exists only to check the CUDA path in
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.  It shares no
 * code with paper_1702_00440_b200/csrc and is never on the product path.
 *
 * The force is the plain definition (Eq. 3 and its time derivative, sign per the erratum P:188
 * fn. 11); the integrator follows P:119-138 steps (i)-(vii) in order.  The paper defers the H4
 * formulas to Makino & Aarseth (1992); the formulas used are the standard ones, listed with
 * every reading of an unstated constant in DESIGN.md "Readings".
 *
 * No blocking, no fusion, no reordering: every pair sum runs j = 0..N-1 in order for one i.
 * OpenMP is used over i only, so results do not depend on the thread count.
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (no fast-math).
 *
 * Pins (tests/test_oracle_*.py): Kepler closed form, momentum invariants, jerk finite difference,
 * long-double brute force, mpmath brute force, exact-polynomial corrector test, 4th-order
 * convergence, Plummer energy drift, Listing-1 statistics, scheduler invariants, hand numbers for the
 * initial step (orc_initial_dt), and for the block rule the paper's energy accuracy at eta = 0.01
 * on the stored C2 runs under both readings (tests/golden/c2_t1_energy*.txt).
 * Parity unpinned (paper silent): the value of dt_min (2^-23) only.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <time.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_API __attribute__((visibility("default")))

ORC_API int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

ORC_API void orc_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ------------------------------------------------------------------------------------------------
 * PAIRSUM  [P:145 Eq. 3; jerk: P:125 step iii, sign P:188 fn. 11; BASELINE.json north_star]
 *   r = X_j - X_i ; w = V_j - V_i ; s = r.r + eps^2 ; q = 1/sqrt(s)
 *   a_i    += m_j q^3 r
 *   jerk_i += m_j q^3 ( w - 3 (r.w) q^2 r )
 * j == i is skipped by index (Eq. 3: j != i).
 * idx == NULL means i = 0..n_act-1.  x, v are [n,3] row-major; outputs [n_act,3].
 * mode 0: double accumulators (the timed baseline); mode 1: long double accumulators (parity reference;
 * pair terms are still FP64).
 * ---------------------------------------------------------------------------------------------- */
static inline void pair_term(const double *xi, const double *vi, const double *xj, const double *vj,
                             double mj, double eps2, double t[6])
{
    double rx = xj[0] - xi[0], ry = xj[1] - xi[1], rz = xj[2] - xi[2];
    double wx = vj[0] - vi[0], wy = vj[1] - vi[1], wz = vj[2] - vi[2];
    double s = rx * rx + ry * ry + rz * rz + eps2;
    double q = 1.0 / sqrt(s);
    double q2 = q * q;
    double mq3 = mj * q2 * q;
    double rw = rx * wx + ry * wy + rz * wz;
    double c = 3.0 * rw * q2;
    t[0] = mq3 * rx;
    t[1] = mq3 * ry;
    t[2] = mq3 * rz;
    t[3] = mq3 * (wx - c * rx);
    t[4] = mq3 * (wy - c * ry);
    t[5] = mq3 * (wz - c * rz);
}

ORC_API void orc_pairsum(int64_t n, const double *m, const double *x, const double *v, double eps2,
                         const int32_t *idx, int64_t n_act, double *a_out, double *j_out, int mode)
{
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < n_act; ++k) {
        int64_t i = idx ? (int64_t)idx[k] : k;
        const double *xi = x + 3 * i, *vi = v + 3 * i;
        double t[6];
        if (mode == 0) {
            double acc[6] = {0, 0, 0, 0, 0, 0};
            for (int64_t j = 0; j < n; ++j) {
                if (j == i) continue;
                pair_term(xi, vi, x + 3 * j, v + 3 * j, m[j], eps2, t);
                for (int c = 0; c < 6; ++c) acc[c] += t[c];
            }
            for (int c = 0; c < 3; ++c) { a_out[3 * k + c] = acc[c]; j_out[3 * k + c] = acc[3 + c]; }
        } else {
            long double acc[6] = {0, 0, 0, 0, 0, 0};
            for (int64_t j = 0; j < n; ++j) {
                if (j == i) continue;
                pair_term(xi, vi, x + 3 * j, v + 3 * j, m[j], eps2, t);
                for (int c = 0; c < 6; ++c) acc[c] += (long double)t[c];
            }
            for (int c = 0; c < 3; ++c) { a_out[3 * k + c] = (double)acc[c]; j_out[3 * k + c] = (double)acc[3 + c]; }
        }
    }
}

/* Same definition with EVERY operation in long double (x87 80-bit): the brute-force pin for N <= 64. */
ORC_API void orc_pairsum_longdouble(int64_t n, const double *m, const double *x, const double *v,
                                    double eps2, long double *a_out, long double *j_out)
{
    for (int64_t i = 0; i < n; ++i) {
        long double acc[6] = {0, 0, 0, 0, 0, 0};
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            long double r[3], w[3];
            for (int c = 0; c < 3; ++c) {
                r[c] = (long double)x[3 * j + c] - (long double)x[3 * i + c];
                w[c] = (long double)v[3 * j + c] - (long double)v[3 * i + c];
            }
            long double s = r[0] * r[0] + r[1] * r[1] + r[2] * r[2] + (long double)eps2;
            long double q = 1.0L / sqrtl(s);
            long double q2 = q * q, mq3 = (long double)m[j] * q2 * q;
            long double rw = r[0] * w[0] + r[1] * w[1] + r[2] * w[2];
            for (int c = 0; c < 3; ++c) {
                acc[c] += mq3 * r[c];
                acc[3 + c] += mq3 * (w[c] - 3.0L * rw * q2 * r[c]);
            }
        }
        for (int c = 0; c < 3; ++c) { a_out[3 * i + c] = acc[c]; j_out[3 * i + c] = acc[3 + c]; }
    }
}

/* ------------------------------------------------------------------------------------------------
 * Block time steps  [P:149 "block time steps (Press 1986)"; constants: DESIGN.md readings R5-R7]
 * dt in { 2^-k }, dt_min <= dt <= dt_max (both powers of two).
 * ---------------------------------------------------------------------------------------------- */
static double norm3(const double *u) { return sqrt(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]); }

/* BLOCKINIT: largest power of two <= value, clamped.  value <= 0 or NaN -> dt_min; +inf -> dt_max. */
ORC_API double orc_block_init(double value, double dt_min, double dt_max)
{
    if (!(value > 0.0)) return dt_min;
    if (value >= dt_max) return dt_max;
    if (value <= dt_min) return dt_min;
    int e;
    (void)frexp(value, &e);            /* value = f * 2^e, f in [0.5, 1)  ->  2^(e-1) <= value */
    return ldexp(1.0, e - 1);
}

/* Initial step [P:241 "from the initial calculation"; reading R4]: dt = eta |a| / |jerk|; |jerk| = 0 -> dt_max. */
ORC_API void orc_initial_dt(int64_t n, const double *a, const double *j, double eta,
                            double dt_min, double dt_max, double *dt_out)
{
    for (int64_t i = 0; i < n; ++i) {
        double an = norm3(a + 3 * i), jn = norm3(j + 3 * i);
        double raw = (jn == 0.0) ? INFINITY : eta * an / jn;
        dt_out[i] = orc_block_init(raw, dt_min, dt_max);
    }
}

/* BLOCKUPDATE [reading R7]: h = current step, t_new = time just reached (multiple of h).
 *   dt_req <  h                         -> halving_mode 1 (default): h/2, h/4, ... until <= dt_req;
 *                                          halving_mode 0 (variant): a single halving, h/2
 *   dt_req >= 2h and t_new mod 2h == 0  -> 2h
 *   otherwise                           -> h ;   then clamp to [dt_min, dt_max].  NaN -> keep h. */
ORC_API double orc_block_update(double h, double dt_req, double t_new, double dt_min, double dt_max,
                                int halving_mode)
{
    double d = h;
    if (dt_req != dt_req) {
        d = h;
    } else if (dt_req < h) {
        d = 0.5 * h;
        if (halving_mode == 1)
            while (d > dt_req && d > dt_min) d *= 0.5;
    } else if (dt_req >= 2.0 * h && fmod(t_new, 2.0 * h) == 0.0) {
        d = 2.0 * h;
    }
    if (d < dt_min) d = dt_min;
    if (d > dt_max) d = dt_max;
    return d;
}

/* ------------------------------------------------------------------------------------------------
 * Step 1 [P:127 step v]: t+ = min_i (t_i + dt_i); active = { i ascending : t_i + dt_i == t+ }.
 * Times are exact dyadic doubles, so the equality is exact.
 * ---------------------------------------------------------------------------------------------- */
ORC_API double orc_next_block(int64_t n, const double *t_i, const double *dt, int32_t *active, int64_t *n_act)
{
    double tmin = INFINITY;
    for (int64_t i = 0; i < n; ++i) {
        double tn = t_i[i] + dt[i];
        if (tn < tmin) tmin = tn;
    }
    int64_t c = 0;
    for (int64_t i = 0; i < n; ++i)
        if (t_i[i] + dt[i] == tmin) active[c++] = (int32_t)i;
    *n_act = c;
    return tmin;
}

/* ------------------------------------------------------------------------------------------------
 * Step 2 [P:130 step vii-a]: predictor for ALL n particles to time t:
 *   D = t - t_j ;  xp = x + v D + a D^2/2 + jerk D^3/6 ;  vp = v + a D + jerk D^2/2
 * ---------------------------------------------------------------------------------------------- */
ORC_API void orc_predict(int64_t n, double t, const double *x, const double *v, const double *a,
                         const double *j, const double *t_i, double *xp, double *vp)
{
    for (int64_t i = 0; i < n; ++i) {
        double D = t - t_i[i];
        double D2 = D * D / 2.0, D3 = D * D * D / 6.0;
        for (int c = 0; c < 3; ++c) {
            xp[3 * i + c] = x[3 * i + c] + v[3 * i + c] * D + a[3 * i + c] * D2 + j[3 * i + c] * D3;
            vp[3 * i + c] = v[3 * i + c] + a[3 * i + c] * D + j[3 * i + c] * D2;
        }
    }
}

/* ------------------------------------------------------------------------------------------------
 * Step 4 [P:137 step vii-d corrector; P:241 eta criterion; P:128 step vi "save old forces"]
 * For each active i with h = dt_i, old (a0, j0) = stored a_i, jerk_i, new (a1, j1) from PAIRSUM on the
 * predicted state:
 *   a2 = ( -6 (a0 - a1) - h (4 j0 + 2 j1) ) / h^2        2nd derivative of a at t_i
 *   a3 = ( 12 (a0 - a1) + 6 h (j0 + j1) ) / h^3          3rd derivative (constant over the step)
 *   x  = xp + a2 h^4/24 + a3 h^5/120 ;  v = vp + a2 h^3/6 + a3 h^4/24
 *   a2e = a2 + h a3                                       2nd derivative at t+
 *   dt_req = sqrt( eta ( |a1||a2e| + |j1|^2 ) / ( |j1||a3| + |a2e|^2 ) )       (Aarseth criterion)
 *   denominator == 0 -> dt_req = +inf
 *   dt_i = BLOCKUPDATE(h, dt_req, t+) ; a_i = a1 ; jerk_i = j1 ; t_i = t+
 * a1, j1 are [n_act,3] in active-list order; xp, vp are [n,3].  diag[0] counts NaN criteria,
 * diag[1] counts clamps at dt_min, diag[2] the minimum |dt_req/h - 1| or |dt_req/2h - 1| margin seen
 * (as a double stored in diag_margin).  dt_req_out (nullable) receives the raw criterion per active i.
 * ---------------------------------------------------------------------------------------------- */
ORC_API void orc_correct(int64_t n_act, const int32_t *active, double t_new, double eta,
                         double dt_min, double dt_max, int halving_mode,
                         double *x, double *v, double *a, double *j, double *t_i, double *dt,
                         const double *xp, const double *vp, const double *a1, const double *j1,
                         int64_t *diag, double *diag_margin, double *dt_req_out)
{
    for (int64_t k = 0; k < n_act; ++k) {
        int64_t i = active[k];
        double h = dt[i];
        double h2 = h * h, h3 = h2 * h, h4 = h2 * h2, h5 = h4 * h;
        double a2[3], a3[3], a2e[3];
        for (int c = 0; c < 3; ++c) {
            double a0 = a[3 * i + c], j0 = j[3 * i + c];
            double an = a1[3 * k + c], jn = j1[3 * k + c];
            a2[c] = (-6.0 * (a0 - an) - h * (4.0 * j0 + 2.0 * jn)) / h2;
            a3[c] = (12.0 * (a0 - an) + 6.0 * h * (j0 + jn)) / h3;
            x[3 * i + c] = xp[3 * i + c] + a2[c] * h4 / 24.0 + a3[c] * h5 / 120.0;
            v[3 * i + c] = vp[3 * i + c] + a2[c] * h3 / 6.0 + a3[c] * h4 / 24.0;
            a2e[c] = a2[c] + h * a3[c];
        }
        double na1 = norm3(a1 + 3 * k), nj1 = norm3(j1 + 3 * k), na2 = norm3(a2e), na3 = norm3(a3);
        double num = na1 * na2 + nj1 * nj1;
        double den = nj1 * na3 + na2 * na2;
        double dt_req = (den == 0.0) ? INFINITY : sqrt(eta * num / den);
        if (dt_req_out) dt_req_out[k] = dt_req;
        if (dt_req != dt_req && diag) diag[0] += 1;
        if (diag_margin && dt_req == dt_req && isfinite(dt_req)) {
            double m1 = fabs(dt_req / h - 1.0), m2 = fabs(dt_req / (2.0 * h) - 1.0);
            double mm = m1 < m2 ? m1 : m2;
            if (mm < *diag_margin) *diag_margin = mm;
        }
        double dnew = orc_block_update(h, dt_req, t_new, dt_min, dt_max, halving_mode);
        if (diag && dnew == dt_min && dt_req < dt_min) diag[1] += 1;
        for (int c = 0; c < 3; ++c) { a[3 * i + c] = a1[3 * k + c]; j[3 * i + c] = j1[3 * k + c]; }
        t_i[i] = t_new;
        dt[i] = dnew;
    }
}

/* ------------------------------------------------------------------------------------------------
 * ENERGY [P:71 Eq. 2; reading R8: softened potential consistent with Eq. 3]
 *   K = 1/2 sum m_i |v_i|^2 ;  U = - sum_{i<j} m_i m_j / sqrt(|r_ij|^2 + eps^2)
 * Row sums over j > i are formed independently (OpenMP over i), then added in index order in long double.
 * ---------------------------------------------------------------------------------------------- */
ORC_API void orc_energy(int64_t n, const double *m, const double *x, const double *v, double eps2,
                        double *kinetic, double *potential)
{
    double *row = (double *)malloc((size_t)n * sizeof(double));
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        long double s = 0.0L;
        for (int64_t j = i + 1; j < n; ++j) {
            double rx = x[3 * j] - x[3 * i], ry = x[3 * j + 1] - x[3 * i + 1], rz = x[3 * j + 2] - x[3 * i + 2];
            s += (long double)(m[j] / sqrt(rx * rx + ry * ry + rz * rz + eps2));
        }
        row[i] = (double)(s * (long double)m[i]);
    }
    long double U = 0.0L, K = 0.0L;
    for (int64_t i = 0; i < n; ++i) {
        U -= (long double)row[i];
        K += 0.5L * (long double)(m[i] * (v[3 * i] * v[3 * i] + v[3 * i + 1] * v[3 * i + 1] + v[3 * i + 2] * v[3 * i + 2]));
    }
    free(row);
    *kinetic = (double)K;
    *potential = (double)U;
}

/* ------------------------------------------------------------------------------------------------
 * Driver: INIT [P:123-126 steps i-iv] and STEP loop [P:127-138 steps v-vii], state in caller arrays.
 * ---------------------------------------------------------------------------------------------- */
typedef struct {
    int64_t n;
    double eps2, eta, dt_min, dt_max;
    int32_t halving_mode, acc_mode;      /* acc_mode: PAIRSUM accumulator mode for the integration */
    double t;                            /* current time */
    double *m, *x, *v, *a, *j, *t_i, *dt;   /* [n], [n,3] ... owned by the caller */
    double *xp, *vp, *a1, *j1;              /* scratch [n,3] owned by the caller */
    int32_t *active;                        /* scratch [n] */
    int64_t n_act;
    int64_t block_steps, particle_steps;    /* counters ("Iter", "Nsteps" of P:419-420 Listing 1) */
    int64_t diag[2];                        /* NaN criteria, dt_min clamps */
    double min_margin;                      /* closest approach of dt_req to a decision threshold */
    int64_t level_hist[64];                 /* particle steps taken with dt = 2^-k */
    double sec_force, sec_total;            /* wall seconds inside PAIRSUM / inside orc_init + orc_step ("95 %") */
} orc_state;

static double orc_now(void)
{
    struct timespec ts;
    clock_gettime(CLOCK_MONOTONIC, &ts);
    return (double)ts.tv_sec + 1e-9 * (double)ts.tv_nsec;
}

ORC_API int64_t orc_state_size(void) { return (int64_t)sizeof(orc_state); }

ORC_API void orc_init(orc_state *s)
{
    s->t = 0.0;
    s->block_steps = s->particle_steps = 0;
    s->diag[0] = s->diag[1] = 0;
    s->min_margin = INFINITY;
    memset(s->level_hist, 0, sizeof(s->level_hist));
    double w0 = orc_now();
    orc_pairsum(s->n, s->m, s->x, s->v, s->eps2, NULL, s->n, s->a, s->j, s->acc_mode);
    double w1 = orc_now();
    orc_initial_dt(s->n, s->a, s->j, s->eta, s->dt_min, s->dt_max, s->dt);
    for (int64_t i = 0; i < s->n; ++i) s->t_i[i] = 0.0;
    s->n_act = 0;
    s->sec_force = w1 - w0;
    s->sec_total = orc_now() - w0;
}

/* One block step.  Returns the new time. */
ORC_API double orc_step(orc_state *s)
{
    double w0 = orc_now();
    double tn = orc_next_block(s->n, s->t_i, s->dt, s->active, &s->n_act);
    orc_predict(s->n, tn, s->x, s->v, s->a, s->j, s->t_i, s->xp, s->vp);
    double w1 = orc_now();
    orc_pairsum(s->n, s->m, s->xp, s->vp, s->eps2, s->active, s->n_act, s->a1, s->j1, s->acc_mode);
    s->sec_force += orc_now() - w1;
    for (int64_t k = 0; k < s->n_act; ++k) {
        int e;
        (void)frexp(s->dt[s->active[k]], &e);    /* dt = 2^(e-1) */
        int lvl = 1 - e;
        if (lvl >= 0 && lvl < 64) s->level_hist[lvl] += 1;
    }
    orc_correct(s->n_act, s->active, tn, s->eta, s->dt_min, s->dt_max, s->halving_mode,
                s->x, s->v, s->a, s->j, s->t_i, s->dt, s->xp, s->vp, s->a1, s->j1, s->diag, &s->min_margin, NULL);
    s->t = tn;
    s->block_steps += 1;
    s->particle_steps += s->n_act;
    s->sec_total += orc_now() - w0;
    return tn;
}

/* Run until t >= t_end or max_steps block steps were taken (max_steps < 0: unlimited).
 * If rec_t / rec_nact / rec_hash are non-NULL they receive, per step taken from this call, the new
 * time, the active count and an FNV-1a hash of the ascending active index list (capacity rec_cap). */
ORC_API int64_t orc_run(orc_state *s, double t_end, int64_t max_steps,
                        double *rec_t, int64_t *rec_nact, uint64_t *rec_hash, int64_t rec_cap)
{
    int64_t steps = 0;
    while (s->t < t_end && (max_steps < 0 || steps < max_steps)) {
        orc_step(s);
        if (steps < rec_cap) {
            if (rec_t) rec_t[steps] = s->t;
            if (rec_nact) rec_nact[steps] = s->n_act;
            if (rec_hash) {
                uint64_t h = 1469598103934665603ULL;
                for (int64_t k = 0; k < s->n_act; ++k) {
                    uint32_t w = (uint32_t)s->active[k];
                    for (int b = 0; b < 4; ++b) { h ^= (w >> (8 * b)) & 0xffu; h *= 1099511628211ULL; }
                }
                rec_hash[steps] = h;
            }
        }
        ++steps;
    }
    return steps;
}
