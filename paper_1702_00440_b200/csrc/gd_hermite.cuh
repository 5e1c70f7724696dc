// gd_hermite.cuh -- per-particle arithmetic of the 4th-order Hermite scheme (predictor P:130, corrector P:137,
// Aarseth criterion P:241, block rule P:149; formulas per DESIGN.md readings R1, R5-R7, R18-R19), shared by the
// stage kernels (gd_predict.cu, gd_correct.cu) and the persistent block-step loop (gd_loop.cu).
// Every floating-point operation is rounded separately, in the order written (no FMA contraction): the block-step
// decision is discrete, so the arithmetic that feeds it is kept reproducible.  Not shared with oracle/.
#pragma once
#include "gd_common.cuh"

__device__ __forceinline__ double gd_mul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double gd_add(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double gd_sub(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ double gd_div(double a, double b) { return __ddiv_rn(a, b); }

// x / C for the constants 6, 24, 120 of the predictor and corrector, correctly rounded without the division routine
// (~35 dependent FP64 instructions): with y = RN(1/C), q = RN(x y) is within one ulp of x / C, r = x - q C is exact
// (one FMA), and RN(q + r y) is the correctly rounded quotient (Markstein 1990: y correctly rounded, significand of C
// not all ones).  Outside the range where neither r nor q r can underflow or overflow the division routine runs.
// Bit for bit the result of x / C: gd_selftest_div_const compares the two on random operands.
template <int C>
__device__ __forceinline__ double gd_div_const(double x)
{
    constexpr double c = (double)C, y = 1.0 / (double)C;
    const double ax = fabs(x);
    if (!(ax > 0x1p-900 && ax < 0x1p900)) return __ddiv_rn(x, c);
    const double q = __dmul_rn(x, y);
    const double r = __fma_rn(-q, c, x);
    return __fma_rn(r, y, q);
}

// ---- predictor: D = t - t_i ; xp = x + v D + a D^2/2 + jerk D^3/6 ; vp = v + a D + jerk D^2/2 -------------------
struct gd_pred { double x, y, z, vx, vy, vz; };

__device__ __forceinline__ gd_pred gd_predict_record(const double4 &xm, const double4 &vt, const double4 &ad, const double4 &jk, double t)
{
    double D = gd_sub(t, vt.w);
    double DD = gd_mul(D, D);
    double D2 = gd_mul(DD, 0.5);                              // = DD / 2 exactly
    double D3 = gd_div_const<6>(gd_mul(DD, D));
#define GD_PX(x0, v0, a0, j0) gd_add(gd_add(gd_add((x0), gd_mul((v0), D)), gd_mul((a0), D2)), gd_mul((j0), D3))
#define GD_PV(v0, a0, j0) gd_add(gd_add((v0), gd_mul((a0), D)), gd_mul((j0), D2))
    gd_pred p;
    p.x = GD_PX(xm.x, vt.x, ad.x, jk.x);
    p.y = GD_PX(xm.y, vt.y, ad.y, jk.y);
    p.z = GD_PX(xm.z, vt.z, ad.z, jk.z);
    p.vx = GD_PV(vt.x, ad.x, jk.x);
    p.vy = GD_PV(vt.y, ad.y, jk.y);
    p.vz = GD_PV(vt.z, ad.z, jk.z);
#undef GD_PX
#undef GD_PV
    return p;
}

// ---- corrector, one Cartesian component ----------------------------------------------------------------------
struct gd_corr1 { double xnew, vnew, a2e, a3; };
struct gd_hpow { double h, h2, h3, h4, h5, ih2, ih3; bool pow2; };

// Block steps are powers of two (R5), so x / h^2 and x / h^3 are exact scalings: they are done as
// multiplications by 2^(2k), 2^(3k), bit for bit the quotient (any other h keeps the division).
__device__ __forceinline__ gd_hpow gd_step_powers(double h)
{
    gd_hpow p;
    p.h = h;
    p.h2 = gd_mul(h, h);
    p.h3 = gd_mul(p.h2, h);
    p.h4 = gd_mul(p.h2, p.h2);
    p.h5 = gd_mul(p.h4, h);
    const long long bits = __double_as_longlong(h);
    const long long ef = (bits >> 52) & 0x7ff;
    p.pow2 = bits > 0 && (bits & 0xfffffffffffffLL) == 0 && ef >= 1023 - 300 && ef <= 1023 + 300;
    const double ih = __longlong_as_double((2046LL - ef) << 52);
    p.ih2 = gd_mul(ih, ih);
    p.ih3 = gd_mul(p.ih2, ih);
    return p;
}

__device__ __forceinline__ gd_corr1 gd_correct_component(double xp, double vp, double a0, double j0, double a1, double j1, const gd_hpow &p)
{
    const double h = p.h;
    double da = gd_sub(a0, a1);
    // a2 = (-6 (a0 - a1) - h (4 j0 + 2 j1)) / h^2
    const double n2 = gd_sub(gd_mul(-6.0, da), gd_mul(h, gd_add(gd_mul(4.0, j0), gd_mul(2.0, j1))));
    double a2 = p.pow2 ? gd_mul(n2, p.ih2) : gd_div(n2, p.h2);
    // a3 = (12 (a0 - a1) + 6 h (j0 + j1)) / h^3
    const double n3 = gd_add(gd_mul(12.0, da), gd_mul(gd_mul(6.0, h), gd_add(j0, j1)));
    double a3 = p.pow2 ? gd_mul(n3, p.ih3) : gd_div(n3, p.h3);
    gd_corr1 r;
    // x = xp + a2 h^4/24 + a3 h^5/120 ;  v = vp + a2 h^3/6 + a3 h^4/24
    r.xnew = gd_add(gd_add(xp, gd_div_const<24>(gd_mul(a2, p.h4))), gd_div_const<120>(gd_mul(a3, p.h5)));
    r.vnew = gd_add(gd_add(vp, gd_div_const<6>(gd_mul(a2, p.h3))), gd_div_const<24>(gd_mul(a3, p.h4)));
    r.a2e = gd_add(a2, gd_mul(h, a3));        // second derivative at the end of the step
    r.a3 = a3;
    return r;
}

// ---- Aarseth criterion + block rule ---------------------------------------------------------------------------
// dt_req = sqrt( eta (|a1||a2e| + |j1|^2) / (|j1||a3| + |a2e|^2) ); halve if dt_req < h (halving_mode 1: until
// dt <= dt_req); double if dt_req >= 2h and t_next is a multiple of 2h; clamp; NaN keeps h.
// flags: bit 0 = criterion was NaN, bit 1 = clamped at dt_min with dt_req below it.
__device__ __forceinline__ double gd_new_step(double na1, double nj1, double na2, double na3, double h, double t_next, double eta,
                                              double dt_min, double dt_max, int halving_mode, int &flags)
{
    double num = gd_add(gd_mul(na1, na2), gd_mul(nj1, nj1));
    double den = gd_add(gd_mul(nj1, na3), gd_mul(na2, na2));
    double dt_req = (den == 0.0) ? __longlong_as_double(0x7ff0000000000000LL) : __dsqrt_rn(gd_div(gd_mul(eta, num), den));
    double dnew = h;
    flags = 0;
    if (dt_req != dt_req) {
        flags |= 1;
    } else if (dt_req < h) {
        dnew = 0.5 * h;
        if (halving_mode == 1)
            while (dnew > dt_req && dnew > dt_min) dnew *= 0.5;
    } else if (dt_req >= 2.0 * h) {
        // t_next / 2h: exact when 2h is a power of two (always, for block steps), and then the same double as the product
        // with the exactly representable 1 / 2h -- one multiplication instead of the division routine
        const long long hb = __double_as_longlong(h), ef = (hb >> 52) & 0x7ff;
        const bool pow2 = hb > 0 && (hb & 0xfffffffffffffLL) == 0 && ef >= 1023 - 300 && ef <= 1023 + 300;
        const double q = pow2 ? t_next * __longlong_as_double((2045LL - ef) << 52) : t_next / (2.0 * h);
        if (q == floor(q)) dnew = 2.0 * h;
    }
    if (dnew < dt_min) dnew = dt_min;
    if (dnew > dt_max) dnew = dt_max;
    if (dnew == dt_min && dt_req < dt_min) flags |= 2;
    return dnew;
}

// level of a step h = 2^-lvl
__device__ __forceinline__ int gd_step_level(double h) { return 1023 - (int)((__double_as_longlong(h) >> 52) & 0x7ff); }

// ---- the whole per-particle update: corrector (3 components) + criterion + block rule ---------------------------
struct gd_corrected { double x, y, z, vx, vy, vz, dt; int flags; };

__device__ __forceinline__ gd_corrected gd_correct_particle(double xp, double yp, double zp, double vxp, double vyp, double vzp,
                                                            const double4 &ad, const double4 &jk, const double (&a1)[3],
                                                            const double (&j1)[3], double t_next, double eta, double dt_min,
                                                            double dt_max, int halving_mode)
{
    const double h = ad.w;
    const gd_hpow hp = gd_step_powers(h);
    const gd_corr1 cx = gd_correct_component(xp, vxp, ad.x, jk.x, a1[0], j1[0], hp);
    const gd_corr1 cy = gd_correct_component(yp, vyp, ad.y, jk.y, a1[1], j1[1], hp);
    const gd_corr1 cz = gd_correct_component(zp, vzp, ad.z, jk.z, a1[2], j1[2], hp);
    const double na1 = gd_norm3(a1[0], a1[1], a1[2]), nj1 = gd_norm3(j1[0], j1[1], j1[2]);
    const double na2 = gd_norm3(cx.a2e, cy.a2e, cz.a2e), na3 = gd_norm3(cx.a3, cy.a3, cz.a3);
    gd_corrected r;
    r.dt = gd_new_step(na1, nj1, na2, na3, h, t_next, eta, dt_min, dt_max, halving_mode, r.flags);
    r.x = cx.xnew; r.y = cy.xnew; r.z = cz.xnew;
    r.vx = cx.vnew; r.vy = cy.vnew; r.vz = cz.vnew;
    return r;
}
