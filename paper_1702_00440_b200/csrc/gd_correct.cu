// gd_correct.cu -- fused Hermite corrector + Aarseth time-step criterion + block-step rule for the active list
// (steps vi, vii-d, vii-e: P:128; eta criterion P:241; block steps P:149).  The H4 formulas are the
// standard ones the paper defers to Makino & Aarseth 1992; constants the paper leaves open are the
// readings R4-R7, R18-R19 of DESIGN.md.
//
// Bound: memory latency / bandwidth.  Per active particle: reads idx (4 B), predicted record (56 B), ad, jk
// (64 B), a1, j1 (48 B), xm (32 B, to keep m); writes xm, vt, ad, jk (128 B), tnext (8 B) = 340 B, scattered by
// index.  Every floating-point operation is rounded separately, in the order written (no FMA contraction):
// the block-step decision is discrete, so the arithmetic that feeds it is kept reproducible.
#include "gd_common.cuh"

#define GD_CB 128

__device__ __forceinline__ double gd_mul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double gd_add(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double gd_sub(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ double gd_div(double a, double b) { return __ddiv_rn(a, b); }

struct gd_corr1 { double xnew, vnew, a2e, a3; };

// one Cartesian component of the corrector
__device__ __forceinline__ gd_corr1 gd_correct_component(double xp, double vp, double a0, double j0, double a1, double j1,
                                                         double h, double h2, double h3, double h4, double h5)
{
    double da = gd_sub(a0, a1);
    // a2 = (-6 (a0 - a1) - h (4 j0 + 2 j1)) / h^2
    double a2 = gd_div(gd_sub(gd_mul(-6.0, da), gd_mul(h, gd_add(gd_mul(4.0, j0), gd_mul(2.0, j1)))), h2);
    // a3 = (12 (a0 - a1) + 6 h (j0 + j1)) / h^3
    double a3 = gd_div(gd_add(gd_mul(12.0, da), gd_mul(gd_mul(6.0, h), gd_add(j0, j1))), h3);
    gd_corr1 r;
    // x = xp + a2 h^4/24 + a3 h^5/120 ;  v = vp + a2 h^3/6 + a3 h^4/24
    r.xnew = gd_add(gd_add(xp, gd_div(gd_mul(a2, h4), 24.0)), gd_div(gd_mul(a3, h5), 120.0));
    r.vnew = gd_add(gd_add(vp, gd_div(gd_mul(a2, h3), 6.0)), gd_div(gd_mul(a3, h4), 24.0));
    r.a2e = gd_add(a2, gd_mul(h, a3));        // second derivative at the end of the step
    r.a3 = a3;
    return r;
}

__global__ void __launch_bounds__(GD_CB)
k_correct_timestep(gd_dev d, int n_act, double t_next, double eta, double dt_min, double dt_max, int halving_mode, int dev)
{
    // dev != 0 (block-step graph): the active count and t_next come from device memory, the grid is fixed and
    // strides over the list, and block 0 advances the run counters once the step is committed
    if (dev) {
        if (d.ctrl->finished) return;
        n_act = (int)((const long long *)d.cell)[1];
        t_next = d.cell[0];
    }
    __shared__ unsigned int s_hist[64];
    __shared__ unsigned int s_diag[2];
    if (threadIdx.x < 64) s_hist[threadIdx.x] = 0;
    if (threadIdx.x < 2) s_diag[threadIdx.x] = 0;
    __syncthreads();

    for (int k = blockIdx.x * GD_CB + threadIdx.x; k < n_act; k += gridDim.x * GD_CB) {
        const int32_t i = d.idx[k];
        double2 pxy = d.pxy[i], pzm = d.pzm[i], pvxy = d.vxy[i];
        double pvz = d.vz[i];
        double4 ad = d.ad[i], jk = d.jk[i];
        const double *a1 = d.a1 + 3 * (int64_t)k, *j1 = d.j1 + 3 * (int64_t)k;
        double a1x = a1[0], a1y = a1[1], a1z = a1[2], j1x = j1[0], j1y = j1[1], j1z = j1[2];

        const double h = ad.w;
        const double h2 = gd_mul(h, h), h3 = gd_mul(h2, h), h4 = gd_mul(h2, h2), h5 = gd_mul(h4, h);
        gd_corr1 cx = gd_correct_component(pxy.x, pvxy.x, ad.x, jk.x, a1x, j1x, h, h2, h3, h4, h5);
        gd_corr1 cy = gd_correct_component(pxy.y, pvxy.y, ad.y, jk.y, a1y, j1y, h, h2, h3, h4, h5);
        gd_corr1 cz = gd_correct_component(pzm.x, pvz, ad.z, jk.z, a1z, j1z, h, h2, h3, h4, h5);

        // Aarseth criterion: dt_req = sqrt( eta (|a1||a2e| + |j1|^2) / (|j1||a3| + |a2e|^2) )
        double na1 = gd_norm3(a1x, a1y, a1z), nj1 = gd_norm3(j1x, j1y, j1z);
        double na2 = gd_norm3(cx.a2e, cy.a2e, cz.a2e), na3 = gd_norm3(cx.a3, cy.a3, cz.a3);
        double num = gd_add(gd_mul(na1, na2), gd_mul(nj1, nj1));
        double den = gd_add(gd_mul(nj1, na3), gd_mul(na2, na2));
        double dt_req = (den == 0.0) ? __longlong_as_double(0x7ff0000000000000LL) : __dsqrt_rn(gd_div(gd_mul(eta, num), den));

        // block rule: halve if dt_req < h; double if dt_req >= 2h and t_next is a multiple of 2h; clamp; NaN keeps h
        double dnew = h;
        if (dt_req != dt_req) {
            atomicAdd(&s_diag[0], 1u);
        } else if (dt_req < h) {
            dnew = 0.5 * h;
            if (halving_mode == 1)
                while (dnew > dt_req && dnew > dt_min) dnew *= 0.5;
        } else if (dt_req >= 2.0 * h) {
            double q = t_next / (2.0 * h);                    // exact: 2h is a power of two
            if (q == floor(q)) dnew = 2.0 * h;
        }
        if (dnew < dt_min) dnew = dt_min;
        if (dnew > dt_max) dnew = dt_max;
        if (dnew == dt_min && dt_req < dt_min) atomicAdd(&s_diag[1], 1u);

        // level of the step just taken: h = 2^-lvl
        int lvl = 1023 - (int)((__double_as_longlong(h) >> 52) & 0x7ff);
        if (lvl >= 0 && lvl < 64) atomicAdd(&s_hist[lvl], 1u);

        d.xm[i] = make_double4(cx.xnew, cy.xnew, cz.xnew, pzm.y);
        d.vt[i] = make_double4(cx.vnew, cy.vnew, cz.vnew, t_next);
        d.ad[i] = make_double4(a1x, a1y, a1z, dnew);
        d.jk[i] = make_double4(j1x, j1y, j1z, 0.0);
        d.tnext[i] = t_next + dnew;                           // exact (dyadic)
    }
    __syncthreads();
    if (threadIdx.x < 64 && s_hist[threadIdx.x]) atomicAdd((unsigned long long *)&d.hist[threadIdx.x], (unsigned long long)s_hist[threadIdx.x]);
    if (threadIdx.x < 2 && s_diag[threadIdx.x]) atomicAdd((unsigned long long *)&d.diag[threadIdx.x], (unsigned long long)s_diag[threadIdx.x]);
    if (dev && blockIdx.x == 0 && threadIdx.x == 0) {
        gd_ctrl *ct = d.ctrl;
        ct->t = t_next;
        ct->steps += 1;
        ct->psteps += n_act;
    }
}

int gdk_correct(gd_ctx *c, double t_next, bool dev)
{
    if (!dev && c->n_act <= 0) return 0;
    const int64_t want = dev ? c->n : c->n_act;
    int64_t blocks = (want + GD_CB - 1) / GD_CB;
    if (dev && blocks > 4 * (int64_t)c->sm_count) blocks = 4 * (int64_t)c->sm_count;
    k_correct_timestep<<<(unsigned)blocks, GD_CB, 0, c->stream>>>(c->d, (int)c->n_act, t_next, c->eta, c->dt_min, c->dt_max,
                                                                  c->halving_mode, dev ? 1 : 0);
    GD_LAUNCH_CHECK(c, "k_correct_timestep");
    return 0;
}
