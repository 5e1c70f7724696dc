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
#include "gd_hermite.cuh"

#define GD_CB 128
#ifndef GD_CB_MIN
#define GD_CB_MIN 8              // resident CTAs per SM the compiler is asked to fit (register cap 65536 / (GD_CB x GD_CB_MIN))
#endif

__global__ void __launch_bounds__(GD_CB, GD_CB_MIN)
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

        const double a1v[3] = {a1x, a1y, a1z}, j1v[3] = {j1x, j1y, j1z};
        const gd_corrected r = gd_correct_particle(pxy.x, pxy.y, pzm.x, pvxy.x, pvxy.y, pvz, ad, jk, a1v, j1v, t_next, eta, dt_min,
                                                   dt_max, halving_mode);
        const double dnew = r.dt;
        if (r.flags & 1) atomicAdd(&s_diag[0], 1u);
        if (r.flags & 2) atomicAdd(&s_diag[1], 1u);

        // level of the step just taken: h = 2^-lvl
        int lvl = gd_step_level(ad.w);
        if (lvl >= 0 && lvl < 64) atomicAdd(&s_hist[lvl], 1u);

        d.xm[i] = make_double4(r.x, r.y, r.z, pzm.y);
        d.vt[i] = make_double4(r.vx, r.vy, r.vz, t_next);
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
