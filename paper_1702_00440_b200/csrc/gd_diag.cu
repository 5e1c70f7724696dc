// gd_diag.cu -- on-device diagnostics: Lagrange radii, "the radii of spheres containing a certain
// mass fraction of the system" (Fig. 9 P:327 and Fig. 11 P:347 plot them for 0.5 ... 90 % of the mass).
//
// Readings (R23, R24; the paper states neither):
//   centre  the centre of mass of the predicted positions at the current time, sum m x / sum m (or one given by the caller)
//   masses  counted in fixed point, w_i = rint(m_i 2^e) with e = 62 - ceil(log2 n) - (ilogb(max m) + 1), so that mass
//           sums are exact integers, the same in any order: the radius of fraction f is sqrt of the smallest
//           r_i^2 = |x_i - c|^2 whose cumulative weight over { j : r_j^2 <= r_i^2 } reaches max(1, trunc(f W)),
//           W = sum w_i.
// Method: no sort.  Non-negative doubles order like their bit patterns, so the answer's 64-bit key is found by an
// 8-pass radix select (256 bins of exact integer weight per pass, all requested fractions at once).
// Bound: memory bandwidth, 16 B per particle and pass; not on the hot path.
#include "gd_common.cuh"
#include <math.h>

#define GD_LG_THREADS 256
#define GD_LG_MAXF 16

// scratch (u64 words of d.diag_scratch): [0..4) centre x, y, z and total mass (double bits); [4] scale exponent e;
// [5] W; [8 + k] remaining target of fraction k; [24 + k] key prefix of fraction k; [64 ...) hist[k][256]
#define GD_LG_TARGET 8
#define GD_LG_PREFIX 24
#define GD_LG_HIST 64

// sum m, sum m x (fixed order: contiguous slice per thread in index order, then a binary tree) and max m
__global__ void __launch_bounds__(1024) k_diag_moments(gd_dev d, int64_t n, int have_center, double cx, double cy, double cz)
{
    __shared__ double s[4][1024];
    __shared__ double s_max[1024];
    const int tid = threadIdx.x;
    const int64_t per = (n + 1023) / 1024, b = (int64_t)tid * per, e = min(n, b + per);
    double m0 = 0.0, mx = 0.0, my = 0.0, mz = 0.0, mm = 0.0;
    for (int64_t i = b; i < e; ++i) {
        const double2 xy = d.pxy[i], zm = d.pzm[i];
        m0 += zm.y;
        mx += zm.y * xy.x;
        my += zm.y * xy.y;
        mz += zm.y * zm.x;
        mm = fmax(mm, zm.y);
    }
    s[0][tid] = m0; s[1][tid] = mx; s[2][tid] = my; s[3][tid] = mz; s_max[tid] = mm;
    __syncthreads();
    for (int o = 512; o > 0; o >>= 1) {
        if (tid < o) {
            for (int k = 0; k < 4; ++k) s[k][tid] += s[k][tid + o];
            s_max[tid] = fmax(s_max[tid], s_max[tid + o]);
        }
        __syncthreads();
    }
    if (tid == 0) {
        unsigned long long *q = d.diag_scratch;
        const double M = s[0][0];
        if (!have_center) { cx = s[1][0] / M; cy = s[2][0] / M; cz = s[3][0] / M; }
        q[0] = (unsigned long long)__double_as_longlong(cx);
        q[1] = (unsigned long long)__double_as_longlong(cy);
        q[2] = (unsigned long long)__double_as_longlong(cz);
        q[3] = (unsigned long long)__double_as_longlong(M);
        int lg = 0;
        while (((int64_t)1 << lg) < n) ++lg;
        const int e2 = 62 - lg - (ilogb(s_max[0]) + 1);
        q[4] = (unsigned long long)(long long)e2;
        q[5] = 0ull;
    }
}

// keys (bit patterns of r^2) -> d.phi, fixed-point weights -> d.kin, W = sum of the weights (integer: exact in any order)
__global__ void __launch_bounds__(GD_LG_THREADS) k_diag_keys(gd_dev d, int64_t n)
{
    __shared__ unsigned long long s_w;
    if (threadIdx.x == 0) s_w = 0ull;
    __syncthreads();
    const unsigned long long *q = d.diag_scratch;
    const double cx = __longlong_as_double((long long)q[0]), cy = __longlong_as_double((long long)q[1]);
    const double cz = __longlong_as_double((long long)q[2]);
    const int e2 = (int)(long long)q[4];
    const int64_t i = (int64_t)blockIdx.x * GD_LG_THREADS + threadIdx.x;
    if (i < n) {
        const double2 xy = d.pxy[i], zm = d.pzm[i];
        const double dx = __dsub_rn(xy.x, cx), dy = __dsub_rn(xy.y, cy), dz = __dsub_rn(zm.x, cz);
        const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
        const unsigned long long w = (unsigned long long)llrint(ldexp(zm.y, e2));
        reinterpret_cast<unsigned long long *>(d.phi)[i] = (unsigned long long)__double_as_longlong(r2);
        reinterpret_cast<unsigned long long *>(d.kin)[i] = w;
        atomicAdd(&s_w, w);
    }
    __syncthreads();
    if (threadIdx.x == 0 && s_w) atomicAdd(&d.diag_scratch[5], s_w);
}

// targets max(1, trunc(f W)), empty prefixes, clear histograms
__global__ void __launch_bounds__(GD_LG_THREADS) k_diag_targets(gd_dev d, int n_frac, const double *frac)
{
    unsigned long long *q = d.diag_scratch;
    const int tid = threadIdx.x;
    if (tid < n_frac) {
        const double W = (double)q[5];
        double t = frac[tid] * W;
        unsigned long long tu = t >= 18446744073709549568.0 ? 0xffffffffffffffffull : (t > 0.0 ? (unsigned long long)t : 0ull);
        if (tu < 1ull) tu = 1ull;
        if (tu > q[5]) tu = q[5];
        q[GD_LG_TARGET + tid] = tu;
        q[GD_LG_PREFIX + tid] = 0ull;
    }
    for (int k = tid; k < GD_LG_MAXF * 256; k += GD_LG_THREADS) q[GD_LG_HIST + k] = 0ull;
}

// pass p: weight per value of the p-th byte (from the top) among the keys that match each fraction's prefix
__global__ void __launch_bounds__(GD_LG_THREADS) k_diag_hist(gd_dev d, int64_t n, int n_frac, int pass)
{
    extern __shared__ unsigned long long s_hist[];           // [n_frac][256]
    for (int k = threadIdx.x; k < n_frac * 256; k += GD_LG_THREADS) s_hist[k] = 0ull;
    __syncthreads();
    const unsigned long long *q = d.diag_scratch;
    const int shift = 56 - 8 * pass;
    for (int64_t i = (int64_t)blockIdx.x * GD_LG_THREADS + threadIdx.x; i < n; i += (int64_t)gridDim.x * GD_LG_THREADS) {
        const unsigned long long key = reinterpret_cast<const unsigned long long *>(d.phi)[i];
        const unsigned long long w = reinterpret_cast<const unsigned long long *>(d.kin)[i];
        const unsigned long long hi = pass == 0 ? 0ull : key >> (shift + 8);
        const int bin = (int)((key >> shift) & 255ull);
        for (int k = 0; k < n_frac; ++k)
            if (hi == q[GD_LG_PREFIX + k]) atomicAdd(&s_hist[k * 256 + bin], w);
    }
    __syncthreads();
    for (int k = threadIdx.x; k < n_frac * 256; k += GD_LG_THREADS)
        if (s_hist[k]) atomicAdd(&d.diag_scratch[GD_LG_HIST + k], s_hist[k]);
}

// pass p: per fraction, the first bin (ascending) whose cumulative weight reaches the remaining target
__global__ void __launch_bounds__(GD_LG_MAXF) k_diag_pick(gd_dev d, int n_frac, int pass, double *radii)
{
    unsigned long long *q = d.diag_scratch;
    const int k = threadIdx.x;
    if (k >= n_frac) return;
    unsigned long long rem = q[GD_LG_TARGET + k], cum = 0ull;
    int bin = 255;
    for (int b = 0; b < 256; ++b) {
        const unsigned long long h = q[GD_LG_HIST + k * 256 + b];
        if (cum + h >= rem) { bin = b; break; }
        cum += h;
    }
    for (int b = 0; b < 256; ++b) q[GD_LG_HIST + k * 256 + b] = 0ull;
    q[GD_LG_TARGET + k] = rem - cum;
    const unsigned long long prefix = (q[GD_LG_PREFIX + k] << 8) | (unsigned long long)bin;
    q[GD_LG_PREFIX + k] = prefix;
    if (pass == 7) radii[k] = __dsqrt_rn(__longlong_as_double((long long)prefix));
}

// radii_dev[n_frac] and centre_dev[4] = {cx, cy, cz, M} are device staging areas; frac_dev holds the fractions
int gdk_lagrange(gd_ctx *c, const double *center_host, const double *frac_dev, int n_frac, double *radii_dev)
{
    const int have = center_host ? 1 : 0;
    k_diag_moments<<<1, 1024, 0, c->stream>>>(c->d, c->n, have, have ? center_host[0] : 0.0, have ? center_host[1] : 0.0,
                                              have ? center_host[2] : 0.0);
    GD_LAUNCH_CHECK(c, "k_diag_moments");
    const unsigned blocks = (unsigned)((c->n + GD_LG_THREADS - 1) / GD_LG_THREADS);
    k_diag_keys<<<blocks, GD_LG_THREADS, 0, c->stream>>>(c->d, c->n);
    GD_LAUNCH_CHECK(c, "k_diag_keys");
    k_diag_targets<<<1, GD_LG_THREADS, 0, c->stream>>>(c->d, n_frac, frac_dev);
    GD_LAUNCH_CHECK(c, "k_diag_targets");
    const unsigned hb = blocks < (unsigned)(4 * c->sm_count) ? blocks : (unsigned)(4 * c->sm_count);
    for (int pass = 0; pass < 8; ++pass) {
        k_diag_hist<<<hb, GD_LG_THREADS, (size_t)n_frac * 256 * 8, c->stream>>>(c->d, c->n, n_frac, pass);
        GD_LAUNCH_CHECK(c, "k_diag_hist");
        k_diag_pick<<<1, GD_LG_MAXF, 0, c->stream>>>(c->d, n_frac, pass, radii_dev);
        GD_LAUNCH_CHECK(c, "k_diag_pick");
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------------------------------------
// Time-step census ("the distribution of the time steps"; Fig. 13): counts[k] = number of particles whose
// CURRENT block step is 2^-k.  (The histogram of particle steps TAKEN per level is d.hist, kept by the corrector.)
// Integer counts: exact in any order.  Memory-bound, 32 B per particle (the {a, dt} vector); not on the hot path.
__global__ void __launch_bounds__(GD_LG_THREADS) k_diag_census(gd_dev d, int64_t n, unsigned long long *counts)
{
    __shared__ unsigned int s_cnt[64];
    if (threadIdx.x < 64) s_cnt[threadIdx.x] = 0u;
    __syncthreads();
    for (int64_t i = (int64_t)blockIdx.x * GD_LG_THREADS + threadIdx.x; i < n; i += (int64_t)gridDim.x * GD_LG_THREADS) {
        const long long bits = __double_as_longlong(d.ad[i].w);
        const int lvl = 1023 - (int)((bits >> 52) & 0x7ff);
        if (bits > 0 && (bits & 0xfffffffffffffLL) == 0 && lvl >= 0 && lvl < 64) atomicAdd(&s_cnt[lvl], 1u);
    }
    __syncthreads();
    if (threadIdx.x < 64 && s_cnt[threadIdx.x]) atomicAdd(&counts[threadIdx.x], (unsigned long long)s_cnt[threadIdx.x]);
}

int gdk_census(gd_ctx *c, unsigned long long *counts_dev)
{
    GD_CUDA(c, cudaMemsetAsync(counts_dev, 0, 64 * sizeof(unsigned long long), c->stream));
    unsigned blocks = (unsigned)((c->n + GD_LG_THREADS - 1) / GD_LG_THREADS);
    if (blocks > (unsigned)(8 * c->sm_count)) blocks = (unsigned)(8 * c->sm_count);
    k_diag_census<<<blocks, GD_LG_THREADS, 0, c->stream>>>(c->d, c->n, counts_dev);
    GD_LAUNCH_CHECK(c, "k_diag_census");
    return 0;
}

// ---------------------------------------------------------------------------------------------------------------------------
// Density centre and core radius ("the core radius as calculated at T=0", Fig. 12; the paper prints no
// definition: reading R25 = Casertano & Hut 1985 as the direct-summation codes use it):
//   rho_i = (masses of the K - 1 nearest neighbours of i) / (4 pi / 3 r_iK^3),   r_iK = distance to the K-th nearest
//   x_d = sum rho_i x_i / sum rho_i ;   r_c = sqrt( sum rho_i^2 |x_i - x_d|^2 / sum rho_i^2 )
// on the positions predicted to the current time.
// k_diag_knn: one thread per particle i, all n sources streamed through shared memory in tiles; every thread keeps the
// K smallest squared distances seen so far (and the masses that go with them) in registers, ascending, a new source
// entering only if strictly closer than the K-th (so equal distances keep index order).  Every operation is rounded
// separately in the order the definition is written, so r^2, the choice of neighbours and rho_i are the doubles a
// plain evaluation gives.  ALU-bound: n^2 x ~10 FP64 instructions; a diagnostic, not on the hot path.
#define GD_KNN_MAXK 8
#define GD_KNN_TILE 256

template <int K>
__global__ void __launch_bounds__(GD_KNN_TILE) k_diag_knn(gd_dev d, int64_t n, double *rho)
{
    static_assert(K >= 2 && K <= GD_KNN_MAXK, "k_diag_knn: 2 <= K <= GD_KNN_MAXK");
    __shared__ double2 s_xy[GD_KNN_TILE], s_zm[GD_KNN_TILE];
    const int64_t i = (int64_t)blockIdx.x * GD_KNN_TILE + threadIdx.x;
    const bool live = i < n;
    const double2 xy = live ? d.pxy[i] : make_double2(0.0, 0.0), zm = live ? d.pzm[i] : make_double2(0.0, 0.0);
    double r2k[K], mk[K];                                    // only the K nearest are kept: a source enters if closer than the K-th
#pragma unroll
    for (int k = 0; k < K; ++k) { r2k[k] = __longlong_as_double(0x7ff0000000000000LL); mk[k] = 0.0; }
    for (int64_t j0 = 0; j0 < n; j0 += GD_KNN_TILE) {
        const int64_t j = j0 + threadIdx.x;
        __syncthreads();
        if (j < n) { s_xy[threadIdx.x] = d.pxy[j]; s_zm[threadIdx.x] = d.pzm[j]; }
        __syncthreads();
        const int cnt = (int)min((int64_t)GD_KNN_TILE, n - j0);
        for (int t = 0; t < cnt; ++t) {
            const double2 sxy = s_xy[t], szm = s_zm[t];
            const double dx = __dsub_rn(sxy.x, xy.x), dy = __dsub_rn(sxy.y, xy.y), dz = __dsub_rn(szm.x, zm.x);
            const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
            if (r2 < r2k[K - 1] && j0 + t != i) {
                // insert, keeping the list ascending; an equal distance goes behind the ones already there
                double cr = r2, cm = szm.y;
#pragma unroll
                for (int k = 0; k < K; ++k) {
                    if (cr < r2k[k]) {
                        const double tr = r2k[k], tm = mk[k];
                        r2k[k] = cr; mk[k] = cm;
                        cr = tr; cm = tm;
                    }
                }
            }
        }
    }
    if (!live) return;
    // the K - 1 nearest masses, nearest first; the sphere through the K-th
    double mass = 0.0;
#pragma unroll
    for (int k = 0; k < K - 1; ++k) mass = __dadd_rn(mass, mk[k]);
    const double r = __dsqrt_rn(r2k[K - 1]);
    const double c43 = 4.0 * 3.141592653589793 / 3.0;
    rho[i] = __ddiv_rn(mass, __dmul_rn(__dmul_rn(__dmul_rn(c43, r), r), r));
}

// x_d and r_c from rho (fixed order: a contiguous slice per thread in index order, then a binary tree) -> out[0..2] = x_d,
// out[3] = r_c, out[4] = sum rho, out[5] = largest rho_i (+inf when a particle has K others on its own point: gd_core_radius reports that)
__global__ void __launch_bounds__(1024) k_diag_core(gd_dev d, int64_t n, const double *rho, double *out)
{
    __shared__ double s[4][1024];
    __shared__ double s_c[3];
    const int tid = threadIdx.x;
    const int64_t per = (n + 1023) / 1024, b = (int64_t)tid * per, e = min(n, b + per);
    double w0 = 0.0, wx = 0.0, wy = 0.0, wz = 0.0, wm = 0.0;
    for (int64_t i = b; i < e; ++i) {
        const double2 xy = d.pxy[i], zm = d.pzm[i];
        const double r = rho[i];
        w0 += r; wx += r * xy.x; wy += r * xy.y; wz += r * zm.x;
        wm = fmax(wm, r);
    }
    s[0][tid] = w0; s[1][tid] = wx; s[2][tid] = wy; s[3][tid] = wz;
    __syncthreads();
    for (int o = 512; o > 0; o >>= 1) {
        if (tid < o) for (int k = 0; k < 4; ++k) s[k][tid] += s[k][tid + o];
        __syncthreads();
    }
    if (tid == 0) {
        s_c[0] = s[1][0] / s[0][0]; s_c[1] = s[2][0] / s[0][0]; s_c[2] = s[3][0] / s[0][0];
        out[0] = s_c[0]; out[1] = s_c[1]; out[2] = s_c[2]; out[4] = s[0][0];
    }
    __syncthreads();
    const double cx = s_c[0], cy = s_c[1], cz = s_c[2];
    double num = 0.0, den = 0.0;
    for (int64_t i = b; i < e; ++i) {
        const double2 xy = d.pxy[i], zm = d.pzm[i];
        const double r = rho[i], w = r * r;
        const double dx = xy.x - cx, dy = xy.y - cy, dz = zm.x - cz;
        num += w * ((dx * dx + dy * dy) + dz * dz);
        den += w;
    }
    __syncthreads();
    s[0][tid] = num; s[1][tid] = den; s[2][tid] = wm;
    __syncthreads();
    for (int o = 512; o > 0; o >>= 1) {
        if (tid < o) { s[0][tid] += s[0][tid + o]; s[1][tid] += s[1][tid + o]; s[2][tid] = fmax(s[2][tid], s[2][tid + o]); }
        __syncthreads();
    }
    if (tid == 0) { out[3] = sqrt(s[0][0] / s[1][0]); out[5] = s[2][0]; }
}

// rho -> rho_dev (the caller's [n] array, or the internal scratch d.phi when NULL); out_dev[6] as k_diag_core writes it
int gdk_core_radius(gd_ctx *c, int K, double *rho_dev, double *out_dev)
{
    double *rho = rho_dev ? rho_dev : c->d.phi;
    const unsigned blocks = (unsigned)((c->n + GD_KNN_TILE - 1) / GD_KNN_TILE);
    switch (K) {
#define GD_KNN_CASE(k) case k: k_diag_knn<k><<<blocks, GD_KNN_TILE, 0, c->stream>>>(c->d, c->n, rho); break;
        GD_KNN_CASE(2) GD_KNN_CASE(3) GD_KNN_CASE(4) GD_KNN_CASE(5) GD_KNN_CASE(6) GD_KNN_CASE(7) GD_KNN_CASE(8)
#undef GD_KNN_CASE
        default: return -1;                                  // GD_EINVAL: gd_core_radius checks the range before
    }
    GD_LAUNCH_CHECK(c, "k_diag_knn");
    k_diag_core<<<1, 1024, 0, c->stream>>>(c->d, c->n, rho, out_dev);
    GD_LAUNCH_CHECK(c, "k_diag_core");
    return 0;
}
