// gd_energy_static.cu -- gd_energy_static: the total energy (Eq. 2, softened like Eq. 3, DESIGN.md
// reading R8) for callers that are not able to allocate device memory.
//
// Who this is for.  Every other call of this library works out of a workspace that the caller got from cudaMalloc (or
// from an allocator built on it), and gd_init pins host memory besides.  Some programs that want an energy cannot do
// that at the moment they want it:
//   * a driver that handed all free HBM to its own pool at start-up -- a later cudaMalloc just returns "out of memory";
//   * a time-critical loop: cudaMalloc / cudaFree make the whole device wait, which stalls every other stream;
//   * a plug-in inside an application whose rules forbid driver allocations once it is running.
// For them this file keeps the scratch of the energy reduction (one {K, U} pair per tile of 256 particles) in a
// file-scope __device__ array of fixed size, which the CUDA runtime places on every GPU that loads the library and
// keeps there until the process exits: GD_ENERGY_STATIC_MAX_N / 256 pairs = 128 KiB per GPU.  The call itself runs
// no cudaMalloc, cudaFree, cudaHostAlloc, event or graph creation, and no library routine that allocates; inputs and
// the two-double result are the caller's own device buffers.
//
// What a user has to know:
//   * n is limited to GD_ENERGY_STATIC_MAX_N; larger systems are refused (GD_EINVAL), never truncated.
//   * The first call on each GPU looks up the device address of the array (cudaGetSymbolAddress, with that GPU
//     current; the array's name as host code sees it is only a handle, not something a kernel may dereference).  That
//     first call may also make the runtime load this library's device code.  Make it outside any stream capture.
//   * All calls on one GPU share the one array and it still holds what the previous call left.  Nothing in it has to
//     start at zero: a call reads only the slots that its own first kernel has written.  Calls in one stream run one
//     after the other and are safe; two calls that can run at the same time on one GPU (different streams, no event
//     between them) overwrite each other's partial sums -- order them yourself.
//
//   k_energy_static_pairs  the pair loop of k_energy_pairs (gd_energy.cu) reading the caller's plain m [n], x [n,3],
//                          v [n,3] instead of packed records, with the CTA's 256 sinks folded to one {K, U} pair
//   k_energy_static_fold   one CTA adds the pairs in a fixed order -> out[0] = K, out[1] = U
#include "gd_common.cuh"
#include "../../include/gravidy_b200.h"
#include <math.h>
#include <mutex>
#include <stdio.h>

#define GD_ES_THREADS 128
#define GD_ES_BI 2
#define GD_ES_TILE (GD_ES_THREADS * GD_ES_BI)
#define GD_ES_MAX_TILES (GD_ENERGY_STATIC_MAX_N / GD_ES_TILE)
#define GD_ES_FOLD_THREADS 1024
#define GD_ES_MAX_DEVICES 64

static_assert(GD_ENERGY_STATIC_MAX_N % GD_ES_TILE == 0, "the size limit is a whole number of tiles");

// The scratch itself: {K, U} of tile t at [2 t], [2 t + 1].  In host code this name is a stand-in for the symbol and
// must only be handed to cudaGetSymbolAddress; kernels get the address that call returns.
static __device__ __align__(256) double g_es_scratch[2 * GD_ES_MAX_TILES];

static std::mutex g_es_mutex;
static double *g_es_addr[GD_ES_MAX_DEVICES];          // device address of g_es_scratch on GPU k, once looked up
static thread_local char g_es_err[384] = "";

static int gd_es_fail(int code, const char *msg)
{
    snprintf(g_es_err, sizeof g_es_err, "gd_energy_static: %s", msg);
    return code;
}

static int gd_es_fail_cuda(cudaError_t e, const char *what)
{
    snprintf(g_es_err, sizeof g_es_err, "gd_energy_static: CUDA error %d (%s) at %s", (int)e, cudaGetErrorString(e), what);
    return GD_ECUDA;
}

// The once-per-GPU set-up: the address of g_es_scratch on the GPU that is current in the calling thread.
static int gd_es_scratch(double **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return gd_es_fail_cuda(e, "cudaGetDevice");
    if (dev < 0 || dev >= GD_ES_MAX_DEVICES) return gd_es_fail(GD_EINVAL, "device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_es_mutex);
    if (!g_es_addr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_es_scratch);
        if (e != cudaSuccess) return gd_es_fail_cuda(e, "cudaGetSymbolAddress(g_es_scratch)");
        if (!p) return gd_es_fail(GD_ECUDA, "cudaGetSymbolAddress returned a null address");
        g_es_addr[dev] = static_cast<double *>(p);
    }
    *out = g_es_addr[dev];
    return GD_OK;
}

// 1/sqrt(s) as k_energy_pairs takes it (hardware estimate + one third-order step; s == 0, the coincident pair at
// eps = 0, counts as no interaction).  Restated here so that gd_energy.cu stays as it is.
__device__ __forceinline__ double gd_es_rsqrt(double s)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(s));
    if (__double2hiint(s) == 0) y = 0.0;
    double t = s * y;
    double e = fma(-t, y, 1.0);
    double p = fma(0.375, e, 0.5);
    double g = y * e;
    return fma(g, p, y);
}

// CTA `tile` owns sinks [256 tile, 256 tile + 256) and walks the source tiles from its own to the last one (pairs
// j > i only).  Particles at or beyond n are zero-mass points at the origin: they add exact zeros.
__global__ void __launch_bounds__(GD_ES_THREADS)
k_energy_static_pairs(const double *__restrict__ m, const double *__restrict__ x, const double *__restrict__ v,
                      int64_t n, int n_tiles, double eps2, double *__restrict__ scratch)
{
    __shared__ double2 s_xy[GD_ES_TILE];
    __shared__ double2 s_zm[GD_ES_TILE];
    __shared__ double s_k[GD_ES_THREADS], s_u[GD_ES_THREADS];
    const int tid = threadIdx.x;
    const int my_tile = blockIdx.x;
    int64_t i[GD_ES_BI];
    double xi[GD_ES_BI], yi[GD_ES_BI], zi[GD_ES_BI], phi[GD_ES_BI];
#pragma unroll
    for (int b = 0; b < GD_ES_BI; ++b) {
        i[b] = (int64_t)my_tile * GD_ES_TILE + b * GD_ES_THREADS + tid;
        const bool in = i[b] < n;
        xi[b] = in ? x[3 * i[b]] : 0.0;
        yi[b] = in ? x[3 * i[b] + 1] : 0.0;
        zi[b] = in ? x[3 * i[b] + 2] : 0.0;
        phi[b] = 0.0;
    }
    for (int t = my_tile; t < n_tiles; ++t) {
        const int64_t j0 = (int64_t)t * GD_ES_TILE;
        __syncthreads();
        for (int e = tid; e < GD_ES_TILE; e += GD_ES_THREADS) {
            const int64_t j = j0 + e;
            const bool in = j < n;
            s_xy[e] = make_double2(in ? x[3 * j] : 0.0, in ? x[3 * j + 1] : 0.0);
            s_zm[e] = make_double2(in ? x[3 * j + 2] : 0.0, in ? m[j] : 0.0);
        }
        __syncthreads();
        if (t == my_tile) {
#pragma unroll 2
            for (int jj = 0; jj < GD_ES_TILE; ++jj) {
                double2 xy = s_xy[jj], zm = s_zm[jj];
#pragma unroll
                for (int b = 0; b < GD_ES_BI; ++b) {
                    double rx = xy.x - xi[b], ry = xy.y - yi[b], rz = zm.x - zi[b];
                    double s = fma(rx, rx, fma(ry, ry, fma(rz, rz, eps2)));
                    double mq = zm.y * gd_es_rsqrt(s);
                    phi[b] += (j0 + jj > i[b]) ? mq : 0.0;
                }
            }
        } else {
#pragma unroll 2
            for (int jj = 0; jj < GD_ES_TILE; ++jj) {
                double2 xy = s_xy[jj], zm = s_zm[jj];
#pragma unroll
                for (int b = 0; b < GD_ES_BI; ++b) {
                    double rx = xy.x - xi[b], ry = xy.y - yi[b], rz = zm.x - zi[b];
                    double s = fma(rx, rx, fma(ry, ry, fma(rz, rz, eps2)));
                    phi[b] = fma(zm.y, gd_es_rsqrt(s), phi[b]);
                }
            }
        }
    }
    double k = 0.0, u = 0.0;
#pragma unroll
    for (int b = 0; b < GD_ES_BI; ++b) {
        if (i[b] < n) {
            const double mi = m[i[b]];
            const double vx = v[3 * i[b]], vy = v[3 * i[b] + 1], vz = v[3 * i[b] + 2];
            u += mi * phi[b];
            k += 0.5 * mi * (vx * vx + vy * vy + vz * vz);
        }
    }
    s_k[tid] = k;
    s_u[tid] = u;
    __syncthreads();
    for (int o = GD_ES_THREADS / 2; o > 0; o >>= 1) {
        if (tid < o) { s_k[tid] += s_k[tid + o]; s_u[tid] += s_u[tid + o]; }
        __syncthreads();
    }
    if (tid == 0) { scratch[2 * my_tile] = s_k[0]; scratch[2 * my_tile + 1] = s_u[0]; }
}

// Thread t adds tiles t, t + 1024, ... in that order, then a binary tree over the threads: the order of summation
// depends on n alone.  Reads scratch[0 .. 2 n_tiles) only -- exactly what the kernel above has just written.
__global__ void __launch_bounds__(GD_ES_FOLD_THREADS)
k_energy_static_fold(const double *__restrict__ scratch, int n_tiles, double *__restrict__ out)
{
    __shared__ double s_k[GD_ES_FOLD_THREADS], s_u[GD_ES_FOLD_THREADS];
    const int tid = threadIdx.x;
    double k = 0.0, u = 0.0;
    for (int t = tid; t < n_tiles; t += GD_ES_FOLD_THREADS) { k += scratch[2 * t]; u += scratch[2 * t + 1]; }
    s_k[tid] = k;
    s_u[tid] = u;
    __syncthreads();
    for (int o = GD_ES_FOLD_THREADS / 2; o > 0; o >>= 1) {
        if (tid < o) { s_k[tid] += s_k[tid + o]; s_u[tid] += s_u[tid + o]; }
        __syncthreads();
    }
    if (tid == 0) { out[0] = s_k[0]; out[1] = -s_u[0]; }
}

extern "C" const char *gd_energy_static_last_error(void) { return g_es_err; }

extern "C" int gd_energy_static(int64_t n, const double *m_dev, const double *x_dev, const double *v_dev, double eps,
                                double *out_dev, void *cuda_stream)
{
    // argument checks come before the first CUDA call
    if (n < 1) return gd_es_fail(GD_EINVAL, "n < 1");
    if (n > (int64_t)GD_ENERGY_STATIC_MAX_N) {
        char msg[320];
        snprintf(msg, sizeof msg, "n = %lld is beyond GD_ENERGY_STATIC_MAX_N = %d, the size the built-in scratch array "
                 "holds (use gd_init + gd_energy with a workspace for larger systems)", (long long)n, GD_ENERGY_STATIC_MAX_N);
        return gd_es_fail(GD_EINVAL, msg);
    }
    if (!m_dev || !x_dev || !v_dev || !out_dev) return gd_es_fail(GD_EINVAL, "NULL pointer");
    if (!(eps >= 0.0) || !isfinite(eps)) return gd_es_fail(GD_EINVAL, "eps must be finite and >= 0");

    double *scratch = nullptr;
    int rc = gd_es_scratch(&scratch);
    if (rc) return rc;

    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const int n_tiles = (int)((n + GD_ES_TILE - 1) / GD_ES_TILE);
    k_energy_static_pairs<<<(unsigned)n_tiles, GD_ES_THREADS, 0, stream>>>(m_dev, x_dev, v_dev, n, n_tiles, eps * eps, scratch);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return gd_es_fail_cuda(e, "k_energy_static_pairs");
    k_energy_static_fold<<<1, GD_ES_FOLD_THREADS, 0, stream>>>(scratch, n_tiles, out_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) return gd_es_fail_cuda(e, "k_energy_static_fold");
    return GD_OK;
}
