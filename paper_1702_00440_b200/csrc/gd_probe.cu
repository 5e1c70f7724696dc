// gd_probe.cu -- register-only DFMA loop: measures the FP64 rate that bounds the force kernels ("alu" roofline).
// 16 independent FMA chains per thread, 4 x 256-thread CTAs per SM, no memory traffic inside the loop.
#include "gd_common.cuh"
#include "gd_hermite.cuh"

#define GD_PROBE_CHAINS 16
#define GD_PROBE_THREADS 256

__global__ void __launch_bounds__(GD_PROBE_THREADS) k_fp64_probe(int iters, double seed, double *sink)
{
    double a[GD_PROBE_CHAINS];
    const double m = 1.0 - 1e-9 * seed, c = 1e-9 * (threadIdx.x + 1);
#pragma unroll
    for (int k = 0; k < GD_PROBE_CHAINS; ++k) a[k] = seed + k;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < GD_PROBE_CHAINS; ++k) a[k] = fma(a[k], m, c);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < GD_PROBE_CHAINS; ++k) s += a[k];
    if (s == 123.456) sink[0] = s;          // keeps the loop alive; practically never true
}

int gdk_fp64_probe(int iters, double *flops, double *ms)
{
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -1;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1;
    double *sink = nullptr;
    if (cudaMalloc(&sink, sizeof(double)) != cudaSuccess) return -1;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int blocks = sms * 8;
    k_fp64_probe<<<blocks, GD_PROBE_THREADS>>>(iters / 8 + 1, 1.0, sink);          // warm-up
    cudaEventRecord(e0);
    k_fp64_probe<<<blocks, GD_PROBE_THREADS>>>(iters, 1.0, sink);
    cudaEventRecord(e1);
    cudaError_t e = cudaEventSynchronize(e1);
    float t = 0.f;
    cudaEventElapsedTime(&t, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) return -1;
    if (ms) *ms = t;
    if (flops) *flops = 2.0 * GD_PROBE_CHAINS * (double)iters * GD_PROBE_THREADS * blocks / (t * 1e-3);
    return 0;
}

// ---- self-test of gd_div_const (gd_hermite.cuh) against the division routine on random operands --------------------
// operand k of the stream `seed`: a splitmix64 word -> sign, a binary exponent in [-960, 960) (so that both branches of
// gd_div_const are exercised), 52 random significand bits
__global__ void __launch_bounds__(256) k_selftest_div_const(long long n, unsigned long long seed, unsigned long long *mismatch)
{
    unsigned long long bad = 0;
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (long long)gridDim.x * blockDim.x) {
        unsigned long long z = seed + 0x9e3779b97f4a7c15ull * (unsigned long long)(k + 1);
        z = (z ^ (z >> 30)) * 0xbf58476d1ce4e5b9ull;
        z = (z ^ (z >> 27)) * 0x94d049bb133111ebull;
        z ^= z >> 31;
        const unsigned long long frac = z & 0xfffffffffffffull, sign = z >> 63;
        const long long e = 1023 - 960 + (long long)((z >> 52) & 0x7ff) % 1920;
        const double x = __longlong_as_double((long long)((sign << 63) | ((unsigned long long)e << 52) | frac));
        bad += __double_as_longlong(gd_div_const<6>(x)) != __double_as_longlong(__ddiv_rn(x, 6.0));
        bad += __double_as_longlong(gd_div_const<24>(x)) != __double_as_longlong(__ddiv_rn(x, 24.0));
        bad += __double_as_longlong(gd_div_const<120>(x)) != __double_as_longlong(__ddiv_rn(x, 120.0));
    }
    if (bad) atomicAdd(mismatch, bad);
}

int gdk_selftest_div_const(long long n, unsigned long long seed, long long *mismatches)
{
    unsigned long long *d = nullptr, h = 0;
    if (cudaMalloc(&d, sizeof h) != cudaSuccess) return -1;
    cudaMemset(d, 0, sizeof h);
    k_selftest_div_const<<<1184, 256>>>(n, seed, d);
    cudaError_t e = cudaMemcpy(&h, d, sizeof h, cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) return -1;
    *mismatches = (long long)h;
    return 0;
}
