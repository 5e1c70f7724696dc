// gd_probe.cu -- register-only DFMA loop: measures the FP64 rate that bounds the force kernels ("alu" roofline).
// 16 independent FMA chains per thread, 4 x 256-thread CTAs per SM, no memory traffic inside the loop.
#include "gd_common.cuh"

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
