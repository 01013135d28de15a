// Register-only FP64 peak probes (roofline denominators for bench.py; SURVEY build plan
// step 0).  kind 0: independent DFMA chains on the FP64 FMA pipe.  kind 1: independent
// mma.sync.m8n8k4.f64 chains (SASS DMMA.8x8x4 on sm_100a).  No memory traffic.
#include "chase_internal.h"

namespace chase {
namespace {

constexpr int kChains = 8;

__global__ void __launch_bounds__(256) dfma_probe(int iters, double seed, double *sink) {
    double x[kChains];
#pragma unroll
    for (int i = 0; i < kChains; ++i) x[i] = seed + threadIdx.x * 1e-9 + i;
    const double a = 1.0 - 1e-12, b = 1e-12;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int i = 0; i < kChains; ++i) x[i] = fma(x[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < kChains; ++i) s += x[i];
    if (s == 123.456) sink[0] = s;   // never true; keeps the chains alive
}

__device__ __forceinline__ void dmma884(double &d0, double &d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(256) dmma_probe(int iters, double seed, double *sink) {
    double c0[kChains], c1[kChains];
#pragma unroll
    for (int i = 0; i < kChains; ++i) { c0[i] = seed + i; c1[i] = seed - i; }
    const double a = 1e-3 * (threadIdx.x & 3), b = 1e-3 * (threadIdx.x >> 2);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int i = 0; i < kChains; ++i) dmma884(c0[i], c1[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < kChains; ++i) s += c0[i] + c1[i];
    if (s == 123.456) sink[0] = s;
}

}  // namespace
}  // namespace chase

extern "C" int chase_fp64_peak_probe(int kind, int iters, double *gflops) {
    using namespace chase;
    if (!gflops || iters <= 0 || (kind != 0 && kind != 1)) return CHASE_ERR_ARG;
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return (int)e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return (int)e;
    double *sink = nullptr;
    if ((e = cudaMalloc(&sink, sizeof(double))) != cudaSuccess) return (int)e;
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0);
    cudaEventCreate(&t1);
    const int grid = sms * 4, block = 256;
    for (int rep = 0; rep < 2; ++rep) {   // rep 0 = warm-up
        cudaEventRecord(t0);
        if (kind == 0) dfma_probe<<<grid, block>>>(iters, 1.0, sink);
        else dmma_probe<<<grid, block>>>(iters, 1.0, sink);
        count_launch();
        cudaEventRecord(t1);
        if ((e = cudaEventSynchronize(t1)) != cudaSuccess) break;
    }
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, t0, t1);
    cudaEventDestroy(t0);
    cudaEventDestroy(t1);
    cudaFree(sink);
    if (e != cudaSuccess) return (int)e;
    const double per_thread_iter = 4.0 * kChains;   // instructions per thread (or per warp) per iteration
    double flops;
    if (kind == 0) flops = (double)grid * block * iters * per_thread_iter * 2.0;
    else flops = (double)grid * (block / 32) * iters * per_thread_iter * 512.0;
    *gflops = flops / (ms * 1e-3) * 1e-9;
    return 0;
}
