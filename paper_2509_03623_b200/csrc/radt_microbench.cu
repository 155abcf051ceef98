// radt_microbench.cu -- M1: issue-rate micro-benchmarks of the pipes the march is bounded by
// (MUFU.EX2, FFMA, DFMA, packed FFMA2), measured at the clock the GPU actually runs at.
// The roofline denominators in bench.py come from these.
#include "radt_dev.cuh"
#include "radt_kernels.h"

#define MB_ITERS 4096
#define MB_ILP 8

template <int KIND>
__global__ void __launch_bounds__(1024) k_pipe(float *sink, unsigned long long *clk, float seed)
{
    unsigned long long t0 = 0, c0 = 0;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
        c0 = clock64();
    }
    float acc = 0.f;
    if (KIND == 0) {
        float v[MB_ILP];
#pragma unroll
        for (int i = 0; i < MB_ILP; ++i) v[i] = seed + 0.001f * (float)(threadIdx.x + i);
        for (int it = 0; it < MB_ITERS; ++it) {
#pragma unroll
            for (int i = 0; i < MB_ILP; ++i) v[i] = ex2_approx(v[i]);   // converges to a fixed point; still issues MUFU
        }
#pragma unroll
        for (int i = 0; i < MB_ILP; ++i) acc += v[i];
    } else if (KIND == 1) {
        float v[MB_ILP];
        float a = 1.0f + seed * 1e-7f, b = seed * 1e-9f;
#pragma unroll
        for (int i = 0; i < MB_ILP; ++i) v[i] = seed + (float)(threadIdx.x + i);
        for (int it = 0; it < MB_ITERS; ++it) {
#pragma unroll
            for (int i = 0; i < MB_ILP; ++i) v[i] = fmaf(v[i], a, b);
        }
#pragma unroll
        for (int i = 0; i < MB_ILP; ++i) acc += v[i];
    } else if (KIND == 2) {
        double v[MB_ILP];
        double a = 1.0 + (double)seed * 1e-12, b = (double)seed * 1e-15;
#pragma unroll
        for (int i = 0; i < MB_ILP; ++i) v[i] = (double)seed + (double)(threadIdx.x + i);
        for (int it = 0; it < MB_ITERS; ++it) {
#pragma unroll
            for (int i = 0; i < MB_ILP; ++i) v[i] = fma(v[i], a, b);
        }
#pragma unroll
        for (int i = 0; i < MB_ILP; ++i) acc += (float)v[i];
    } else {
        unsigned long long v[MB_ILP];
        float2 af = make_float2(1.0f + seed * 1e-7f, 1.0f - seed * 1e-7f), bf = make_float2(seed * 1e-9f, -seed * 1e-9f);
        unsigned long long a = *reinterpret_cast<unsigned long long *>(&af), b = *reinterpret_cast<unsigned long long *>(&bf);
#pragma unroll
        for (int i = 0; i < MB_ILP; ++i) {
            float2 f = make_float2(seed + (float)(threadIdx.x + i), seed - (float)i);
            v[i] = *reinterpret_cast<unsigned long long *>(&f);
        }
        for (int it = 0; it < MB_ITERS; ++it) {
#pragma unroll
            for (int i = 0; i < MB_ILP; ++i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(v[i]) : "l"(a), "l"(b));
        }
#pragma unroll
        for (int i = 0; i < MB_ILP; ++i) {
            float2 f = *reinterpret_cast<float2 *>(&v[i]);
            acc += f.x + f.y;
        }
    }
    if (acc == 123.456f) sink[0] = acc;   // keep the chains alive
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        unsigned long long t1, c1 = clock64();
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
        clk[0] = c1 - c0;
        clk[1] = t1 - t0;
    }
}

cudaError_t radt_run_pipe_peak(int kind, double *ops_per_s, double *clock_mhz)
{
    int dev = 0, sms = 0;
    cudaError_t e;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    float *sink = nullptr;
    unsigned long long *clk = nullptr;
    if ((e = cudaMalloc(&sink, 16)) != cudaSuccess) return e;
    if ((e = cudaMalloc(&clk, 16)) != cudaSuccess) { cudaFree(sink); return e; }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    int grid = sms * 2;
    float best_ms = 1e30f;
    unsigned long long h[2] = { 0, 0 }, hb[2] = { 0, 1 };
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0, 0);
        switch (kind) {
        case 0: k_pipe<0><<<grid, 1024>>>(sink, clk, 0.5f); break;
        case 1: k_pipe<1><<<grid, 1024>>>(sink, clk, 0.5f); break;
        case 2: k_pipe<2><<<grid, 1024>>>(sink, clk, 0.5f); break;
        default: k_pipe<3><<<grid, 1024>>>(sink, clk, 0.5f); break;
        }
        cudaEventRecord(e1, 0);
        if ((e = cudaEventSynchronize(e1)) != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        cudaMemcpy(h, clk, sizeof(h), cudaMemcpyDeviceToHost);
        if (rep > 0 && ms < best_ms) { best_ms = ms; hb[0] = h[0]; hb[1] = h[1]; }
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    double lane_ops = (double)grid * 1024.0 * (double)MB_ITERS * (double)MB_ILP * (kind == 3 ? 2.0 : 1.0);
    *ops_per_s = lane_ops / ((double)best_ms * 1e-3);
    *clock_mhz = hb[1] ? (double)hb[0] / (double)hb[1] * 1e3 : 0.0;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    cudaFree(clk);
    return e;
}
