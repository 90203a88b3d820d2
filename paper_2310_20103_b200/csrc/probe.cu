// Measurement helper (not part of the method): register-resident FP64 issue-rate probes.  They give the
// FP64 tensor (DMMA) and FP64 FMA peaks of the device under its own clocks; DESIGN.md uses the DMMA figure as
// the roofline denominator of the contraction kernels next to the MEASURED_PEAKS.json-derived one.
#include "gwl_internal.h"

namespace gwl {

namespace {

__global__ void __launch_bounds__(256) k_probe_dmma(int iters, double* sink) {
    double c[8][2];
#pragma unroll
    for (int u = 0; u < 8; ++u) c[u][0] = c[u][1] = 0.0;
    double a = 1.0 + 1e-9 * threadIdx.x, b = 1.0 - 1e-9 * threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                         : "+d"(c[u][0]), "+d"(c[u][1])
                         : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int u = 0; u < 8; ++u) s += c[u][0] + c[u][1];
    if (s == 123.456) sink[0] = s;
}

__global__ void __launch_bounds__(256) k_probe_dfma(int iters, double* sink) {
    double x[16];
#pragma unroll
    for (int u = 0; u < 16; ++u) x[u] = 1e-3 * (u + threadIdx.x);
    const double a = 0.999999, b = 1e-7;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 16; ++u) x[u] = fma(x[u], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int u = 0; u < 16; ++u) s += x[u];
    if (s == 123.456) sink[0] = s;
}

}  // namespace

cudaError_t probe_fp64_peak(int kind, double* tflops) {
    int dev = 0, n_sm = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    double* sink = nullptr;
    e = cudaMalloc(&sink, 8);
    if (e != cudaSuccess) return e;
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0);
    cudaEventCreate(&t1);
    const int blocks = n_sm * 4, threads = 256;
    const int iters = kind == 0 ? 20000 : 40000;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(t0);
        if (kind == 0)
            k_probe_dmma<<<blocks, threads>>>(iters, sink);
        else
            k_probe_dfma<<<blocks, threads>>>(iters, sink);
        cudaEventRecord(t1);
        e = cudaEventSynchronize(t1);
        if (e != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, t0, t1);
        double flop;
        if (kind == 0)
            flop = (double)blocks * (threads / 32) * (double)iters * 8.0 * 512.0;  // 8x8x4 MACs x 2
        else
            flop = (double)blocks * threads * (double)iters * 16.0 * 2.0;
        const double tf = flop / (ms * 1e-3) / 1e12;
        if (rep > 0 && tf > best) best = tf;
    }
    cudaEventDestroy(t0);
    cudaEventDestroy(t1);
    cudaFree(sink);
    if (e == cudaSuccess) e = cudaGetLastError();
    *tflops = best;
    return e;
}

}  // namespace gwl
