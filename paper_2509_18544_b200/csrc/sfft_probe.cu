// sfft_probe.cu -- FP64 rate probes: the ALU roofline bench.py divides by is
// MEASURED on the box, since MEASURED_PEAKS.json has no FP64 entry.  kind 0: register-resident
// DFMA chains; kind 1: DMMA m8n8k4 (the instruction the Cholesky trailing update uses).
#include "sfft_internal.h"

namespace sfft {

__global__ void __launch_bounds__(256) probe_dfma_kernel(double *out, int iters, double seed) {
    double a[8];
#pragma unroll
    for (int k = 0; k < 8; k++) a[k] = seed + k + threadIdx.x * 1e-3;
    const double m = 0.999999, c = 1e-9;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int r = 0; r < 8; r++)
#pragma unroll
            for (int k = 0; k < 8; k++) a[k] = fma(a[k], m, c);
    }
    double s = 0;
#pragma unroll
    for (int k = 0; k < 8; k++) s += a[k];
    if (s == 12345.678) out[0] = s; // never true; keeps the chain alive
}

__global__ void __launch_bounds__(256) probe_dmma_kernel(double *out, int iters, double seed) {
    double d[8][2];
#pragma unroll
    for (int k = 0; k < 8; k++) { d[k][0] = seed; d[k][1] = seed + k; }
    const double a = 1e-3 * (threadIdx.x & 7), b = 1e-3;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int r = 0; r < 4; r++)
#pragma unroll
            for (int k = 0; k < 8; k++)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                             : "+d"(d[k][0]), "+d"(d[k][1]) : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int k = 0; k < 8; k++) s += d[k][0] + d[k][1];
    if (s == 12345.678) out[0] = s;
}

cudaError_t run_probe_fp64(int kind, int iters, double *tflops) {
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    double *out = nullptr;
    e = cudaMalloc(&out, sizeof(double));
    if (e != cudaSuccess) return e;
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int blocks = sms * 8, threads = 256;
    double flops;
    for (int rep = 0; rep < 2; rep++) { // rep 0 = warm-up
        cudaEventRecord(e0);
        if (kind == 0) probe_dfma_kernel<<<blocks, threads>>>(out, iters, 1.0);
        else probe_dmma_kernel<<<blocks, threads>>>(out, iters, 1.0);
        cudaEventRecord(e1);
        e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) break;
    }
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    if (kind == 0) flops = 2.0 * 64.0 * iters * (double)blocks * threads;                  // 64 DFMA per thread-iteration
    else flops = 2.0 * 8 * 8 * 4 * 32.0 * iters * (double)blocks * (threads / 32);          // 32 m8n8k4 per warp-iteration
    if (e == cudaSuccess) *tflops = flops / (ms * 1e-3) / 1e12;
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(out);
    if (e == cudaSuccess) e = cudaGetLastError();
    return e;
}

} // namespace sfft
