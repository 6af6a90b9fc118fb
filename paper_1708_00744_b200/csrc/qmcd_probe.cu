// qmcd_probe.cu -- register-resident FP64 throughput probes (roofline
// denominators for the flush; not part of the method).  kind 0: DFMA loop,
// kind 1: DMMA m8n8k4 loop (the FP64 tensor instruction sm_100a has).
#include <cuda_runtime.h>
#include "../../include/qmcd.h"

#define PROBE_THREADS 256
#define PROBE_ILP 8

__global__ void __launch_bounds__(PROBE_THREADS) qmcd_probe_dfma(int iters, double* out) {
    double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-9;
    double acc[PROBE_ILP];
#pragma unroll
    for (int u = 0; u < PROBE_ILP; ++u) acc[u] = u;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < PROBE_ILP; ++u) acc[u] = fma(acc[u], a, b);
    }
    double s = 0;
#pragma unroll
    for (int u = 0; u < PROBE_ILP; ++u) s += acc[u];
    if (s == 123.456) out[0] = s;
}

__global__ void __launch_bounds__(PROBE_THREADS) qmcd_probe_dmma(int iters, double* out) {
    double a = 1e-3 * (threadIdx.x & 7), b = 1e-3;
    double c0[PROBE_ILP], c1[PROBE_ILP];
#pragma unroll
    for (int u = 0; u < PROBE_ILP; ++u) { c0[u] = u; c1[u] = -u; }
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < PROBE_ILP; ++u)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c0[u]), "+d"(c1[u]) : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int u = 0; u < PROBE_ILP; ++u) s += c0[u] + c1[u];
    if (s == 123.456) out[0] = s;
}

extern "C" int qmcd_probe_fp64(int kind, int iters, void* cuda_stream, double* tflops_out) {
    if ((kind != 0 && kind != 1) || iters < 1 || !tflops_out) return QMCD_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return QMCD_ECUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return QMCD_ECUDA;
    const int blocks = sms * 4;          // 4 x 256 threads = 32 warps per SM
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return QMCD_ECUDA;
    double* dummy = nullptr;
    if (cudaMalloc(&dummy, 8) != cudaSuccess) return QMCD_ECUDA;   // probe-only scratch
    float best = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0, st);
        if (kind == 0) qmcd_probe_dfma<<<blocks, PROBE_THREADS, 0, st>>>(iters, dummy);
        else qmcd_probe_dmma<<<blocks, PROBE_THREADS, 0, st>>>(iters, dummy);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(dummy); return QMCD_ECUDA; }
        float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaFree(dummy); cudaEventDestroy(e0); cudaEventDestroy(e1);
    double flops_per_thread_iter = (kind == 0) ? 2.0 * PROBE_ILP : (512.0 / 32.0) * PROBE_ILP;
    double total = flops_per_thread_iter * (double)iters * (double)blocks * PROBE_THREADS;
    *tflops_out = total / (best * 1e-3) / 1e12;
    return QMCD_OK;
}
