/*
 * ia_peak.cu -- K4: FP64 FMA peak microbenchmark, the denominator of the roofline
 * (BASELINE.json metric "% of FP64 FMA peak"; MEASURED_PEAKS.json carries no FP64 figure).
 * Every thread runs 8 independent DFMA chains; the grid fills every SM with 1024 threads.
 */
#include "ia_kernels.cuh"

#define PEAK_CHAINS 8
#define PEAK_INNER 64

__global__ void __launch_bounds__(256) ia_dfma_peak_kernel(double *sink, unsigned iters, double a, double b) {
    double acc[PEAK_CHAINS];
#pragma unroll
    for (int k = 0; k < PEAK_CHAINS; ++k) acc[k] = (double)(threadIdx.x + k) * 1e-3;
    for (unsigned it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < PEAK_INNER; ++u) {
#pragma unroll
            for (int k = 0; k < PEAK_CHAINS; ++k) acc[k] = fma(acc[k], a, b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < PEAK_CHAINS; ++k) s += acc[k];
    if (s == 123.456) sink[0] = s; /* never true for the a, b used; keeps the chains alive */
}

cudaError_t ia_run_fp64_peak(int device, double target_ms, double *tflops, double *elapsed_ms) {
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return e;
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, device);
    if (e != cudaSuccess) return e;
    double *sink = nullptr;
    e = cudaMalloc(&sink, sizeof(double));
    if (e != cudaSuccess) return e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int blocks = prop.multiProcessorCount * 4, threads = 256;
    auto run = [&](unsigned iters, float *ms) -> cudaError_t {
        cudaEventRecord(e0, 0);
        ia_dfma_peak_kernel<<<blocks, threads>>>(sink, iters, 0.999999, 1e-7);
        cudaEventRecord(e1, 0);
        cudaError_t err = cudaEventSynchronize(e1);
        if (err != cudaSuccess) return err;
        return cudaEventElapsedTime(ms, e0, e1);
    };
    float ms = 0.f;
    unsigned iters = 2000;
    e = run(iters, &ms); /* warm-up + calibration */
    if (e == cudaSuccess) e = run(iters, &ms);
    if (e == cudaSuccess) {
        if (target_ms < 1.0) target_ms = 1.0;
        if (target_ms > 5000.0) target_ms = 5000.0;
        double scale = target_ms / (ms > 1e-3 ? ms : 1e-3);
        if (scale > 1000.0) scale = 1000.0;
        iters = (unsigned)(iters * scale) + 1;
        e = run(iters, &ms);
    }
    if (e == cudaSuccess) {
        const double fmas = (double)blocks * threads * (double)iters * PEAK_INNER * PEAK_CHAINS;
        *tflops = 2.0 * fmas / (ms * 1e-3) / 1e12;
        *elapsed_ms = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    return e;
}

/* Latency of DEPENDENT FP64 operations, in SM cycles: one warp, one chain.  What bounds the step of a lone warp
 * (the end of a stream) is the length of the step's dependent chain times this. */
__global__ void ia_fp64_latency_kernel(double *out, unsigned n, double a, double b) {
    double x = 0.5 + 1e-3 * (double)threadIdx.x;
    long long t0 = clock64();
#pragma unroll 1
    for (unsigned it = 0; it < n; ++it) {
#pragma unroll
        for (int u = 0; u < 64; ++u) x = fma(x, a, b);
    }
    long long t1 = clock64();
    double y = 1.5 + 1e-3 * (double)threadIdx.x;
#pragma unroll 1
    for (unsigned it = 0; it < n; ++it) {
#pragma unroll
        for (int u = 0; u < 16; ++u) y = ia_rcp(y) + a; /* MUFU.RCP64H + 3 DFMA, then one DADD */
    }
    long long t2 = clock64();
    if (threadIdx.x == 0) {
        out[0] = (double)(t1 - t0) / (64.0 * n);
        out[1] = (double)(t2 - t1) / (16.0 * n);
        out[2] = x + y;
    }
}

cudaError_t ia_run_fp64_latency(int device, double *cycles_dfma, double *cycles_rcp_add) {
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return e;
    double *out = nullptr;
    e = cudaMalloc(&out, 3 * sizeof(double));
    if (e != cudaSuccess) return e;
    double h[3] = {0, 0, 0};
    for (int rep = 0; rep < 2 && e == cudaSuccess; ++rep) { /* the second launch is the measurement */
        ia_fp64_latency_kernel<<<1, 32>>>(out, 2000u, 0.999999, 1e-7);
        e = cudaMemcpy(h, out, sizeof(h), cudaMemcpyDeviceToHost);
    }
    cudaFree(out);
    if (e == cudaSuccess) {
        *cycles_dfma = h[0];
        *cycles_rcp_add = h[1];
    }
    return e;
}
