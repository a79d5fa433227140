// probe.cu -- FP64 peak probe: register-resident DMMA.8x8x4 / DFMA chains on every SM
// (the FP64 tensor peak is not in MEASURED_PEAKS.json and has to be
// measured on the box; it is the denominator of the Schur update's roofline fraction).
#include "common.cuh"
#include "internal.h"

namespace lsms {

constexpr int PROBE_ACC = 16;    // independent accumulator tiles per warp

__global__ void __launch_bounds__(256) k_probe_dmma(int iters, double* out) {
    double c0[PROBE_ACC], c1[PROBE_ACC];
#pragma unroll
    for (int i = 0; i < PROBE_ACC; ++i) { c0[i] = threadIdx.x * 1e-9; c1[i] = i * 1e-9; }
    double a[PROBE_ACC], b[PROBE_ACC];       // distinct operand registers per accumulator
#pragma unroll
    for (int i = 0; i < PROBE_ACC; ++i) { a[i] = 1.0 + (threadIdx.x + i) * 1e-12; b[i] = 1.0 - (threadIdx.x + 3 * i) * 1e-12; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < PROBE_ACC; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c0[i]), "+d"(c1[i]) : "d"(a[i]), "d"(b[i]));
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < PROBE_ACC; ++i) s += c0[i] + c1[i];
    if (s == 123.456) out[0] = s;
}

__global__ void __launch_bounds__(256) k_probe_dfma(int iters, double* out) {
    double c[PROBE_ACC];
#pragma unroll
    for (int i = 0; i < PROBE_ACC; ++i) c[i] = threadIdx.x * 1e-9 + i;
    double a = 1.0 + threadIdx.x * 1e-12, b = 1e-9;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < PROBE_ACC; ++i) c[i] = fma(c[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < PROBE_ACC; ++i) s += c[i];
    if (s == 123.456) out[0] = s;
}

int run_peak_probe(int which, int iters, double* sink, double* tflops, cudaStream_t st) {
    int dev = 0, sms = 0;
    LSMS_CUDA_OK(cudaGetDevice(&dev));
    LSMS_CUDA_OK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double* dummy = sink;
    cudaEvent_t e0, e1;
    LSMS_CUDA_OK(cudaEventCreate(&e0)); LSMS_CUDA_OK(cudaEventCreate(&e1));
    const int ctas = sms * 2, thr = 256;      // 16 warps per SM: enough to saturate the DMMA pipe
    for (int rep = 0; rep < 2; ++rep) {      // first pass warms up
        LSMS_CUDA_OK(cudaEventRecord(e0, st));
        if (which == 0) k_probe_dmma<<<ctas, thr, 0, st>>>(iters, dummy);
        else k_probe_dfma<<<ctas, thr, 0, st>>>(iters, dummy);
        LSMS_CUDA_OK(cudaEventRecord(e1, st));
        LSMS_CUDA_OK(cudaEventSynchronize(e1));
    }
    float ms = 0.f;
    LSMS_CUDA_OK(cudaEventElapsedTime(&ms, e0, e1));
    double flops;
    if (which == 0) flops = (double)ctas * (thr / 32) * (double)iters * PROBE_ACC * 512.0;   // 8*8*4 FMA = 512 flop per warp MMA
    else flops = (double)ctas * thr * (double)iters * PROBE_ACC * 2.0;
    *tflops = flops / (ms * 1e-3) / 1e12;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    return 0;
}

}  // namespace lsms
