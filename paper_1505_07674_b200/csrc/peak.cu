// peak.cu -- FP32 FFMA micro-benchmark: the measured denominator of the ALU roofline.
// MEASURED_PEAKS.json holds HBM and bf16 tensor peaks only; the path here is bound by the
// plain FP32 pipe, so bench.py reports its fraction of both the nominal figure
// (148 SM x 128 lanes x 2 flop x SM clock) and of what this kernel sustains.
#include "lensed_internal.h"

namespace lensed {
namespace {

constexpr int kChains = 16;

__global__ void __launch_bounds__(256) fma_peak_kernel(float *out, int iters, float a, float b)
{
    float x[kChains];
#pragma unroll
    for (int c = 0; c < kChains; ++c) x[c] = (float)(threadIdx.x + c) * 1e-3f;
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u)
#pragma unroll
            for (int c = 0; c < kChains; ++c) x[c] = fmaf(x[c], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < kChains; ++c) s += x[c];
    if (s == 123.456f) out[0] = s;    // keeps the chains live; never true in practice
}

}  // namespace

cudaError_t run_fma_peak(int iters, double *tflops)
{
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    float *d = nullptr;
    e = cudaMalloc(&d, sizeof(float));
    if (e != cudaSuccess) return e;
    cudaEvent_t a, b;
    cudaEventCreate(&a); cudaEventCreate(&b);
    const int blocks = sms * 8, threads = 256;
    fma_peak_kernel<<<blocks, threads>>>(d, iters / 4 + 1, 0.999f, 1e-3f);   // warm-up
    double best = 0.0;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(a);
        fma_peak_kernel<<<blocks, threads>>>(d, iters, 0.999f, 1e-3f);
        cudaEventRecord(b);
        e = cudaEventSynchronize(b);
        if (e != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, a, b);
        const double flops = 2.0 * (double)blocks * threads * kChains * 8.0 * iters;
        best = fmax(best, flops / (ms * 1e-3) * 1e-12);
    }
    cudaEventDestroy(a); cudaEventDestroy(b);
    cudaFree(d);
    if (e == cudaSuccess) e = cudaGetLastError();
    *tflops = best;
    return e;
}

}  // namespace lensed
