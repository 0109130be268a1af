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

// ---- issue-slot probe ----------------------------------------------------------------------
// What does an instruction of another kind cost in FP32-pipe time when it sits between packed
// FFMA2?  One loop body = 64 FFMA2 on 16 independent accumulator pairs (128 cycles at the pipe's
// full rate) with n_extra instructions of KIND spread evenly among them; one block per SM with
// `warps` warps per scheduler; returns clock64 cycles per body of one warp's timeline.
//   KIND 0 none, 1 LOP3 (ALU pipe), 2 MUFU.EX2 (XU pipe), 3 scalar FFMA, 4 IMAD
// Read-outs used in DESIGN.md / profiles/r2b.md: an ALU- or XU-pipe instruction costs about a
// third of a cycle, a scalar FP32 instruction 1.3-1.5, an integer multiply-add 2.
typedef unsigned long long u64;
__device__ __forceinline__ u64 probe_fma2(u64 a, u64 b, u64 c)
{
    u64 r;
    asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}

template <int KIND, int NX>
__global__ void issue_probe_kernel(float *out, int iters, long long *cyc)
{
    u64 acc[16];
    for (int i = 0; i < 16; ++i) acc[i] = (u64)threadIdx.x + i;
    const u64 a = 0x3f8000003f800000ull + (u64)(threadIdx.x & 1), b = 0x3a8000003a800000ull + (u64)(iters & 1);
    unsigned x[8];
    float f[8];
    for (int i = 0; i < 8; ++i) { x[i] = threadIdx.x + i; f[i] = 0.001f * (threadIdx.x + i); }
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 64; ++r) {
            acc[r & 15] = probe_fma2(a, b, acc[r & 15]);
            constexpr int every = NX > 0 ? 64 / NX : 64;
            if (KIND != 0 && r % every == 0 && r / every < NX) {
                const int j = r & 7;
                if (KIND == 1) asm volatile("xor.b32 %0, %0, %1;" : "+r"(x[j]) : "r"(x[(j + 1) & 7]));
                if (KIND == 2) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(f[j]));
                if (KIND == 3) asm volatile("fma.rn.f32 %0, %0, %1, %1;" : "+f"(f[j]) : "f"(f[(j + 1) & 7]));
                if (KIND == 4) asm volatile("mad.lo.u32 %0, %0, %1, %1;" : "+r"(x[j]) : "r"(x[(j + 1) & 7]));
            }
        }
    }
    const long long t1 = clock64();
    float s = 0.0f;
    for (int i = 0; i < 16; ++i) s += (float)(acc[i] & 0xff);
    for (int i = 0; i < 8; ++i) s += x[i] + f[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0 && blockIdx.x == 0) *cyc = t1 - t0;
}

template <int KIND>
cudaError_t probe_nx(int n_extra, int grid, int threads, float *out, int iters, long long *cyc)
{
    switch (n_extra) {
    case 0: issue_probe_kernel<0, 0><<<grid, threads>>>(out, iters, cyc); break;
    case 8: issue_probe_kernel<KIND, 8><<<grid, threads>>>(out, iters, cyc); break;
    case 16: issue_probe_kernel<KIND, 16><<<grid, threads>>>(out, iters, cyc); break;
    case 32: issue_probe_kernel<KIND, 32><<<grid, threads>>>(out, iters, cyc); break;
    case 64: issue_probe_kernel<KIND, 64><<<grid, threads>>>(out, iters, cyc); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

}  // namespace

// n_extra in {0, 8, 16, 32, 64}; warps in {1, 2, 4} per scheduler
cudaError_t run_issue_probe(int kind, int n_extra, int warps, double *cycles_per_body)
{
    if (kind < 0 || kind > 4 || (warps != 1 && warps != 2 && warps != 4)) return cudaErrorInvalidValue;
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    const int threads = 128 * warps, iters = 2000;
    float *out = nullptr;
    long long *cyc = nullptr, h = 0;
    if ((e = cudaMalloc(&out, (size_t)sms * threads * sizeof(float))) != cudaSuccess) return e;
    if ((e = cudaMalloc(&cyc, sizeof(long long))) != cudaSuccess) { cudaFree(out); return e; }
    for (int rep = 0; rep < 2 && e == cudaSuccess; ++rep) {
        switch (kind) {
        case 0: e = probe_nx<0>(0, sms, threads, out, iters, cyc); break;
        case 1: e = probe_nx<1>(n_extra, sms, threads, out, iters, cyc); break;
        case 2: e = probe_nx<2>(n_extra, sms, threads, out, iters, cyc); break;
        case 3: e = probe_nx<3>(n_extra, sms, threads, out, iters, cyc); break;
        default: e = probe_nx<4>(n_extra, sms, threads, out, iters, cyc); break;
        }
    }
    if (e == cudaSuccess) e = cudaMemcpy(&h, cyc, sizeof h, cudaMemcpyDeviceToHost);
    cudaFree(out); cudaFree(cyc);
    *cycles_per_body = (double)h / iters / warps;
    return e;
}

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
