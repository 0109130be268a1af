// conv.cu -- steps a5-a6: direct PSF convolution with replicate padding and, fused into its
// epilogue, the weighted chi-square.
//
//   L*_ij = sum_{k=-p..p} sum_{l=-q..q} F_{-k,-l} L_{clamp(i+k), clamp(j+l)}   PAPER.md:159-164 eq. 15
//   loglike = -1/2 sum_i w_i (d_i - L*_i)^2                                    PAPER.md:178-182 eq. 17
//
// FP32 direct convolution on the FMA pipe (not a GEMM: DESIGN.md "why no tensor cores").
// blockIdx.y = parameter vector, blockIdx.x = active output tile (tiles with no unmasked
// pixel are not launched).  A block stages its input tile with the PSF halo in shared
// memory (border pixels repeated, L164) next to the pre-flipped, normalised taps, then each
// thread accumulates a kTR x 4 register tile of outputs:
//
//   loop over tap-column chunks c (4 taps each)
//     loop over input rows r of the thread's strip (kTR + KH - 1 of them)
//       2 x LDS.128  input  in[r][4 tx + 4c .. + 7]          (conflict-free: 8 lanes = 128 B)
//       1 x LDS.128  taps   G[r][4c .. 4c+3]                 (broadcast)
//       kTR x 16 FFMA: output row o uses tap row ky = r - o
//
// The tap row used by output row o at input row r is the one row o+1 uses at r+1, so the
// tap vectors live in kTR register slots indexed by (ky mod kTR) and the row loop is
// unrolled by kTR ("super-step") to make every slot index static.  Super-steps whose tap
// rows are all inside the PSF run branch-free; the first and last ones test each (row, o)
// pair with block-uniform branches, so no multiply by a padded zero is ever issued in y.
//
// Epilogue: loglike -> per-thread FP32 sum over its 4 kTR pixels, then FP64: warp shuffle
// tree, the block's warps, and one FP64 partial per (vector, tile), summed in a fixed
// order by final_kernel: bitwise reproducible, no float atomics.
#include "lensed_internal.h"
#include <math.h>

namespace lensed {
namespace {

constexpr int kTR = 4;                 // output rows per thread
constexpr int kNTX = 16, kNTY = 16;    // threads per block in x / y (warps are 8 x 4 threads)
constexpr int kThreads = kNTX * kNTY;
constexpr int kTW = 4 * kNTX;          // 64 output columns per tile
constexpr int kTH = kTR * kNTY;        // 64 output rows per tile

__device__ __forceinline__ void fma16(float (&acc)[4], const float4 &t, const float4 &v0, const float4 &v1)
{
    const float v[8] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w};
    const float tp[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
    for (int k = 0; k < 4; ++k)
#pragma unroll
        for (int e = 0; e < 4; ++e) acc[e] = fmaf(tp[k], v[e + k], acc[e]);
}

// One super-step: input rows r = g kTR + s, s = 0..kTR-1.  EDGE = test the tap rows.
template <bool EDGE>
__device__ __forceinline__ void super_step(float (&acc)[kTR][4], float4 (&T)[kTR], const float4 *in_row,
                                           const float4 *tap_c, int g, int KH, int NC, int IW4)
{
#pragma unroll
    for (int s = 0; s < kTR; ++s) {
        const int r = g * kTR + s;
        if (EDGE && r >= KH + kTR - 1) break;
        const float4 v0 = in_row[(size_t)r * IW4], v1 = in_row[(size_t)r * IW4 + 1];
        if (!EDGE || r < KH) T[s] = tap_c[r * NC];
#pragma unroll
        for (int o = 0; o < kTR; ++o) {
            const int ky = r - o;
            if (!EDGE || (ky >= 0 && ky < KH)) fma16(acc[o], T[(s - o + kTR) % kTR], v0, v1);
        }
    }
}

template <bool RENDER>
__global__ void __launch_bounds__(kThreads, 2) conv_kernel(ConvArgs a)
{
    extern __shared__ float4 smem4[];
    const int IW = kTW + 4 * a.NC, IW4 = IW / 4;
    const int IH = kTH + a.KH - 1;
    float *s_in = reinterpret_cast<float *>(smem4);                 // [IH][IW]
    float4 *s_tap = smem4 + (size_t)IH * IW4;                       // [KH][NC]
    __shared__ double s_red[kThreads / 32];

    const int bvec = blockIdx.y;
    const uint32_t tile = a.tiles[blockIdx.x];
    const int Y0 = (int)(tile >> 16) * kTH, X0 = (int)(tile & 0xffffu) * kTW;
    const float *Lb = a.L + (size_t)bvec * a.l_stride;

    // stage taps and the clamped input tile
    {
        const float4 *gt = reinterpret_cast<const float4 *>(a.taps);
        for (int i = threadIdx.x; i < a.KH * a.NC; i += kThreads) s_tap[i] = gt[i];
        const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
        for (int r = warp; r < IH; r += kThreads / 32) {
            const int y = min(max(Y0 - a.p + r, 0), a.H - 1);
            const float *src = Lb + (size_t)y * a.W;
            for (int c = lane; c < IW; c += 32) {
                const int x = min(max(X0 - a.q + c, 0), a.W - 1);
                s_in[r * IW + c] = src[x];
            }
        }
    }
    __syncthreads();

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int tx = (warp & 1) * 8 + (lane & 7);
    const int ty = (warp >> 1) * 4 + (lane >> 3);
    const int oy = Y0 + ty * kTR, ox = X0 + tx * 4;

    // does this warp own any pixel that counts?  (uniform per warp: skipping is free)
    bool any = false;
    if (RENDER) {
        any = oy < a.H && ox < a.W;
    } else {
#pragma unroll
        for (int o = 0; o < kTR; ++o)
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int y = oy + o, x = ox + e;
                if (y < a.H && x < a.W) any = any || a.wmask[(size_t)y * a.W + x] != 0.0f;
            }
    }
    const bool warp_any = __any_sync(0xffffffffu, any);

    // acc: running sum over tap-column chunks; part: the current chunk (blocked summation:
    // a chunk adds 4 KH products, the running sum adds NC chunk totals)
    float acc[kTR][4];
#pragma unroll
    for (int o = 0; o < kTR; ++o)
#pragma unroll
        for (int e = 0; e < 4; ++e) acc[o][e] = 0.0f;

    if (warp_any) {
        const int S = a.KH + kTR - 1;              // input rows per thread strip
        const int G = (S + kTR - 1) / kTR;         // super-steps
        const int g_hi = a.KH / kTR - 1;           // steady super-steps are 1 .. g_hi
        const float4 *in_base = reinterpret_cast<const float4 *>(s_in) + (size_t)(ty * kTR) * IW4 + tx;
#pragma unroll 1
        for (int c = 0; c < a.NC; ++c) {
            float part[kTR][4];
            float4 T[kTR];
#pragma unroll
            for (int s = 0; s < kTR; ++s) {
                T[s] = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                for (int e = 0; e < 4; ++e) part[s][e] = 0.0f;
            }
            const float4 *in_c = in_base + c;
            const float4 *tap_c = s_tap + c;
            super_step<true>(part, T, in_c, tap_c, 0, a.KH, a.NC, IW4);
            int g = 1;
#pragma unroll 1
            for (; g <= g_hi; ++g) super_step<false>(part, T, in_c, tap_c, g, a.KH, a.NC, IW4);
#pragma unroll 1
            for (; g < G; ++g) super_step<true>(part, T, in_c, tap_c, g, a.KH, a.NC, IW4);
#pragma unroll
            for (int o = 0; o < kTR; ++o)
#pragma unroll
                for (int e = 0; e < 4; ++e) acc[o][e] += part[o][e];
        }
    }

    if (RENDER) {
        const bool valid = a.derived[(size_t)bvec * a.D] != 0.0f;
        float *mb = a.model + (size_t)bvec * a.l_stride;
#pragma unroll
        for (int o = 0; o < kTR; ++o)
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int y = oy + o, x = ox + e;
                if (y < a.H && x < a.W) mb[(size_t)y * a.W + x] = valid ? acc[o][e] : nanf("");
            }
    } else {
        float part = 0.0f;
        if (warp_any) {
#pragma unroll
            for (int o = 0; o < kTR; ++o)
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int y = oy + o, x = ox + e;
                    if (y < a.H && x < a.W) {
                        const size_t i = (size_t)y * a.W + x;
                        const float w = a.wmask[i];
                        if (w != 0.0f) {                   // masked pixels may see untraced L: never touch them
                            const float diff = a.image[i] - acc[o][e];
                            part = fmaf(w * diff, diff, part);
                        }
                    }
                }
        }
        double dpart = (double)part;
#pragma unroll
        for (int sft = 16; sft > 0; sft >>= 1) dpart += __shfl_xor_sync(0xffffffffu, dpart, sft);
        if (lane == 0) s_red[warp] = dpart;
        __syncthreads();
        if (threadIdx.x == 0) {
            double s = 0.0;
#pragma unroll
            for (int i = 0; i < kThreads / 32; ++i) s += s_red[i];
            a.partial[(size_t)bvec * a.n_tiles + blockIdx.x] = s;
        }
    }
}

__global__ void __launch_bounds__(128) final_kernel(FinalArgs a)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= a.B) return;
    double s = 0.0;
    const double *p = a.partial + (size_t)b * a.n_tiles;
    for (int t = 0; t < a.n_tiles; ++t) s += p[t];
    const bool valid = a.derived[(size_t)b * a.D] != 0.0f;
    a.logl[b] = valid ? (float)(-0.5 * s) : -INFINITY;
}

}  // namespace

void conv_tile_shape(int *tile_w, int *tile_h) { *tile_w = kTW; *tile_h = kTH; }

size_t conv_smem_bytes(int KH, int NC)
{
    const size_t IW = kTW + 4 * NC, IH = kTH + KH - 1;
    return (IH * IW + (size_t)KH * 4 * NC) * sizeof(float);
}

cudaError_t conv_setup()
{
    const int max_smem = (int)conv_smem_bytes(kMaxPsf, (kMaxPsf + 3) / 4);
    cudaError_t e = cudaFuncSetAttribute(conv_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(conv_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
}

cudaError_t launch_conv(const ConvArgs &a, bool render, int nvec, cudaStream_t st)
{
    const size_t smem = conv_smem_bytes(a.KH, a.NC);
    dim3 grid(a.n_tiles, nvec);
    if (render) conv_kernel<true><<<grid, kThreads, smem, st>>>(a);
    else conv_kernel<false><<<grid, kThreads, smem, st>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_final(const FinalArgs &a, cudaStream_t st)
{
    final_kernel<<<(a.B + 127) / 128, 128, 0, st>>>(a);
    return cudaGetLastError();
}

}  // namespace lensed
