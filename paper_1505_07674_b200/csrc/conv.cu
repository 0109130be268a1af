// conv.cu -- steps a5-a6: direct PSF convolution with replicate padding and, fused into its
// epilogue, the weighted chi-square.
//
//   L*_ij = sum_{k=-p..p} sum_{l=-q..q} F_{-k,-l} L_{clamp(i+k), clamp(j+l)}   PAPER.md:159-164 eq. 15
//   loglike = -1/2 sum_i w_i (d_i - L*_i)^2                                    PAPER.md:178-182 eq. 17
//
// FP32 direct convolution on the FMA pipe (not a GEMM: DESIGN.md "why no tensor cores"),
// written on packed pairs (FFMA2, f32x2.cuh): one issue slot per two multiply-adds.
// blockIdx.y = parameter vector, blockIdx.x = active output tile (tiles with no unmasked
// pixel are not launched).  A block stages its 64 x 128 input tile with the PSF halo in shared
// memory (border pixels repeated, L164) next to the tap pairs, then each thread accumulates
// 4 rows x 8 columns of outputs (two 4-column groups 64 columns apart, so that the 8 lanes
// of a quarter-warp read consecutive 16-byte words: conflict-free LDS.128).
//
// Pairing.  A register pair holds the SAME column of two vertically adjacent output rows
// (o, o+1).  At input row r they need tap rows r-o and r-o-1, so the pair multiplies the
// broadcast scalar in[r][x+k] by the tap pair  Q[j][k] = (G[j][k], G[j-1][k]),  j = r-o,
// G = flipped normalised PSF, G[-1] = G[KH] = 0.  Q is built on the host (api.cu) and sits
// in shared memory; both operands of the FFMA2 come as they are loaded -- no shuffling of
// register halves.  The thread's two row pairs (rows 0-1, 2-3) use Q[r] and Q[r-2].
//
//   loop over tap-column chunks c (4 taps each)
//     loop over input rows r of the thread's strip (KH + 3 of them)
//       4 x LDS.128  input  in[r][4 tx + 4c .. +7]  and  .. + 64        (conflict-free)
//       4 x LDS.128  taps   Q[r][c], Q[r-2][c]                          (broadcast)
//       64 x FFMA2
//
// Zero padding exists only in the tap columns (KW -> multiple of 4) and in the first / last
// tap row of each pair; the staged input is zero beyond the KW-1 halo columns, and the traced
// set is dilated by p+1 rows (api.cu), so a zero tap never meets an untraced value.
// Summation is blocked (per chunk, then across chunks): FP32 error growth ~ sqrt(4 KH) + sqrt(NC).
//
// Epilogue: loglike -> per-thread FP32 sum over its 32 pixels, then FP64: warp shuffle
// tree, the block's warps, and one FP64 partial per (vector, tile), summed in a fixed
// order by final_kernel: bitwise reproducible, no float atomics.
#include "lensed_internal.h"
#include "f32x2.cuh"
#include <math.h>

namespace lensed {
namespace {

constexpr int kTR = 4;                 // output rows per thread (two pairs)
constexpr int kNTX = 16, kNTY = 16;    // threads per block in x / y (warps are 8 x 4 threads)
constexpr int kThreads = kNTX * kNTY;
constexpr int kGroup = 4 * kNTX;       // 64: distance of a thread's two column groups
constexpr int kTW = 2 * kGroup;        // 128 output columns per tile
constexpr int kTH = kTR * kNTY;        // 64 output rows per tile

__device__ __forceinline__ f2 as_f2(unsigned long long v) { f2 r; r.v = v; return r; }

// One input row r of the thread's strip against one 4-tap chunk.  P0 / P1: row pair 0 (tap
// pairs Q[r]) / row pair 1 (Q[r-2]) takes part.  in_r -> in[r][4 tx + 4 c], q0 -> Q[r][c],
// q1 -> Q[r-2][c].
template <bool P0, bool P1>
__device__ __forceinline__ void row_step(f2 (&part)[2][8], const float4 *in_r, const ulonglong2 *q0,
                                         const ulonglong2 *q1)
{
    const float4 a0 = in_r[0], a1 = in_r[1], b0 = in_r[kGroup / 4], b1 = in_r[kGroup / 4 + 1];
    const float va[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
    const float vb[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
    if (P0) {
        const ulonglong2 t0 = q0[0], t1 = q0[1];
        const f2 q[4] = {as_f2(t0.x), as_f2(t0.y), as_f2(t1.x), as_f2(t1.y)};
#pragma unroll
        for (int k = 0; k < 4; ++k)
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                part[0][e] = fma2(q[k], bc(va[e + k]), part[0][e]);
                part[0][4 + e] = fma2(q[k], bc(vb[e + k]), part[0][4 + e]);
            }
    }
    if (P1) {
        const ulonglong2 t0 = q1[0], t1 = q1[1];
        const f2 q[4] = {as_f2(t0.x), as_f2(t0.y), as_f2(t1.x), as_f2(t1.y)};
#pragma unroll
        for (int k = 0; k < 4; ++k)
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                part[1][e] = fma2(q[k], bc(va[e + k]), part[1][e]);
                part[1][4 + e] = fma2(q[k], bc(vb[e + k]), part[1][4 + e]);
            }
    }
}

template <bool RENDER>
__global__ void __launch_bounds__(kThreads, 2) conv_kernel(ConvArgs a)
{
    extern __shared__ float4 smem4[];
    const int IW4 = kTW / 4 + a.NC, IW = 4 * IW4;
    const int IH = kTH + a.KH - 1;
    float *s_in = reinterpret_cast<float *>(smem4);                                    // [IH][IW]
    ulonglong2 *s_q = reinterpret_cast<ulonglong2 *>(smem4 + (size_t)IH * IW4);        // [KH+1][NC][2]
    __shared__ double s_red[kThreads / 32];

    const int bvec = blockIdx.y;
    const uint32_t tile = a.tiles[blockIdx.x];
    const int Y0 = (int)(tile >> 16) * kTH, X0 = (int)(tile & 0xffffu) * kTW;
    const float *Lb = a.L + (size_t)bvec * a.l_stride;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    // stage the tap pairs and the clamped input tile (zero beyond the KW-1 halo columns)
    {
        const ulonglong2 *gq = reinterpret_cast<const ulonglong2 *>(a.taps);
        for (int i = threadIdx.x; i < (a.KH + 1) * a.NC * 2; i += kThreads) s_q[i] = gq[i];
        const int used = kTW + a.KW - 1;
        for (int r = warp; r < IH; r += kThreads / 32) {
            const int y = min(max(Y0 - a.p + r, 0), a.H - 1);
            const float *src = Lb + (size_t)y * a.W;
            for (int c = lane; c < IW; c += 32) {
                const int x = min(max(X0 - a.q + c, 0), a.W - 1);
                s_in[r * IW + c] = c < used ? src[x] : 0.0f;
            }
        }
    }
    __syncthreads();

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
            for (int e = 0; e < 8; ++e) {
                const int y = oy + o, x = ox + (e & 3) + (e >> 2) * kGroup;
                if (y < a.H && x < a.W) any = any || a.wmask[(size_t)y * a.W + x] != 0.0f;
            }
    }
    const bool warp_any = __any_sync(0xffffffffu, any);

    // acc[pair][column]: running sum over tap-column chunks; part: the current chunk
    f2 acc[2][8];
#pragma unroll
    for (int p = 0; p < 2; ++p)
#pragma unroll
        for (int e = 0; e < 8; ++e) acc[p][e] = bc(0.0f);

    if (warp_any) {
        const int KH = a.KH, NC2 = 2 * a.NC;
        const float4 *in_base = reinterpret_cast<const float4 *>(s_in) + (size_t)(ty * kTR) * IW4 + tx;
#pragma unroll 1
        for (int c = 0; c < a.NC; ++c) {
            f2 part[2][8];
#pragma unroll
            for (int p = 0; p < 2; ++p)
#pragma unroll
                for (int e = 0; e < 8; ++e) part[p][e] = bc(0.0f);
            const float4 *in_r = in_base + c;
            const ulonglong2 *q_r = s_q + 2 * c;
            row_step<true, false>(part, in_r, q_r, nullptr);
            row_step<true, false>(part, in_r + IW4, q_r + NC2, nullptr);
            in_r += 2 * IW4;
#pragma unroll 2
            for (int r = 2; r <= KH; ++r) {
                row_step<true, true>(part, in_r, q_r + 2 * NC2, q_r);
                in_r += IW4;
                q_r += NC2;
            }
            row_step<false, true>(part, in_r, nullptr, q_r);
            row_step<false, true>(part, in_r + IW4, nullptr, q_r + NC2);
#pragma unroll
            for (int p = 0; p < 2; ++p)
#pragma unroll
                for (int e = 0; e < 8; ++e) acc[p][e] = add2(acc[p][e], part[p][e]);
        }
    }

    float out[kTR][8];
#pragma unroll
    for (int p = 0; p < 2; ++p)
#pragma unroll
        for (int e = 0; e < 8; ++e) un2(acc[p][e], out[2 * p][e], out[2 * p + 1][e]);

    if (RENDER) {
        const bool valid = a.derived[(size_t)bvec * a.D] != 0.0f;
        float *mb = a.model + (size_t)bvec * a.l_stride;
#pragma unroll
        for (int o = 0; o < kTR; ++o)
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const int y = oy + o, x = ox + (e & 3) + (e >> 2) * kGroup;
                if (y < a.H && x < a.W) mb[(size_t)y * a.W + x] = valid ? out[o][e] : nanf("");
            }
    } else {
        float part = 0.0f;
        if (warp_any) {
#pragma unroll
            for (int o = 0; o < kTR; ++o)
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int y = oy + o, x = ox + (e & 3) + (e >> 2) * kGroup;
                    if (y < a.H && x < a.W) {
                        const size_t i = (size_t)y * a.W + x;
                        const float w = a.wmask[i];
                        if (w != 0.0f) {                   // masked pixels may see untraced L: never touch them
                            const float diff = a.image[i] - out[o][e];
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
    return (IH * IW + (size_t)(KH + 1) * 8 * NC) * sizeof(float);
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
