// conv.cu -- steps a5-a6: PSF convolution with replicated borders, fused with the weighted
// chi-square reduction (loglike) or with the store of the model image (render).
//
//   L*_ij = sum_{k=-p..p} sum_{l=-q..q} F_{-k,-l} L_{clamp(i+k), clamp(j+l)}   PAPER.md:159-164 eq. 15
//   loglike = -1/2 sum_i w_i (d_i - L*_i)^2                                    PAPER.md:178-182 eq. 17
//
// FP32 direct convolution on the FMA pipe (not a GEMM: DESIGN.md "why no tensor cores"),
// written on packed pairs (FFMA2, f32x2.cuh): one issue slot per two multiply-adds.
//
// Input.  The tracer writes the unconvolved images into a PADDED buffer: pixel (i, j) sits at
// (i + p, j + q) of a [Hp][Wp] frame and border pixels are replicated into the pad (L164), so
// a tile with its PSF halo is a plain rectangle of that frame -- no clamping here.
// The frame spans the image and every tile in use (+ KH - 1 rows, + 4 NC columns, NC =
// ceil(KW / 4)): tiles that overhang the image read zeros / stale finite values whose outputs
// are dropped.  The loglike tile grid starts at the corner of the counted pixels' bounding
// box (a.ox, a.oy), the render grid at (0, 0).
//
// Work.  Persistent blocks: one of 256 threads per SM ("wide", 64 x 128 output tiles) or two of
// 128 threads ("narrow", 64 x 64 tiles; see Shape below).  A work item is (output tile,
// parameter vector); items are ordered tile-major and split evenly over the blocks, so a block
// stays on one tile position for many vectors: the tile's data d and weights w are staged in
// shared memory once per position.  The input tile with its halo (64 + KH - 1 rows of
// tile width + 4 NC floats) is a plain box of the padded frame: ONE thread moves it with one TMA
// tensor copy (cp.async.bulk.tensor.3d over (x, y, vector), completion on an mbarrier), double
// buffered: item i+1 loads while item i is convolved (single buffer when two do not fit: PSFs
// beyond ~45 x 45).  Against 256 threads x cp.async 16 B with an integer divide per element
// (LENSED_CONV_TMA=0) the tensor copy is worth 0.7 % at 31 x 31 and 3-11 % at 9 x 9 ... 21 x 21
// (profiles/r2b.md).
//
// Thread tile: 4 rows x 8 columns of outputs (two 4-column groups 64 columns apart, so that
// the 8 lanes of a quarter-warp read consecutive 16-byte words: conflict-free LDS.128).
//
// Pairing.  A register pair holds the SAME column of two vertically adjacent output rows
// (o, o+1).  At input row r they need tap rows r-o and r-o-1, so the pair multiplies the
// broadcast scalar in[r][x+k] by the tap pair  Q[j][k] = (G[j][k], G[j-1][k]),  j = r-o,
// G = flipped normalised PSF, G[-1] = G[KH] = 0.  Q is built on the host (api.cu).  At step
// j = 0..KH the thread's two row pairs (rows 0-1, 2-3) both use Q[j]: pair 0 against input
// row j of the thread's strip, pair 1 against row j + 2.  Four staged rows live in registers
// and change roles every two steps, so each staged row is loaded once per chunk.
//
// Taps.  Q is block-uniform, so it is read through the UNIFORM datapath: it lives in the
// constant bank (c_taps, a pool shared by the live handles) and FFMA2 takes the pair straight
// from a uniform register (FFMA2 R, R.F32, UR.F32x2, R): no shared-memory traffic, no vector
// registers for taps.
//
//   loop over tap-column chunks c (4 taps each)
//     loop over steps j = 0 .. KH
//       4 x LDS.128   input  in[j + 4][4 tx + 4c .. +7]  and  .. + 64    (conflict-free)
//       4 x LDCU.64   taps   Q[j][c][0..3]                               (uniform datapath)
//       64 x FFMA2
//
// Zero padding exists only in the tap columns (KW -> multiple of 4) and in the first / last
// tap row of each pair; the traced set is dilated by p+1 rows (api.cu), the padded frame is
// zero-initialised and the tracers clamp what they store to the finite range (store_pixel), so
// a zero tap never meets a non-finite value.
// Summation is blocked (per chunk, then across chunks): FP32 error growth ~ sqrt(4 KH) + sqrt(NC).
//
// Epilogue: loglike -> per-thread FP32 sum over its 32 pixels, then FP64: warp shuffle
// tree, the block's warps, and one FP64 partial per (vector, tile), summed in a fixed
// order by final_kernel: bitwise reproducible, no float atomics.
#include "lensed_internal.h"
#include "f32x2.cuh"
#include <math.h>
#include <cuda.h>                 // CUtensorMap (types only; the encoder is fetched from the driver at run time)
#include <cudaTypedefs.h>
#include <algorithm>
#include <stdlib.h>

#ifndef LENSED_CONV_TMA
#define LENSED_CONV_TMA 1         // input tiles by one cp.async.bulk.tensor per tile (0: cp.async per 16 bytes)
#endif

namespace lensed {

// tap pairs of all live handles (api.cu allocates ranges); 60 KB of the 64 KB constant bank
__constant__ unsigned long long c_taps[kTapPoolPairs];

namespace {

constexpr int kTR = 4;                 // output rows per thread (two pairs)
constexpr int kNTY = 16;               // threads per block in y (warps are 8 x 4 threads)
constexpr int kTH = kTR * kNTY;        // 64 output rows per tile
constexpr int kSlackRows = 2;          // rows past a staged tile the last loop body loads but never uses

// Two block shapes (api.cu picks one per handle, ConvArgs::wide):
//   wide   NTX = 16: 256 threads, 64 x 128 tile, one block per SM   -- large images, large PSFs
//   narrow NTX =  8: 128 threads, 64 x 64 tile, two blocks per SM   -- small or masked images and
//          small PSFs, where a tile's prologue (staging, barriers) and epilogue (reduction) are
//          not small against its inner loop: the second block's inner loop hides them, and the
//          64-column tiles waste less of a masked or small image.
template <int NTX>
struct Shape {
    static constexpr int kThreads = NTX * kNTY;
    static constexpr int kGroup = 4 * NTX;      // distance of a thread's two column groups
    static constexpr int kTW = 2 * kGroup;      // output columns per tile
};

__device__ __forceinline__ f2 as_f2(unsigned long long v) { f2 r; r.v = v; return r; }

#if !LENSED_CONV_TMA
__device__ __forceinline__ void cp_async16(void *smem, const void *gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
#endif

// ---- TMA: one elected thread moves the whole (64 + KH - 1) x (tile width + 4 NC) box of the padded
// frame with a single 3-D tensor copy (x, y, vector) that completes on an mbarrier.
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    const unsigned b = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile(
        "{\n.reg .pred p;\nWAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\nbra WAIT_%=;\nDONE_%=:\n}" ::"r"(b), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void *smem, const CUtensorMap *map, unsigned long long *bar, int x, int y, int z)
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // earlier generic reads of this stage are done
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
                 ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(map), "r"((unsigned)__cvta_generic_to_shared(bar)),
                   "r"(x), "r"(y), "r"(z) : "memory");
}

// The 16 input floats a thread needs from one staged row for one 4-tap chunk: columns
// 4 tx + 4 c .. + 7 of both column groups.
struct InRow { float4 a0, a1, b0, b1; };

template <int NTX>
__device__ __forceinline__ void load_row(InRow &x, const float4 *p)
{
    x.a0 = p[0]; x.a1 = p[1]; x.b0 = p[NTX]; x.b1 = p[NTX + 1];
}

// One step j of a 4-tap chunk: both row pairs against the SAME tap pairs Q[j][c][0..3]
// (iq = their index in c_taps).  Pair 0 (output rows 0-1) takes input row j of the strip
// (x0), pair 1 (rows 2-3) takes input row j + 2 (x1).  NT = taps of the chunk (4, or the
// 1-3 of the last chunk when KW is not a multiple of 4: no multiply by a padded zero column).
// GT: the tap pairs come from global memory (gt) instead of the constant pool: the fallback
// for handles that found the pool full (api.cu); same values, LDG through L1 instead of LDCU.
template <int NT, bool GT>
__device__ __forceinline__ void tap_step(f2 (&part)[2][8], const InRow &x0, const InRow &x1, int iq,
                                         const unsigned long long *gt)
{
    const float va0[8] = {x0.a0.x, x0.a0.y, x0.a0.z, x0.a0.w, x0.a1.x, x0.a1.y, x0.a1.z, x0.a1.w};
    const float vb0[8] = {x0.b0.x, x0.b0.y, x0.b0.z, x0.b0.w, x0.b1.x, x0.b1.y, x0.b1.z, x0.b1.w};
    const float va1[8] = {x1.a0.x, x1.a0.y, x1.a0.z, x1.a0.w, x1.a1.x, x1.a1.y, x1.a1.z, x1.a1.w};
    const float vb1[8] = {x1.b0.x, x1.b0.y, x1.b0.z, x1.b0.w, x1.b1.x, x1.b1.y, x1.b1.z, x1.b1.w};
#pragma unroll
    for (int k = 0; k < NT; ++k) {
        const f2 q = as_f2(GT ? __ldg(gt + iq + k) : c_taps[iq + k]);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            part[0][e] = fma2(q, bc(va0[e + k]), part[0][e]);
            part[0][4 + e] = fma2(q, bc(vb0[e + k]), part[0][4 + e]);
            part[1][e] = fma2(q, bc(va1[e + k]), part[1][e]);
            part[1][4 + e] = fma2(q, bc(vb1[e + k]), part[1][4 + e]);
        }
    }
}

// One 4-tap chunk: steps j = 0 .. KH (tap pair rows Q[j], first pair at c_taps[iq]) into
// `part`, then `acc += part`.  Four staged rows live in registers and change roles every two
// steps without moves: the loop body is four steps.  in_r -> in[strip row 0][4 tx + 4 c].
template <int NT, int NTX, bool GT>
__device__ __forceinline__ void conv_chunk(f2 (&acc)[2][8], const float4 *in_r, int iq, int n4, bool tail2, int IW4,
                                           int NC4, const unsigned long long *gt)
{
    f2 part[2][8];
#pragma unroll
    for (int p = 0; p < 2; ++p)
#pragma unroll
        for (int e = 0; e < 8; ++e) part[p][e] = bc(0.0f);
    InRow A, B, C, D;
    load_row<NTX>(A, in_r);
    load_row<NTX>(B, in_r + IW4);
    load_row<NTX>(C, in_r + 2 * IW4);
    load_row<NTX>(D, in_r + 3 * IW4);
    in_r += 4 * IW4;
#pragma unroll 1
    for (int j4 = 0; j4 < n4; ++j4) {
        tap_step<NT, GT>(part, A, C, iq, gt);
        load_row<NTX>(A, in_r);
        tap_step<NT, GT>(part, B, D, iq + NC4, gt);
        load_row<NTX>(B, in_r + IW4);
        tap_step<NT, GT>(part, C, A, iq + 2 * NC4, gt);
        load_row<NTX>(C, in_r + 2 * IW4);
        tap_step<NT, GT>(part, D, B, iq + 3 * NC4, gt);
        load_row<NTX>(D, in_r + 3 * IW4);
        in_r += 4 * IW4;
        iq += 4 * NC4;
    }
    if (tail2) {
        tap_step<NT, GT>(part, A, C, iq, gt);
        tap_step<NT, GT>(part, B, D, iq + NC4, gt);
    }
#pragma unroll
    for (int p = 0; p < 2; ++p)
#pragma unroll
        for (int e = 0; e < 8; ++e) acc[p][e] = add2(acc[p][e], part[p][e]);
}

// __maxnreg__(176) instead of __launch_bounds__: with the looser budget of (256, 1) ptxas rotates one
// staged row through 16 MOVs per loop body (317 instructions); capped at 176 it allocates the four
// rows without moves (301; 157 registers used, no spills) -- profiles/r2b.md.
template <bool RENDER, int NTX, bool GT>
__global__ void __maxnreg__(176) conv_kernel(const __grid_constant__ ConvArgs a,
                                                                             const __grid_constant__ CUtensorMap tmap)
{
    constexpr int kThreads = Shape<NTX>::kThreads, kGroup = Shape<NTX>::kGroup, kTW = Shape<NTX>::kTW;
    const unsigned long long *gt = a.gtaps;
    extern __shared__ __align__(128) float4 smem4[];
    const int IW4 = kTW / 4 + a.NC, IW = 4 * IW4;
    const int IH = kTH + a.KH - 1 + kSlackRows;
    const int stage_floats = (IH * IW + 31) / 32 * 32;                    // stages start on 128-byte boundaries (TMA)
    float *s_stage = reinterpret_cast<float *>(smem4);                    // [n_stages][IH][IW]
    float *s_d = s_stage + (size_t)a.n_stages * stage_floats;             // [kTH][kTW] data      (loglike)
    float *s_w = s_d + kTH * kTW;                                         // [kTH][kTW] weights   (loglike)
    __shared__ double s_red[kThreads / 32];
#if LENSED_CONV_TMA
    __shared__ __align__(8) unsigned long long s_bar[2];
    if (threadIdx.x == 0) {
        mbar_init(&s_bar[0], 1);
        mbar_init(&s_bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
#endif

    // this block's share of the (tile, vector) items, tile-major
    const long long n_items = (long long)a.n_tiles * a.nb;
    const int lo = (int)(n_items * blockIdx.x / gridDim.x), hi = (int)(n_items * (blockIdx.x + 1) / gridDim.x);
    if (lo >= hi) return;

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int tx = NTX == 16 ? (warp & 1) * 8 + (lane & 7) : (lane & 7);
    const int ty = (NTX == 16 ? (warp >> 1) : warp) * 4 + (lane >> 3);

    // input tile of an item -> stage s
    auto issue = [&](int item, int s) {
        const int t = item / a.nb, b = item - t * a.nb;
        const uint32_t tile = a.tiles[t];
        const int Y0 = a.oy + (int)(tile >> 16) * kTH, X0 = a.ox + (int)(tile & 0xffffu) * kTW;
        float *dst = s_stage + (size_t)s * stage_floats;
#if LENSED_CONV_TMA
        if (threadIdx.x == 0) {                   // one thread, one copy; completion on the stage's mbarrier
            mbar_expect_tx(&s_bar[s], (unsigned)((IH - kSlackRows) * IW * sizeof(float)));
            tma_load_3d(dst, &tmap, &s_bar[s], X0, Y0, b);
        }
#else                                             // all threads; one commit group
        const float *src = a.Lp + (size_t)b * a.lp_stride + (size_t)Y0 * a.Wp + X0;
        for (int i = threadIdx.x; i < (IH - kSlackRows) * IW4; i += kThreads) {
            const int r = i / IW4, c4 = i - r * IW4;
            cp_async16(dst + r * IW + 4 * c4, src + (size_t)r * a.Wp + 4 * c4);
        }
        cp_async_commit();
#endif
    };

    issue(lo, 0);
    int cur_t = -1;
    bool warp_any = true;
    const int NC4 = 4 * a.NC;
    const int n4 = (a.KH + 1) >> 2;                 // KH + 1 steps (KH is odd): n4 bodies of four
    const bool tail2 = ((a.KH + 1) & 2) != 0;       // + two more

#pragma unroll 1
    for (int item = lo; item < hi; ++item) {
        const int s = a.n_stages == 2 ? ((item - lo) & 1) : 0;
        const int t = item / a.nb, b = item - t * a.nb;
        const uint32_t tile = a.tiles[t];
        const int Y0 = a.oy + (int)(tile >> 16) * kTH, X0 = a.ox + (int)(tile & 0xffffu) * kTW;
        const bool more = item + 1 < hi;
        if (a.n_stages == 2 && more) issue(item + 1, s ^ 1);

        if (!RENDER && t != cur_t) {
            // data and weights of this tile position (the previous item's epilogue is done:
            // barrier at the end of the loop body); w = 0 outside the image
            for (int i = threadIdx.x; i < kTH * kTW / 4; i += kThreads) {
                const int r = i / (kTW / 4), c = 4 * (i - r * (kTW / 4));
                const int y = Y0 + r;
                float dv[4], wv[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int x = X0 + c + e;
                    const bool in = y < a.H && x < a.W;
                    dv[e] = in ? a.image[(size_t)y * a.W + x] : 0.0f;
                    wv[e] = in ? a.wmask[(size_t)y * a.W + x] : 0.0f;
                }
                *reinterpret_cast<float4 *>(s_d + r * kTW + c) = make_float4(dv[0], dv[1], dv[2], dv[3]);
                *reinterpret_cast<float4 *>(s_w + r * kTW + c) = make_float4(wv[0], wv[1], wv[2], wv[3]);
            }
        }
#if LENSED_CONV_TMA
        mbar_wait(&s_bar[s], a.n_stages == 2 ? (((item - lo) >> 1) & 1) : ((item - lo) & 1));
#else
        if (a.n_stages == 2 && more) cp_async_wait<1>(); else cp_async_wait<0>();
#endif
        __syncthreads();

        if (t != cur_t) {
            cur_t = t;
            if (!RENDER) {
                // warps whose 16 x 64 outputs are all masked skip the convolution
                bool any = false;
#pragma unroll
                for (int o = 0; o < kTR; ++o)
#pragma unroll
                    for (int g = 0; g < 2; ++g) {
                        const float4 w4 = *reinterpret_cast<const float4 *>(s_w + (ty * kTR + o) * kTW + 4 * tx + g * kGroup);
                        any = any || w4.x != 0.0f || w4.y != 0.0f || w4.z != 0.0f || w4.w != 0.0f;
                    }
                warp_any = __any_sync(0xffffffffu, any);
            }
        }

        // acc[pair][column]: running sum over tap-column chunks; part: the current chunk
        f2 acc[2][8];
#pragma unroll
        for (int p = 0; p < 2; ++p)
#pragma unroll
            for (int e = 0; e < 8; ++e) acc[p][e] = bc(0.0f);

        if (warp_any) {
            const float4 *in_base = reinterpret_cast<const float4 *>(s_stage + (size_t)s * stage_floats) +
                                    (size_t)(ty * kTR) * IW4 + tx;
            const int last_taps = a.KW - 4 * (a.NC - 1);          // taps of the last chunk, 1..4
            const int n_full = last_taps == 4 ? a.NC : a.NC - 1;
#pragma unroll 1
            for (int c = 0; c < n_full; ++c)
                conv_chunk<4, NTX, GT>(acc, in_base + c, a.tap_off + 4 * c, n4, tail2, IW4, NC4, gt);
            if (last_taps != 4) {
                const float4 *in_r = in_base + n_full;
                const int iq = a.tap_off + 4 * n_full;
                if (last_taps == 3) conv_chunk<3, NTX, GT>(acc, in_r, iq, n4, tail2, IW4, NC4, gt);
                else if (last_taps == 2) conv_chunk<2, NTX, GT>(acc, in_r, iq, n4, tail2, IW4, NC4, gt);
                else conv_chunk<1, NTX, GT>(acc, in_r, iq, n4, tail2, IW4, NC4, gt);
            }
        }

        float out[kTR][8];
#pragma unroll
        for (int p = 0; p < 2; ++p)
#pragma unroll
            for (int e = 0; e < 8; ++e) un2(acc[p][e], out[2 * p][e], out[2 * p + 1][e]);

        const int oy = Y0 + ty * kTR, ox = X0 + tx * 4;
        if (RENDER) {
            const bool valid = a.derived[(size_t)b * a.D] != 0.0f;
            float *mb = a.model + (size_t)b * a.H * a.W;
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
                    for (int g = 0; g < 2; ++g) {
                        const int off = (ty * kTR + o) * kTW + 4 * tx + g * kGroup;
                        const float4 w4 = *reinterpret_cast<const float4 *>(s_w + off);
                        const float4 d4 = *reinterpret_cast<const float4 *>(s_d + off);
                        const float wv[4] = {w4.x, w4.y, w4.z, w4.w}, dv[4] = {d4.x, d4.y, d4.z, d4.w};
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            if (wv[e] != 0.0f) {           // masked pixels may see untraced L: never touch them
                                const float diff = dv[e] - out[o][4 * g + e];
                                part = fmaf(wv[e] * diff, diff, part);
                            }
                    }
            }
            double sum = (double)part;
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, off);
            if (lane == 0) s_red[warp] = sum;
            __syncthreads();
            if (threadIdx.x == 0) {
                double tot = 0.0;
                for (int i = 0; i < kThreads / 32; ++i) tot += s_red[i];
                a.partial[(size_t)b * a.n_tiles + t] = tot;
            }
        }
        __syncthreads();           // stage s and s_red are free again
        if (a.n_stages == 1 && more) issue(item + 1, 0);
    }
}


// ---- "strip" shape: every warp is its own worker ---------------------------------------------
// Eight ONE-WARP blocks per SM and no block-level step at all: a work item is (16 x 64 output
// strip, parameter vector), items are ordered strip-major and split evenly over all warps of the
// grid, and a warp owns its input stage(s) in shared memory, its mbarrier(s) and its TMA copies
// (lane 0 issues; box = (16 + KH - 1) rows x (64 + 4 NC) floats).  One warp per block; eight blocks
// per SM are resident because 8 x (registers, shared memory) fit.  The register cap is part of the
// code generation (cuobjdump, profiles/r2b.md): capped at 224 ptxas keeps the tap pairs on the
// uniform datapath (LDCU + UR operands, 305 instructions per loop body); with 255, or with a
// minimum block count in __launch_bounds__, it moves them to vector registers (LDC + 24-28 MOV,
// 327 instructions, 14 % slower).
// What the block shapes above
// lose at their barriers -- the tile prologue (wait for the copy), the epilogue (chi-square
// reduction) and the ramps of the chunk loops, during which a block's warps all leave the FMA pipe
// together -- a warp here loses alone, while the other warp of its scheduler keeps the pipe busy.
// Masked images skip work per strip instead of per tile, and the strips of every 16-row band
// start at the band's own first counted column (api.cu strip_list; a.tiles holds PIXEL
// coordinates for this shape): SLACS annulus, 68 % of the computed pixels are counted instead of 49 %.  The per-thread arithmetic (thread tile 4 x 8, tap pairs,
// rotating rows, blocked summation) is the code of the block shapes, so the results agree with
// theirs bit for bit per pixel; the chi-square partials are per strip.
// Data d and weights w of a strip are loaded once per strip and stay in registers for all its
// vectors (64 of the 255 a one-warp block may use); stages are double buffered when 16 of them fit.
constexpr int kSH = 16, kSW = 64;      // strip: the 4 x 8 lanes of a warp on 4 x 8 thread tiles
constexpr int kStripWarps = 8;
// staged row pitch in float4: strip width + 4 NC; half-width strips pad it to an odd number of float4
// (4 mod 8 floats): see conv_strip_kernel HALF
__host__ __device__ constexpr int strip_pitch4(int NC, bool half) { return half ? (8 + NC) | 1 : kSW / 4 + NC; }

// HALF: strips of 16 x 32 pixels, each half-warp on its own parameter vector (same strip, vectors
// 2 pb and 2 pb + 1; ONE tensor copy with a box two vectors deep fetches both tiles).  For masked
// images: the narrower strips hug the mask better (SLACS annulus: 80 % of the computed pixels are
// counted against 68 % with 64-wide strips).  Thread tile, taps and loops are the same; the staged
// row pitch is kept at 4 (mod 8) floats so that the 4 + 4 lanes of a quarter-warp, two tile rows
// apart in pitch, fall on different halves of the banks.
template <bool RENDER, bool GT, bool HALF>
__global__ void __maxnreg__(224) conv_strip_kernel(const __grid_constant__ ConvArgs a,
                                                   const __grid_constant__ CUtensorMap tmap)
{
    constexpr int NTX = HALF ? 4 : 8, kGroup = 4 * NTX, kW = 2 * kGroup;
    const unsigned long long *gt = a.gtaps;
    extern __shared__ __align__(128) float4 smem4[];
    __shared__ __align__(8) unsigned long long s_bar[2];
    const int lane = threadIdx.x;
    const int IW4 = strip_pitch4(a.NC, HALF), IW = 4 * IW4;
    const int IH = kSH + a.KH - 1 + kSlackRows;
    const int slab4 = (IH - kSlackRows) * IW4;                       // one vector's tile, float4 units
    const int stage_floats = ((HALF ? 2 : 1) * 4 * slab4 + kSlackRows * IW + 31) / 32 * 32;
    float *s_stage = reinterpret_cast<float *>(smem4);
    if (lane == 0) {
        mbar_init(&s_bar[0], 1);
        mbar_init(&s_bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();

    const int n_sub = HALF ? (a.nb + 1) >> 1 : a.nb;                 // items per strip: vectors, or pairs of vectors
    const long long n_items = (long long)a.n_tiles * n_sub;
    const int lo = (int)(n_items * blockIdx.x / gridDim.x), hi = (int)(n_items * (blockIdx.x + 1) / gridDim.x);
    if (lo >= hi) return;
    const int half = HALF ? lane >> 4 : 0;
    const int tx = lane & (NTX - 1), ty = (lane >> (HALF ? 2 : 3)) & 3;

    auto issue = [&](int item, int s) {
        if (lane == 0) {
            const int t = item / n_sub, pb = item - t * n_sub;
            const uint32_t tile = a.tiles[t];
            mbar_expect_tx(&s_bar[s], (unsigned)((HALF ? 2 : 1) * 4 * slab4 * sizeof(float)));
            tma_load_3d(s_stage + (size_t)s * stage_floats, &tmap, &s_bar[s], (int)(tile & 0xffffu), (int)(tile >> 16),
                        HALF ? 2 * pb : pb);
        }
    };

    issue(lo, 0);
    int cur_t = -1;
    bool warp_any = true;
    float wreg[kTR][8], dreg[kTR][8];          // weights and data of the current strip (loglike)
    const int NC4 = 4 * a.NC;
    const int n4 = (a.KH + 1) >> 2;
    const bool tail2 = ((a.KH + 1) & 2) != 0;

#pragma unroll 1
    for (int item = lo; item < hi; ++item) {
        const int s = a.n_stages == 2 ? ((item - lo) & 1) : 0;
        const int t = item / n_sub, pb = item - t * n_sub;
        const int b = HALF ? 2 * pb + half : pb;                      // this (half-)warp's parameter vector
        const bool has_b = b < a.nb;                                  // odd batch: the last pair's second half idles
        const uint32_t tile = a.tiles[t];
        const int oy = (int)(tile >> 16) + ty * kTR, ox = (int)(tile & 0xffffu) + tx * 4;      // strips carry pixel coordinates
        const bool more = item + 1 < hi;
        if (a.n_stages == 2 && more) issue(item + 1, s ^ 1);      // its last readers passed the __syncwarp below

        if (!RENDER && t != cur_t) {
            // data and weights of the strip stay in REGISTERS for all its vectors (a one-warp block
            // may use 255 of them): loaded once per strip, no epilogue latency.  w = 0 outside the image.
            cur_t = t;
            bool any = false;
#pragma unroll
            for (int o = 0; o < kTR; ++o)
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int y = oy + o, x = ox + (e & 3) + (e >> 2) * kGroup;
                    const bool in = y < a.H && x < a.W;
                    wreg[o][e] = in ? __ldg(a.wmask + (size_t)y * a.W + x) : 0.0f;
                    dreg[o][e] = in ? __ldg(a.image + (size_t)y * a.W + x) : 0.0f;
                    any = any | (wreg[o][e] != 0.0f);
                }
            warp_any = __any_sync(0xffffffffu, any);
        }
        mbar_wait(&s_bar[s], a.n_stages == 2 ? (((item - lo) >> 1) & 1) : ((item - lo) & 1));
        __syncwarp();              // lanes leave the wait loop one by one

        f2 acc[2][8];
#pragma unroll
        for (int p = 0; p < 2; ++p)
#pragma unroll
            for (int e = 0; e < 8; ++e) acc[p][e] = bc(0.0f);
        if (warp_any) {
            const float4 *in_base = reinterpret_cast<const float4 *>(s_stage + (size_t)s * stage_floats) +
                                    (size_t)half * slab4 + (size_t)(ty * kTR) * IW4 + tx;
            const int last_taps = a.KW - 4 * (a.NC - 1);
            const int n_full = last_taps == 4 ? a.NC : a.NC - 1;
#pragma unroll 1
            for (int c = 0; c < n_full; ++c)
                conv_chunk<4, NTX, GT>(acc, in_base + c, a.tap_off + 4 * c, n4, tail2, IW4, NC4, gt);
            if (last_taps != 4) {
                const float4 *in_r = in_base + n_full;
                const int iq = a.tap_off + 4 * n_full;
                if (last_taps == 3) conv_chunk<3, NTX, GT>(acc, in_r, iq, n4, tail2, IW4, NC4, gt);
                else if (last_taps == 2) conv_chunk<2, NTX, GT>(acc, in_r, iq, n4, tail2, IW4, NC4, gt);
                else conv_chunk<1, NTX, GT>(acc, in_r, iq, n4, tail2, IW4, NC4, gt);
            }
        }
        float out[kTR][8];
#pragma unroll
        for (int p = 0; p < 2; ++p)
#pragma unroll
            for (int e = 0; e < 8; ++e) un2(acc[p][e], out[2 * p][e], out[2 * p + 1][e]);

        if (RENDER) {
            if (has_b) {
                const bool valid = a.derived[(size_t)b * a.D] != 0.0f;
                float *mb = a.model + (size_t)b * a.H * a.W;
#pragma unroll
                for (int o = 0; o < kTR; ++o)
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const int y = oy + o, x = ox + (e & 3) + (e >> 2) * kGroup;
                        if (y < a.H && x < a.W) mb[(size_t)y * a.W + x] = valid ? out[o][e] : nanf("");
                    }
            }
        } else {
            float part = 0.0f;
            if (warp_any) {
#pragma unroll
                for (int o = 0; o < kTR; ++o)
#pragma unroll
                    for (int e = 0; e < 8; ++e)
                        if (wreg[o][e] != 0.0f) {          // masked pixels may see untraced L: never touch them
                            const float diff = dreg[o][e] - out[o][e];
                            part = fmaf(wreg[o][e] * diff, diff, part);
                        }
            }
            double sum = (double)part;                      // over the lanes of this vector: the warp, or its half
#pragma unroll
            for (int off = HALF ? 8 : 16; off > 0; off >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, off);
            if ((lane & (HALF ? 15 : 31)) == 0 && has_b) a.partial[(size_t)b * a.n_tiles + t] = sum;
        }
        __syncwarp();              // every lane is done with stage s
        if (a.n_stages == 1 && more) issue(item + 1, 0);
    }
}

// logL[b] = -1/2 sum over tiles, in tile order; -inf for vectors outside the model domain
__global__ void final_kernel(FinalArgs a)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= a.B) return;
    if (a.derived[(size_t)b * a.D] == 0.0f) { a.logl[b] = -INFINITY; return; }
    double chi2 = 0.0;
    for (int t = 0; t < a.n_tiles; ++t) chi2 += a.partial[(size_t)b * a.n_tiles + t];
    a.logl[b] = (float)(-0.5 * chi2);
}

}  // namespace

// shape: 0 = narrow, 1 = wide, 2 = strip, 3 = half-width strip (ConvArgs::shape)
void conv_tile_shape(int shape, int *tile_w, int *tile_h)
{
    *tile_w = shape == 1 ? Shape<16>::kTW : shape == 0 ? Shape<8>::kTW : shape == 2 ? kSW : kSW / 2;
    *tile_h = shape >= 2 ? kSH : kTH;
}

// rows x cols = the image rounded up to cover every tile of the grids in use (api.cu)
void conv_padded_shape(int rows, int cols, int KH, int NC, int *Hp, int *Wp)
{
    *Hp = rows + KH - 1;
    *Wp = (cols + 3) / 4 * 4 + 4 * NC + 4;               // + 4: the padded pitch of the half-width strips' boxes
}

namespace {
// dynamic shared memory a block may take: 227 KB per SM minus the static arrays, per resident block
size_t smem_limit(int shape) { return shape == 0 ? 112 * 1024 : shape >= 2 ? 28 * 1024 : 226 * 1024; }   // strips: 8 blocks per SM
size_t stage_bytes(int KH, int NC, int shape)
{
    size_t floats;
    if (shape >= 2) {
        const size_t IW = 4 * (size_t)strip_pitch4(NC, shape == 3);
        floats = (shape == 3 ? 2 : 1) * (size_t)(kSH + KH - 1) * IW + kSlackRows * IW;
    } else {
        int tw, th;
        conv_tile_shape(shape, &tw, &th);
        floats = (size_t)(th + KH - 1 + kSlackRows) * (tw + 4 * NC);
    }
    return (floats + 31) / 32 * 32 * sizeof(float);
}
// d and w of a tile staged in shared memory (block shapes, loglike); the strip shapes keep them in registers
size_t dw_bytes(bool render, int shape) { return render || shape >= 2 ? 0 : (size_t)2 * kTH * (shape == 1 ? 128 : 64) * sizeof(float); }
}  // namespace

int conv_num_stages(int KH, int NC, bool render, int shape)
{
    return 2 * stage_bytes(KH, NC, shape) + dw_bytes(render, shape) <= smem_limit(shape) ? 2 : 1;
}

size_t conv_smem_bytes(int KH, int NC, bool render, int shape)
{
    return conv_num_stages(KH, NC, render, shape) * stage_bytes(KH, NC, shape) + dw_bytes(render, shape);
}

// the narrow shape needs its single stage + d, w to fit twice per SM; the strip shape one stage eight times
bool conv_shape_fits(int KH, int NC, int shape)
{
    return shape == 1 || stage_bytes(KH, NC, shape) + dw_bytes(false, shape) <= smem_limit(shape);
}

namespace {
template <bool RENDER, int NTX, bool GT>
cudaError_t set_attr()
{
    return cudaFuncSetAttribute(conv_kernel<RENDER, NTX, GT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)smem_limit(NTX == 16 ? 1 : 0));
}
template <bool RENDER, bool GT, bool HALF>
cudaError_t set_attr_strip()
{
    return cudaFuncSetAttribute(conv_strip_kernel<RENDER, GT, HALF>, cudaFuncAttributeMaxDynamicSharedMemorySize, 226 * 1024);
}
template <bool RENDER, int NTX, bool GT>
void launch(const ConvArgs &a, const CUtensorMap &tmap, int grid, size_t smem, cudaStream_t st)
{
    conv_kernel<RENDER, NTX, GT><<<grid, NTX * kNTY, smem, st>>>(a, tmap);
}
template <bool RENDER, bool GT>
void launch_strip(const ConvArgs &a, const CUtensorMap &tmap, int grid, size_t smem, cudaStream_t st)
{
    if (a.shape == 3) conv_strip_kernel<RENDER, GT, true><<<grid, 32, smem, st>>>(a, tmap);
    else conv_strip_kernel<RENDER, GT, false><<<grid, 32, smem, st>>>(a, tmap);
}
}  // namespace

cudaError_t conv_setup()
{
    cudaError_t e;
#define LENSED_SET(R, N, G) if ((e = set_attr<R, N, G>()) != cudaSuccess) return e;
    LENSED_SET(false, 16, false) LENSED_SET(true, 16, false) LENSED_SET(false, 8, false) LENSED_SET(true, 8, false)
    LENSED_SET(false, 16, true) LENSED_SET(true, 16, true) LENSED_SET(false, 8, true) LENSED_SET(true, 8, true)
#undef LENSED_SET
#define LENSED_SET(R, G) if ((e = set_attr_strip<R, G, false>()) != cudaSuccess || (e = set_attr_strip<R, G, true>()) != cudaSuccess) return e;
    LENSED_SET(false, false) LENSED_SET(true, false) LENSED_SET(false, true) LENSED_SET(true, true)
#undef LENSED_SET
    return cudaSuccess;
}

cudaError_t conv_upload_taps(const float *pairs, int n_pairs, int pool_offset)
{
    return cudaMemcpyToSymbol(c_taps, pairs, (size_t)n_pairs * sizeof(unsigned long long),
                              (size_t)pool_offset * sizeof(unsigned long long), cudaMemcpyHostToDevice);
}

// Tensor map of the padded frames L[n_frames][Hp][Wp] for boxes of one input tile with its halo
// (conv_kernel "issue").  out: 128 bytes, 64-byte aligned.  The encoder is a driver entry point
// fetched through the runtime, so the library links against nothing but the static runtime.
cudaError_t conv_make_tensor_map(void *out, const float *L, int Wp, int Hp, long long n_frames, int KH, int NC, int shape)
{
    static PFN_cuTensorMapEncodeTiled_v12000 encode = nullptr;
    if (!encode) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult qr;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr);
        if (e != cudaSuccess) return e;
        if (!fn || qr != cudaDriverEntryPointSuccess) return cudaErrorNotSupported;
        encode = (PFN_cuTensorMapEncodeTiled_v12000)fn;
    }
    const cuuint64_t dims[3] = {(cuuint64_t)Wp, (cuuint64_t)Hp, (cuuint64_t)std::max<long long>(n_frames, 1)};
    const cuuint64_t strides[2] = {(cuuint64_t)Wp * sizeof(float), (cuuint64_t)Wp * Hp * sizeof(float)};
    int tw, th;
    conv_tile_shape(shape, &tw, &th);
    const cuuint32_t box[3] = {(cuuint32_t)(shape >= 2 ? 4 * strip_pitch4(NC, shape == 3) : tw + 4 * NC), (cuuint32_t)(th + KH - 1),
                               (cuuint32_t)(shape == 3 ? 2 : 1)};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = encode((CUtensorMap *)out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void *)L, dims, strides, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

// n_sm: persistent blocks = n_sm x (blocks per SM of the shape), fewer when there are fewer items
cudaError_t launch_conv(ConvArgs a, const void *tensor_map, bool render, int n_sm, cudaStream_t st)
{
    const CUtensorMap &tmap = *reinterpret_cast<const CUtensorMap *>(tensor_map);
    const bool gt = a.gtaps != nullptr;
    a.n_stages = conv_num_stages(a.KH, a.NC, render, a.shape);
    size_t smem = conv_smem_bytes(a.KH, a.NC, render, a.shape);
    const long long n_items = (long long)a.n_tiles * a.nb;
    if (a.shape >= 2) {
        const long long n_strip_items = (long long)a.n_tiles * (a.shape == 3 ? (a.nb + 1) / 2 : a.nb);
        // k one-warp blocks per SM: the request is padded so that exactly k fit (228 KB per SM, 1 KB
        // reserved per block) -- otherwise the block scheduler packs up to 12 on some SMs and leaves
        // others empty
        static const int k_env = [] { const char *e = getenv("LENSED_STRIP_WARPS"); return e ? atoi(e) : 0; }();   // tuning
        int k = k_env > 0 ? k_env : kStripWarps;
        k = std::max(1, std::min(k, (int)((228 * 1024) / (smem + 1024 + 64))));
        smem = std::max(smem, (size_t)((228 * 1024) / k - 1024 - 64) / 128 * 128);
        const long long n_warps = (long long)n_sm * k;
        const int grid = (int)(n_strip_items < n_warps ? n_strip_items : n_warps);
        if (grid < 1) return cudaSuccess;
        if (render) { if (gt) launch_strip<true, true>(a, tmap, grid, smem, st); else launch_strip<true, false>(a, tmap, grid, smem, st); }
        else        { if (gt) launch_strip<false, true>(a, tmap, grid, smem, st); else launch_strip<false, false>(a, tmap, grid, smem, st); }
        return cudaGetLastError();
    }
    const bool wide = a.shape == 1;
    const long long n_blocks = (long long)n_sm * (wide ? 1 : 2);
    const int grid = (int)(n_items < n_blocks ? n_items : n_blocks);
    if (grid < 1) return cudaSuccess;
#define LENSED_GO(R, N, G) launch<R, N, G>(a, tmap, grid, smem, st)
    if (wide) { if (render) { if (gt) LENSED_GO(true, 16, true); else LENSED_GO(true, 16, false); }
                else        { if (gt) LENSED_GO(false, 16, true); else LENSED_GO(false, 16, false); } }
    else      { if (render) { if (gt) LENSED_GO(true, 8, true); else LENSED_GO(true, 8, false); }
                else        { if (gt) LENSED_GO(false, 8, true); else LENSED_GO(false, 8, false); } }
#undef LENSED_GO
    return cudaGetLastError();
}

cudaError_t launch_final(const FinalArgs &a, cudaStream_t st)
{
    final_kernel<<<(a.B + 127) / 128, 128, 0, st>>>(a);
    return cudaGetLastError();
}

}  // namespace lensed
