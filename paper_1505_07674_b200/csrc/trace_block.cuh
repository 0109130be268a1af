// trace_block.cuh -- what every ray-tracer kernel shares: block size, the block prologue
// (constants of the block's parameter vector and its frame tables into shared memory) and
// the launch helper.  Included by trace.cu (interpreted model list) and trace_static.cuh
// (model list fixed at compile time).
//
// Shared memory of a block: [D/4] float4 derived constants of its vector, then the frame
// tables  tab[slot][2][nq_pad]  (slot 0 = identity, 1 + m = lens m, 1 + n_lens + m = light
// m; lenses and lights in the canonical order of api.cu), then the rule weights [nq_pad] and
// the difference weights of the embedded rule [nq_pad].
#pragma once
#include "trace_math.cuh"

namespace lensed {

struct FgMoments;

#ifndef LENSED_TRACE_THREADS
#define LENSED_TRACE_THREADS 256          // tuning builds: 128 with twice the resident blocks
#endif
constexpr int kTraceThreads = LENSED_TRACE_THREADS;

struct TraceBlock {
    const float4 *sder;   // derived constants of the vector
    const float *stab;    // frame tables
    const float *sw;      // rule weights
    const float *sdw;     // rule weights minus the embedded rule's (error estimate, trace.cu)
    float4 *smat;         // [n_light] scratch matrices (trace_static.cuh "direct frames")
    struct FgMoments *sfgx; // [n_light] rule moments per foreground Sersic (trace_static.cuh "foreground expansion")
    float sky;            // summed sky levels
    bool valid;
};

// the chunk-local parameter vector of this block (TraceArgs::order)
__device__ __forceinline__ int trace_vector(const TraceArgs &a) { return a.order ? a.order[blockIdx.y] : (int)blockIdx.y; }

// Must be called by all threads of the block; ends with a barrier.
__device__ __forceinline__ TraceBlock trace_prologue(const Program &prog, const TraceArgs &a, float4 *smem4, int vec)
{
    float4 *sder = smem4;
    float *stab = reinterpret_cast<float *>(smem4 + prog.D / 4);
    const int nq = a.nq_pad;
    const int n_slots = 1 + prog.n_lens + prog.n_light;
    float *sw = stab + (size_t)n_slots * 2 * nq;
    {
        const float4 *g = reinterpret_cast<const float4 *>(a.derived + (size_t)vec * prog.D);
        for (int i = threadIdx.x; i < prog.D / 4; i += kTraceThreads) sder[i] = g[i];
    }
    __syncthreads();
    float *sdw = sw + nq;
    float4 *smat = reinterpret_cast<float4 *>(sdw + nq);      // nq is even and the tables are 16-byte aligned
    TraceBlock tb{sder, stab, sw, sdw, smat, reinterpret_cast<struct FgMoments *>(smat + prog.n_light), 0.0f,
                  sder[0].x != 0.0f};
    if (!tb.valid) return tb;                     // vector outside the model domain: block-uniform
    for (int m = 0; m < prog.n_light; ++m)
        if (prog.light_kind[m] == K_SKY) tb.sky += sder[prog.light_off[m] >> 2].x;
    for (int i = threadIdx.x; i < n_slots * nq; i += kTraceThreads) {
        const int slot = i / nq, k = i - slot * nq;
        const float4 qk = a.quad[k];
        float m11 = 1.0f, m12 = 0.0f, m21 = 0.0f, m22 = 1.0f;
        if (slot > 0) {
            const bool lens = slot <= prog.n_lens;
            const int m = lens ? slot - 1 : slot - 1 - prog.n_lens;
            const int kind = lens ? prog.lens_kind[m] : prog.light_kind[m];
            const float4 *d = sder + ((lens ? prog.lens_off[m] : prog.light_off[m]) >> 2);
            if (kind == K_SIE) { m11 = d[1].x; m12 = d[1].y; m21 = -d[1].y; m22 = d[1].x; }
            else if (kind == K_SHEAR) { m11 = d[0].x; m12 = d[0].y; m21 = d[0].y; m22 = -d[0].x; }
            else if (kind >= K_SRC_SERSIC && kind <= K_FG_GAUSS) { m11 = d[1].x; m12 = d[1].y; m21 = d[1].z; m22 = d[1].w; }
        }
        stab[(size_t)(2 * slot) * nq + k] = fmaf(m11, qk.x, m12 * qk.y);
        stab[(size_t)(2 * slot + 1) * nq + k] = fmaf(m21, qk.x, m22 * qk.y);
        if (slot == 0) { sw[k] = qk.z; sdw[k] = qk.w; }
    }
    __syncthreads();
    return tb;
}

// L_i into the padded frame the convolution reads (conv.cu "Input"): pixel (row, col) at
// (row + py, col + px); a border pixel also fills the pad cells that clamp to it
// ("border pixels are repeated").
// The value is clamped to the finite range (NaN -> -FLT_MAX): the convolution multiplies every
// staged value by tap pairs whose partner may be a structural zero (conv.cu "Pairing"), and
// 0 x inf would put a NaN into an output whose PSF window does not hold the pixel at all.  A pixel
// that overflows FP32 still drives its own window to +-inf, i.e. logL to -inf.
__device__ __forceinline__ void store_pixel(const TraceArgs &a, float *Lb, int row, int col, float v)
{
    v = fminf(fmaxf(v, -3.402823466e38f), 3.402823466e38f);
    Lb[(size_t)(row + a.py) * a.Wp + col + a.px] = v;
    if (row == 0 || col == 0 || row == a.H - 1 || col == a.W - 1) {
        const int r0 = row == 0 ? 0 : row + a.py, r1 = row == a.H - 1 ? a.H - 1 + 2 * a.py : row + a.py;
        const int c0 = col == 0 ? 0 : col + a.px, c1 = col == a.W - 1 ? a.W - 1 + 2 * a.px : col + a.px;
        for (int r = r0; r <= r1; ++r)
            for (int c = c0; c <= c1; ++c) Lb[(size_t)r * a.Wp + c] = v;
    }
}

#ifndef __CUDACC_RTC__
template <class Kernel>
cudaError_t launch_trace_kernel(Kernel kernel, const Program &prog, const TraceArgs &a, int nvec, cudaStream_t st)
{
    const size_t smem = trace_smem_bytes(prog, a.nq_pad);
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    dim3 grid((a.npix + a.pix_per_block - 1) / a.pix_per_block, nvec);
    kernel<<<grid, kTraceThreads, smem, st>>>(prog, a);
    return cudaGetLastError();
}

#endif  // !__CUDACC_RTC__

}  // namespace lensed
