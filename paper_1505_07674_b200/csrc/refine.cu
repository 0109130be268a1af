// refine.cu -- FP64 re-trace of the few pixels per vector where FP32 ray positions are not enough.
//
// The tracer forms y = x - alpha(x) (eq. 1) in FP32: with |alpha| ~ 20 pixels the
// source-plane position carries ~1e-6 px of rounding noise.  A compact high-index Sersic source
// (eqs. 22-23; the paper's prior goes to n = 8, L252) turns a displacement dx
// into d ln I = (b_n/n) (R/r_S)^(1/n - 1) / (sqrt(q) r_S) dx, which near the centre of the profile
// exceeds 1e-5 / 1e-6 px: the one or two pixels that hold an image of the source's cusp then miss
// north_star's 1e-4 per pixel, and -- being the brightest pixels of the model -- carry most of the
// chi-square, so logL misses 1e-5 (measured in profiles/r2a.md).
//
// The tracer flags those pixels: per source Sersic it keeps the minimum of (R/r_S)^2 over the
// pixel's rays (one FMNMX3 per pair of rays) and compares it with the threshold T2 prep.cu
// derived from the profile's slope; each tracer thread leaves one 32-bit word, bit i = its i-th
// pixel (TraceArgs::fixmask).  This kernel scans the words and re-traces every flagged pixel --
// all rule points, all components -- in double precision from the unrounded constants
// (derived64), one warp per pixel with the rule points across the lanes, and overwrites the
// pixel's L before the convolution reads it.  Typically 1-20 pixels per vector.
//
// Deterministic: the set of flagged pixels is a function of the inputs and every flagged pixel
// is recomputed with a fixed-shape reduction; the queue between the two passes only spreads
// the work (its order and its capacity never change a value; the counter is a statistic).
#include "trace_block.cuh"
#include <math.h>
#include <algorithm>

namespace lensed {
namespace {

constexpr int kRefineThreads = 128;

// rotated offset from a component centre: (u, v) = R(-pa) (x - c)
__device__ __forceinline__ void frame64(const double *e, double x, double y, double &u, double &v)
{
    const double dx = x - e[0], dy = y - e[1];
    u = e[2] * dx + e[3] * dy;
    v = -e[3] * dx + e[2] * dy;
}

// I(x) of eq. 2 at the image-plane point (x, y), pixel-index coordinates; e = the vector's FP64 blocks
__device__ double brightness64(const Program &prog, const double *e, double x, double y, double cxh, double cyh)
{
    double ax = 0.0, ay = 0.0;
    for (int m = 0; m < prog.n_models; ++m) {
        const double *b = e + m * kD64PerModel;
        switch (prog.kind[m]) {
        case K_SIS: {                                   // R3: alpha = b (u, v)/r
            const double u = x - b[0], v = y - b[1], r = sqrt(u * u + v * v);
            if (r > 0.0) { ax += b[2] * u / r; ay += b[2] * v / r; }
            break;
        }
        case K_POINT: {                                 // R3: alpha = thetaE^2 (u, v)/r^2
            const double u = x - b[0], v = y - b[1], r2 = u * u + v * v;
            if (r2 > 0.0) { ax += b[2] * u / r2; ay += b[2] * v / r2; }
            break;
        }
        case K_SHEAR: {                                 // R4: about the image centre
            const double X = x - cxh, Y = y - cyh;
            ax += b[0] * X + b[1] * Y;
            ay += b[1] * X - b[0] * Y;
            break;
        }
        case K_SIE: {                                   // R2: Kormann et al. 1994
            double u, v;
            frame64(b, x, y, u, v);
            const double q = b[4], amp = b[5];
            const double psi = sqrt(q * q * u * u + v * v);
            if (psi > 0.0) {
                const double qp = sqrt((1.0 - q) * (1.0 + q)), sq = sqrt(q);
                double au, av;
                if (qp < 1e-7) { au = amp * sq * u / psi; av = amp * sq * v / psi; }   // q -> 1
                else { const double A = amp * sq / qp; au = A * atan(qp * u / psi); av = A * atanh(qp * v / psi); }
                ax += b[2] * au - b[3] * av;
                ay += b[3] * au + b[2] * av;
            }
            break;
        }
        default: break;
        }
    }
    const double sx = x - ax, sy = y - ay;              // eq. 1
    double I = 0.0;
    for (int m = 0; m < prog.n_models; ++m) {
        const double *b = e + m * kD64PerModel;
        const int kind = prog.kind[m];
        if (kind == K_SKY) { I += b[0]; continue; }
        if (kind < K_SRC_SERSIC) continue;
        const bool src = kind == K_SRC_SERSIC || kind == K_SRC_GAUSS;
        double u, v;
        frame64(b, src ? sx : x, src ? sy : y, u, v);
        const double R2 = (u * u * b[4] + v * v / b[4]) / (b[5] * b[5]);       // eq. 23, scaled by r_S | sigma
        if (kind == K_SRC_SERSIC || kind == K_FG_SERSIC) I += exp(b[8] - b[7] * pow(R2, 0.5 * b[6]));   // eq. 22
        else I += exp(b[6] - 0.5 * R2);                                                                // R7
    }
    return I;
}

// One flagged pixel, by the whole warp: rule points across the lanes, fixed-shape reduction.
__device__ __forceinline__ void refine_pixel(const Program &prog, const RefineArgs &a, int vec, int ip, int lane)
{
    const double *e = a.derived64 + (size_t)vec * prog.n_models * kD64PerModel;
    const uint32_t rc = a.t.pix[ip];
    const int row = (int)(rc >> 16), col = (int)(rc & 0xffffu);
    double sum = 0.0;
    for (int k = lane; k < a.n_quad; k += 32) {                 // eq. 14
        const float4 qk = a.t.quad[k];
        sum += (double)qk.z * brightness64(prog, e, (double)col + (double)qk.x, (double)row + (double)qk.y,
                                           (double)a.t.cxh, (double)a.t.cyh);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, off);
    if (lane == 0) store_pixel(a.t, a.t.L + (size_t)vec * a.t.l_stride, row, col, (float)sum);
}

// Pass 1: scan the tracer's flag words and queue the flagged pixels as (vector, list index).
// The queue only balances the load of pass 2 (flagged pixels come in clusters that one scanning
// warp would otherwise re-trace one after the other); its order does not matter, and a pixel
// that finds it full is re-traced here and now, so its capacity never changes a result.
__global__ void __launch_bounds__(kRefineThreads) refine_scan_kernel(Program prog, RefineArgs a)
{
    const int lane = threadIdx.x & 31;
    const long long warp = ((long long)blockIdx.x * kRefineThreads + threadIdx.x) >> 5;
    const long long n_warps = ((long long)gridDim.x * kRefineThreads) >> 5;
    const long long n_words = (long long)a.nvec * a.n_blocks * kTraceThreads;
    unsigned long long done = 0;
    for (long long w0 = warp * 32; w0 < n_words; w0 += n_warps * 32) {
        const uint32_t mine = w0 + lane < n_words ? a.t.fixmask[w0 + lane] : 0u;
        uint32_t any = __ballot_sync(0xffffffffu, mine != 0u);
        while (any) {
            const int src_lane = __ffs(any) - 1;
            any &= any - 1;
            uint32_t bits = __shfl_sync(0xffffffffu, mine, src_lane);
            const long long word = w0 + src_lane;
            const int thread = (int)(word % kTraceThreads);
            const long long vb = word / kTraceThreads;
            const int blk = (int)(vb % a.n_blocks), vec = (int)(vb / a.n_blocks);
            while (bits) {
                const int it = __ffs(bits) - 1;
                bits &= bits - 1;
                const int ip = blk * a.t.pix_per_block + it * kTraceThreads + thread;
                if (ip >= a.t.npix) continue;
                ++done;
                unsigned slot = 0;
                if (lane == 0) slot = atomicAdd(a.queue_count, 1u);
                slot = __shfl_sync(0xffffffffu, slot, 0);
                if (slot < (unsigned)a.queue_cap) {
                    if (lane == 0) a.queue[slot] = make_uint2((unsigned)vec, (unsigned)ip);
                } else {
                    refine_pixel(prog, a, vec, ip, lane);
                }
            }
        }
    }
    if (a.count && lane == 0 && done) atomicAdd(a.count, done);
}

// Pass 2: one warp per queued pixel.
__global__ void __launch_bounds__(kRefineThreads) refine_queue_kernel(Program prog, RefineArgs a)
{
    const int lane = threadIdx.x & 31;
    const unsigned warp = (blockIdx.x * kRefineThreads + threadIdx.x) >> 5;
    const unsigned n_warps = (gridDim.x * kRefineThreads) >> 5;
    const unsigned n = min(*a.queue_count, (unsigned)a.queue_cap);
    for (unsigned i = warp; i < n; i += n_warps) {
        const uint2 q = a.queue[i];
        refine_pixel(prog, a, (int)q.x, (int)q.y, lane);
    }
}

}  // namespace

cudaError_t launch_refine(const Program &prog, const RefineArgs &a, int n_sm, cudaStream_t st)
{
    const long long n_words = (long long)a.nvec * a.n_blocks * kTraceThreads;
    if (n_words < 1 || !a.t.fixmask) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(a.queue_count, 0, sizeof(unsigned), st);
    if (e != cudaSuccess) return e;
    const int wpb = kRefineThreads / 32;
    const long long want = (n_words + 32 * wpb - 1) / (32 * wpb);
    refine_scan_kernel<<<(int)std::min<long long>(want, (long long)n_sm * 8), kRefineThreads, 0, st>>>(prog, a);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    const long long wantq = ((long long)a.queue_cap + wpb - 1) / wpb;
    refine_queue_kernel<<<(int)std::min<long long>(wantq, (long long)n_sm * 16), kRefineThreads, 0, st>>>(prog, a);
    return cudaGetLastError();
}

}  // namespace lensed
