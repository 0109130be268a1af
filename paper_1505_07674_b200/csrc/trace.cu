// trace.cu -- steps a1-a4: ray generation, deflection summed over lenses, surface
// brightness, pixel quadrature, fused; one launch covers (pixel chunk) x (parameter vector).
//
//   x_k = pixel centre + (xi_k, eta_k)                       PAPER.md:155-159 eq. 14
//   y_k = x_k - sum_lenses alpha(x_k)                        PAPER.md:53-57  eq. 1
//   I   = sum_src I_S(y_k) + sum_fg I_L(x_k) + sky           PAPER.md:59-63  eq. 2
//   L_i = sum_k w_k I                                        PAPER.md:155-157 eq. 14
//
// Layout.  blockIdx.y -> parameter vector (TraceArgs::order), blockIdx.x = chunk of the traced-pixel list.  A
// thread owns one pixel at a time and carries R = 2 NP rays (rule points) in registers, as
// NP packed FP32 pairs (f32x2.cuh), through the model list.  No per-ray value ever goes to
// memory; one float per traced pixel is written.
//
// Every component works in its own linear frame  (u, v) = M (x - c):  rotation for the SIE,
// rotation + q-stretch + 1/r_S for Sersic / Gaussian, identity for SIS / point mass, the
// shear matrix itself for the shear.  Since x = pixel + rule offset,
//     (u, v) = M (pixel - c)  +  M (xi_k, eta_k)
//            =  per pixel, 6 flops per R rays  +  per (vector, k): a table in shared memory,
// so a ray enters a frame with ONE packed add per coordinate; the block builds the tables
// (frames x rule points) once in its prologue (trace_block.cuh).  Sources see the deflected
// position:  (u, v) = M (x - c) - M alpha,   two packed FMAs per coordinate.
// The shear is linear, so its whole deflection is "per pixel + table"; it is sorted to the
// front of the lens list (api.cu) and initialises alpha.  Sky is added once per pixel (the
// rule weights sum to one).
//
// Two kernels compute this: trace_static_kernel (trace_static.cuh), straight-line code for a
// model list fixed at compile time -- instantiated for the lists of trace_sig_*.cu -- and
// trace_kernel below, which interprets any list (a block-uniform switch per model).
// launch_trace picks the static one when the list's signature matches.
#include "trace_block.cuh"
#include "jit.h"
#include <stdlib.h>

namespace lensed {

// static signatures (trace_sig_*.cu)
#define LENSED_DECLARE_STATIC_TRACER(NAME)                                                              \
    bool NAME(const int (&counts)[K_COUNT], const Program &prog, const TraceArgs &a, int R, int nvec,   \
              cudaStream_t st, cudaError_t *err);
LENSED_DECLARE_STATIC_TRACER(trace_static_a)
LENSED_DECLARE_STATIC_TRACER(trace_static_b)
LENSED_DECLARE_STATIC_TRACER(trace_static_c)
LENSED_DECLARE_STATIC_TRACER(trace_static_d)
LENSED_DECLARE_STATIC_TRACER(trace_static_e)
LENSED_DECLARE_STATIC_TRACER(trace_static_f)
LENSED_DECLARE_STATIC_TRACER(trace_static_g)
LENSED_DECLARE_STATIC_TRACER(trace_static_h)
LENSED_DECLARE_STATIC_TRACER(trace_static_i)

namespace {

template <int NP>
__device__ __forceinline__ void sie_by_mode(int mode, const float4 *d, const float *tu, const float *tv, float u0,
                                            float v0, Rays<NP> &r)
{
    switch (mode) {
    case 0: lens_sie<NP, 0>(d, tu, tv, u0, v0, r); break;
    case 1: lens_sie<NP, 1>(d, tu, tv, u0, v0, r); break;
    case 2: lens_sie<NP, 2>(d, tu, tv, u0, v0, r); break;
    case 3: lens_sie<NP, 3>(d, tu, tv, u0, v0, r); break;
    case 4: lens_sie<NP, 4>(d, tu, tv, u0, v0, r); break;
    default: lens_sie<NP, 5>(d, tu, tv, u0, v0, r); break;
    }
}

// ERR: instead of L_i, write the error estimate of the pixel quadrature
//   | sum_k w_k I(x_k) - sum_k w'_k I(x_k) |,   w' = embedded lower-order rule,
// accumulated as sum_k (w_k - w'_k) I(x_k), into a.err[vector][H][W] (NaN for vectors outside
// the model domain).  A diagnostic output, not on the likelihood path: interpreter only.
#ifndef LENSED_MINB_GENERIC
#define LENSED_MINB_GENERIC 3      // Euclid list 49.5 -> 44.0 ms per 4096 vectors against 2 (multi-lens list 46.2 -> 47.1)
#endif
template <int NP, bool ERR>
__global__ void __launch_bounds__(kTraceThreads, LENSED_MINB_GENERIC) trace_kernel(Program prog, TraceArgs a)
{
    constexpr int R = 2 * NP;
    extern __shared__ float4 smem4[];
    const int vec = trace_vector(a);
    const TraceBlock tb = trace_prologue(prog, a, smem4, vec);
    if (!tb.valid) {
        if (!ERR && a.fixmask) a.fixmask[((size_t)vec * gridDim.x + blockIdx.x) * kTraceThreads + threadIdx.x] = 0;
        if (ERR) {
            const int base = blockIdx.x * a.pix_per_block, end = min(base + a.pix_per_block, a.npix);
            for (int ip = base + threadIdx.x; ip < end; ip += kTraceThreads) {
                const uint32_t rc = a.pix[ip];
                a.err[(size_t)vec * a.H * a.W + (size_t)(rc >> 16) * a.W + (rc & 0xffffu)] = nanf("");
            }
        }
        return;
    }
    const float4 *sder = tb.sder;
    const float *stab = tb.stab;
    const int nq = a.nq_pad;
    const int mode = (int)sder[0].y;
    float *Lb = a.L + (size_t)vec * a.l_stride;

    const int base = blockIdx.x * a.pix_per_block;
    const int end = min(base + a.pix_per_block, a.npix);
    uint32_t flags = 0;                // bit i: this thread's i-th pixel is flagged for refine.cu
#pragma unroll 1
    for (int ip = base + threadIdx.x; ip < end; ip += kTraceThreads) {
        const uint32_t rc = a.pix[ip];
        const int row = (int)(rc >> 16), col = (int)(rc & 0xffffu);
        const float jf = (float)col, rf = (float)row;
        f2 acc = bc(0.0f);
        bool flag = false;
#pragma unroll 1
        for (int q0 = 0; q0 < nq; q0 += R) {
            Rays<NP> r;
#pragma unroll
            for (int k = 0; k < NP; ++k) r.I[k] = bc(0.0f);
            int m = 0;
            float u0, v0;
            if (prog.n_lens > 0 && prog.lens_kind[0] == K_SHEAR) {
                shear_origin(sder + (prog.lens_off[0] >> 2), jf, rf, a.cxh, a.cyh, u0, v0);
                lens_shear<NP, true>(stab + 2 * nq + q0, stab + 3 * nq + q0, u0, v0, r);
                m = 1;
            } else {
#pragma unroll
                for (int k = 0; k < NP; ++k) { r.ax[k] = bc(0.0f); r.ay[k] = bc(0.0f); }
            }
#pragma unroll 1
            for (; m < prog.n_lens; ++m) {
                const float4 *d = sder + (prog.lens_off[m] >> 2);
                const float *tu = stab + (size_t)(2 * (1 + m)) * nq + q0, *tv = tu + nq;
                switch (prog.lens_kind[m]) {
                case K_SIE:
                    sie_origin(d, jf, rf, u0, v0);
                    sie_by_mode<NP>(mode, d, tu, tv, u0, v0, r);
                    break;
                case K_SIS:
                    circular_origin(d, jf, rf, u0, v0);
                    lens_circular<NP, false>(d, stab + q0, stab + nq + q0, u0, v0, r);
                    break;
                case K_POINT:
                    circular_origin(d, jf, rf, u0, v0);
                    lens_circular<NP, true>(d, stab + q0, stab + nq + q0, u0, v0, r);
                    break;
                default:
                    shear_origin(d, jf, rf, a.cxh, a.cyh, u0, v0);
                    lens_shear<NP, false>(tu, tv, u0, v0, r);
                    break;
                }
            }
#pragma unroll 1
            for (m = 0; m < prog.n_light; ++m) {
                const int kind = prog.light_kind[m];
                if (kind == K_SKY) continue;      // added once per pixel below
                const float4 *d = sder + (prog.light_off[m] >> 2);
                const float *tu = stab + (size_t)(2 * (1 + prog.n_lens + m)) * nq + q0, *tv = tu + nq;
                light_origin(d, jf, rf, u0, v0);
                float rmin = 3e38f;
                switch (kind) {
                case K_SRC_SERSIC:
                    light_profile<NP, true, false, false>(d, tu, tv, u0, v0, r, nullptr, rmin);
                    flag = flag || rmin < d[2].w;
                    break;
                case K_FG_SERSIC:  light_profile<NP, false, false, false>(d, tu, tv, u0, v0, r, nullptr, rmin); break;
                case K_SRC_GAUSS:  light_profile<NP, true, true, false>(d, tu, tv, u0, v0, r, nullptr, rmin); break;
                default:           light_profile<NP, false, true, false>(d, tu, tv, u0, v0, r, nullptr, rmin); break;
                }
            }
            f2 w[NP];
            load_pairs<NP>((ERR ? tb.sdw : tb.sw) + q0, w);
#pragma unroll
            for (int k = 0; k < NP; ++k) acc = fma2(w[k], r.I[k], acc);
        }
        if (ERR) a.err[(size_t)vec * a.H * a.W + (size_t)row * a.W + col] = fabsf(lo2(acc) + hi2(acc));
        else store_pixel(a, Lb, row, col, (lo2(acc) + hi2(acc)) + tb.sky);
        if (flag) flags |= 1u << ((ip - base) >> 8);
    }
    if (!ERR && a.fixmask) a.fixmask[((size_t)vec * gridDim.x + blockIdx.x) * kTraceThreads + threadIdx.x] = flags;
}

}  // namespace

size_t trace_smem_bytes(const Program &prog, int nq_pad)
{
    const size_t n_slots = 1 + prog.n_lens + prog.n_light;
    const size_t nq4 = ((size_t)nq_pad + 3) / 4 * 4;          // keeps the float4 scratch after the tables aligned
    return (size_t)prog.D * sizeof(float) + (n_slots * 2 + 2) * nq4 * sizeof(float) + (size_t)prog.n_light * (sizeof(float4) + 8 * sizeof(float));
}

// Rays carried per thread, R = 2 NP in {2, 4, 6, 8, 10}: least padded rule length, weighted
// by a per-pass overhead that shrinks with R (4 -> 4, 9 -> 10, 16 -> 8, 25 -> 4, 49 -> 10;
// measured on the multi-lens config, 25 points: R = 4 / 6 / 8 / 10 -> 34.8 / 37.3 / 38.9 / 38.8 ms).
int trace_pick_R(int n_quad)
{
#ifdef LENSED_TRACE_FORCE_R            // tuning builds (build.py defines=...)
    return LENSED_TRACE_FORCE_R;
#endif
    int best = 2;
    double best_cost = 1e300;
    for (int R = 2; R <= 10; R += 2) {
        const int pad = (n_quad + R - 1) / R * R;
        const double cost = pad * (1.0 + 0.4 / R);
        if (cost < best_cost - 1e-12) { best = R; best_cost = cost; }
    }
    return best;
}

// Rule points per pass of the pixel-pair tracers (trace_static.cuh), NP in {2, 3, 4, 5}: the
// least padded rule length, the larger NP on ties (4 -> 4, 9 -> 3, 16 -> 4, 25 -> 5, 49 -> 5).
int trace_pick_np(int n_quad)
{
#ifdef LENSED_TRACE_FORCE_NP           // tuning builds (build.py defines=...)
    return LENSED_TRACE_FORCE_NP;
#endif
    int best = 2, best_pad = 1 << 30;
    for (int np = 2; np <= 5; ++np) {
        const int pad = (n_quad + np - 1) / np * np;
        if (pad <= best_pad) { best = np; best_pad = pad; }
    }
    return best;
}

namespace {

// every static signature; a NULL err only asks whether the signature matches
typedef bool (*StaticTracer)(const int (&)[K_COUNT], const Program &, const TraceArgs &, int, int, cudaStream_t,
                             cudaError_t *);
const StaticTracer kStaticTracers[] = {trace_static_a, trace_static_b, trace_static_c, trace_static_d,
                                       trace_static_e, trace_static_f, trace_static_g, trace_static_h,
                                       trace_static_i};

void count_kinds(const Program &prog, int (&counts)[K_COUNT])
{
    for (int k = 0; k < K_COUNT; ++k) counts[k] = 0;
    for (int m = 0; m < prog.n_models; ++m) counts[prog.kind[m]] += 1;
}

}  // namespace

// LENSED_NO_BUILTIN=1 (tuning / tests): ignore the built-in signatures, so that a config's list goes
// through the run-time specialisation (jit.cu) and the two can be compared
static bool builtin_enabled()
{
    const char *env = getenv("LENSED_NO_BUILTIN");
    return !(env && env[0] == '1');
}

bool trace_has_static(const Program &prog)
{
    if (!builtin_enabled()) return false;
    int counts[K_COUNT];
    count_kinds(prog, counts);
    for (StaticTracer f : kStaticTracers)
        if (f(counts, prog, TraceArgs{}, 0, 0, nullptr, nullptr)) return true;
    return false;
}

cudaError_t launch_trace(const Program &prog, const TraceArgs &a, int R, int nvec, bool allow_static, const JitTracer *jit,
                         cudaStream_t st)
{
    if (allow_static && a.err == nullptr) {
        int counts[K_COUNT];
        count_kinds(prog, counts);
        cudaError_t err = cudaSuccess;
        if (builtin_enabled())
            for (StaticTracer f : kStaticTracers)
                if (f(counts, prog, a, R, nvec, st, &err)) return err;
        if (jit) return jit_launch(jit, prog, a, nvec, st);
    }
    const bool err = a.err != nullptr;
    switch (R) {
#define LENSED_CASE(NP)                                                                      \
    case 2 * NP:                                                                             \
        return err ? launch_trace_kernel(trace_kernel<NP, true>, prog, a, nvec, st)          \
                   : launch_trace_kernel(trace_kernel<NP, false>, prog, a, nvec, st);
        LENSED_CASE(1)
        LENSED_CASE(2)
        LENSED_CASE(3)
        LENSED_CASE(4)
        LENSED_CASE(5)
#undef LENSED_CASE
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace lensed
