// trace.cu -- steps a1-a4: ray generation, deflection summed over lenses, surface
// brightness, pixel quadrature, fused; one launch covers (pixel chunk) x (parameter vector).
//
//   x_k = pixel centre + (xi_k, eta_k)                       PAPER.md:155-159 eq. 14
//   y_k = x_k - sum_lenses alpha(x_k)                        PAPER.md:53-57  eq. 1
//   I   = sum_src I_S(y_k) + sum_fg I_L(x_k) + sky           PAPER.md:59-63  eq. 2
//   L_i = sum_k w_k I                                        PAPER.md:155-157 eq. 14
//
// Layout.  blockIdx.y = parameter vector, blockIdx.x = chunk of the traced-pixel list.  The
// vector's derived constants (prep.cu) and the rule sit in shared memory and are read with
// broadcast LDS.128.  A thread owns one pixel at a time and carries R rays (rule points) in
// registers through the model list, so the constants of a model are loaded once per R rays
// and the R evaluations give the instruction-level parallelism that hides the MUFU latency.
// No per-ray value ever goes to memory; one float per traced pixel is written.
//
// Arithmetic is FP32 on the FMA pipe with MUFU rsqrt / rcp / lg2 / ex2.  Offsets are formed
// relative to each component's centre in pixel units (see lensed_internal.h).
#include "lensed_internal.h"

namespace lensed {
namespace {

constexpr int kThreads = 256;
constexpr int kPixPerThread = 4;
constexpr int kPixPerBlock = kThreads * kPixPerThread;

__device__ __forceinline__ float mufu_rsq(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_rcp(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_lg2(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_ex2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// atan(z)/z for any z >= 0: minimax polynomial in z^2 on [0, 1] (relative error 1.5e-8),
// atan(z) = pi/2 - atan(1/z) above.  Even in z, equal to 1 at z = 0: no 0/0 anywhere.
__device__ __forceinline__ float atanc_pos(float z)
{
    const bool big = z > 1.0f;
    const float iz = mufu_rcp(fmaxf(z, 1.0f));   // = 1/z when big, 1 otherwise
    const float a = big ? iz : z;
    const float t = a * a;
    float p = 2.8498720241e-03f;
    p = fmaf(p, t, -1.6068558782e-02f);
    p = fmaf(p, t, 4.2691405628e-02f);
    p = fmaf(p, t, -7.5042849627e-02f);
    p = fmaf(p, t, 1.0640929559e-01f);
    p = fmaf(p, t, -1.4203643337e-01f);
    p = fmaf(p, t, 1.9992619252e-01f);
    p = fmaf(p, t, -3.3333073338e-01f);
    p = fmaf(p, t, 9.9999998477e-01f);
    // big: atan(z)/z = (pi/2 - a p(a^2)) / z = iz (pi/2 - iz p)
    const float hi = iz * fmaf(-iz, p, 1.5707963267948966f);
    return big ? hi : p;
}

// atanh(z)/z for 0 <= z < 0.4 as a polynomial in z^2 (relative error 2.8e-8); above that
// the SIE uses (1/2) ln((1+z)/(1-z)) directly, where the logarithm is >= 0.85 and the
// absolute error of MUFU.LG2 is harmless.
__device__ __forceinline__ float atanhc_small(float t)
{
    float p = 1.5752566048e-01f;
    p = fmaf(p, t, 1.3583491165e-01f);
    p = fmaf(p, t, 2.0041753926e-01f);
    p = fmaf(p, t, 3.3332476991e-01f);
    p = fmaf(p, t, 1.0000000279e+00f);
    return p;
}
__device__ __forceinline__ float atanh_large(float z)   // 0.4 <= z < 1
{
    const float zc = fminf(z, 0.99999994f);
    return mufu_lg2((1.0f + zc) * mufu_rcp(1.0f - zc)) * (0.5f * 0.6931471805599453f);
}

template <int R>
struct Rays {
    float xi[R], eta[R], w[R];
    float ax[R], ay[R];   // summed deflection, pixels
    float I[R];
};

template <int R>
__device__ __forceinline__ void lens_sis(const float4 *d, float jf, float rf, Rays<R> &r)
{
    const float4 c0 = d[0], c1 = d[1];
    const float dx0 = (jf - c0.x) - c0.y, dy0 = (rf - c0.z) - c0.w;
#pragma unroll
    for (int k = 0; k < R; ++k) {
        const float u = dx0 + r.xi[k], v = dy0 + r.eta[k];
        const float r2 = fmaf(u, u, v * v);
        const float s = r2 > 0.0f ? c1.x * mufu_rsq(r2) : 0.0f;     // alpha = b (u, v) / r, 0 at r = 0
        r.ax[k] = fmaf(s, u, r.ax[k]);
        r.ay[k] = fmaf(s, v, r.ay[k]);
    }
}

template <int R>
__device__ __forceinline__ void lens_point(const float4 *d, float jf, float rf, Rays<R> &r)
{
    const float4 c0 = d[0], c1 = d[1];
    const float dx0 = (jf - c0.x) - c0.y, dy0 = (rf - c0.z) - c0.w;
#pragma unroll
    for (int k = 0; k < R; ++k) {
        const float u = dx0 + r.xi[k], v = dy0 + r.eta[k];
        const float r2 = fmaf(u, u, v * v);
        const float s = r2 > 0.0f ? c1.x * mufu_rcp(r2) : 0.0f;     // alpha = thetaE^2 (u, v) / r^2
        r.ax[k] = fmaf(s, u, r.ax[k]);
        r.ay[k] = fmaf(s, v, r.ay[k]);
    }
}

template <int R>
__device__ __forceinline__ void lens_shear(const float4 *d, float jf, float rf, float cxh, float cyh, Rays<R> &r)
{
    const float4 c0 = d[0];
    const float x0 = jf - cxh, y0 = rf - cyh;                        // about the image centre (R4)
#pragma unroll
    for (int k = 0; k < R; ++k) {
        const float x = x0 + r.xi[k], y = y0 + r.eta[k];
        r.ax[k] += fmaf(c0.x, x, c0.y * y);                          // g1 x + g2 y
        r.ay[k] += fmaf(c0.y, x, -c0.x * y);                         // g2 x - g1 y
    }
}

// SIE (Kormann et al. 1994; R2):  alpha_u = A atan(q' u/psi), alpha_v = A atanh(q' v/psi),
// A = b sqrt(q)/q', psi = sqrt(q^2 u^2 + v^2), (u, v) in the lens frame (major axis along u).
// Evaluated as b sqrt(q) (u/psi) atanc(q' u/psi) and, for small q' v/psi, as
// b sqrt(q) (v/psi) atanhc(q' v/psi), so that q -> 1 (q' -> 0, A -> inf) needs no special
// case; the atanh branch with A is only selected where q' |v|/psi >= 0.4, i.e. q' >= 0.4.
template <int R>
__device__ __forceinline__ void lens_sie(const float4 *d, float jf, float rf, Rays<R> &r)
{
    const float4 c0 = d[0], c1 = d[1], c2 = d[2];
    const float dx0 = (jf - c0.x) - c0.y, dy0 = (rf - c0.z) - c0.w;
    const float cs = c1.x, sn = c1.y, q2 = c1.z, qp = c1.w, bq = c2.x, A = c2.y;
#pragma unroll
    for (int k = 0; k < R; ++k) {
        const float dx = dx0 + r.xi[k], dy = dy0 + r.eta[k];
        const float u = fmaf(cs, dx, sn * dy), v = fmaf(cs, dy, -sn * dx);
        const float psi2 = fmaf(q2 * u, u, v * v);
        const float ipsi = psi2 > 0.0f ? mufu_rsq(psi2) : 0.0f;
        const float wu = u * ipsi, wv = v * ipsi;
        const float au = bq * wu * atanc_pos(fabsf(qp * wu));
        const float zv = qp * wv, tv = zv * zv;
        const float av_small = bq * wv * atanhc_small(tv);
        const float av_large = copysignf(A * atanh_large(fabsf(zv)), wv);
        const float av = tv < 0.16f ? av_small : av_large;
        r.ax[k] += fmaf(cs, au, -sn * av);
        r.ay[k] += fmaf(sn, au, cs * av);
    }
}

// Sersic, eqs. 22-23:  I = I0 exp(-b_n (R/r_S)^(1/n))
//   = 2^(log2 I0 - (b_n log2 e) 2^(lg2((R/r_S)^2) / (2n))).   R = 0 gives lg2 = -inf, 2^-inf = 0, I = I0.
template <int R, bool SRC>
__device__ __forceinline__ void light_sersic(const float4 *d, float jf, float rf, Rays<R> &r)
{
    const float4 c0 = d[0], c1 = d[1], c2 = d[2];
    const float dx0 = (jf - c0.x) - c0.y, dy0 = (rf - c0.z) - c0.w;
#pragma unroll
    for (int k = 0; k < R; ++k) {
        float dx = dx0 + r.xi[k], dy = dy0 + r.eta[k];
        if (SRC) { dx -= r.ax[k]; dy -= r.ay[k]; }
        const float u = fmaf(c1.x, dx, c1.y * dy), v = fmaf(c1.z, dx, c1.w * dy);
        const float r2 = fmaf(u, u, v * v);
        const float e = mufu_ex2(c2.z * mufu_lg2(r2));
        r.I[k] += mufu_ex2(fmaf(-c2.y, e, c2.x));
    }
}

// Gaussian (R7):  I = I0 exp(-R^2 / (2 sigma^2)) = 2^(log2 I0 - (log2 e / 2) (R/sigma)^2)
template <int R, bool SRC>
__device__ __forceinline__ void light_gauss(const float4 *d, float jf, float rf, Rays<R> &r)
{
    const float4 c0 = d[0], c1 = d[1], c2 = d[2];
    const float dx0 = (jf - c0.x) - c0.y, dy0 = (rf - c0.z) - c0.w;
#pragma unroll
    for (int k = 0; k < R; ++k) {
        float dx = dx0 + r.xi[k], dy = dy0 + r.eta[k];
        if (SRC) { dx -= r.ax[k]; dy -= r.ay[k]; }
        const float u = fmaf(c1.x, dx, c1.y * dy), v = fmaf(c1.z, dx, c1.w * dy);
        const float r2 = fmaf(u, u, v * v);
        r.I[k] += mufu_ex2(fmaf(-c2.y, r2, c2.x));
    }
}

template <int R>
__global__ void __launch_bounds__(kThreads, 2) trace_kernel(Program prog, TraceArgs a)
{
    extern __shared__ float4 smem4[];
    float4 *sder = smem4;                         // [D/4]
    float4 *squad = smem4 + prog.D / 4;           // [nq_pad]
    const int bvec = blockIdx.y;
    {
        const float4 *g = reinterpret_cast<const float4 *>(a.derived + (size_t)bvec * prog.D);
        for (int i = threadIdx.x; i < prog.D / 4; i += kThreads) sder[i] = g[i];
        for (int i = threadIdx.x; i < a.nq_pad; i += kThreads) squad[i] = a.quad[i];
    }
    __syncthreads();
    if (sder[0].x == 0.0f) return;                // vector outside the model domain: skipped
    float *Lb = a.L + (size_t)bvec * a.l_stride;

    const int base = blockIdx.x * kPixPerBlock;
#pragma unroll 1
    for (int it = 0; it < kPixPerThread; ++it) {
        const int ip = base + it * kThreads + threadIdx.x;
        if (ip >= a.npix) break;
        const uint32_t rc = a.pix[ip];
        const int row = (int)(rc >> 16), col = (int)(rc & 0xffffu);
        const float jf = (float)col, rf = (float)row;
        float acc = 0.0f;
#pragma unroll 1
        for (int q0 = 0; q0 < a.nq_pad; q0 += R) {
            Rays<R> r;
#pragma unroll
            for (int k = 0; k < R; ++k) {
                const float4 qk = squad[q0 + k];
                r.xi[k] = qk.x; r.eta[k] = qk.y; r.w[k] = qk.z;
                r.ax[k] = 0.0f; r.ay[k] = 0.0f; r.I[k] = 0.0f;
            }
#pragma unroll 1
            for (int m = 0; m < prog.n_lens; ++m) {
                const float4 *d = sder + (prog.lens_off[m] >> 2);
                switch (prog.lens_kind[m]) {
                case K_SIE:   lens_sie<R>(d, jf, rf, r); break;
                case K_SIS:   lens_sis<R>(d, jf, rf, r); break;
                case K_POINT: lens_point<R>(d, jf, rf, r); break;
                default:      lens_shear<R>(d, jf, rf, a.cxh, a.cyh, r); break;
                }
            }
#pragma unroll 1
            for (int m = 0; m < prog.n_light; ++m) {
                const float4 *d = sder + (prog.light_off[m] >> 2);
                switch (prog.light_kind[m]) {
                case K_SRC_SERSIC: light_sersic<R, true>(d, jf, rf, r); break;
                case K_FG_SERSIC:  light_sersic<R, false>(d, jf, rf, r); break;
                case K_SRC_GAUSS:  light_gauss<R, true>(d, jf, rf, r); break;
                case K_FG_GAUSS:   light_gauss<R, false>(d, jf, rf, r); break;
                default: {
                    const float lvl = d[0].x;
#pragma unroll
                    for (int k = 0; k < R; ++k) r.I[k] += lvl;
                    break;
                }
                }
            }
#pragma unroll
            for (int k = 0; k < R; ++k) acc = fmaf(r.w[k], r.I[k], acc);
        }
        Lb[row * a.W + col] = acc;
    }
}

template <int R>
cudaError_t launch_trace_R(const Program &prog, const TraceArgs &a, int nvec, cudaStream_t st)
{
    const size_t smem = (size_t)(prog.D / 4 + a.nq_pad) * sizeof(float4);
    dim3 grid((a.npix + kPixPerBlock - 1) / kPixPerBlock, nvec);
    trace_kernel<R><<<grid, kThreads, smem, st>>>(prog, a);
    return cudaGetLastError();
}

}  // namespace

// Rays carried per thread, R in 1..9: least padded rule length, weighted by a per-block
// overhead that shrinks with R (4 -> 4, 9 -> 9, 16 -> 8, 25 -> 5, 49 -> 7, 121 -> 9, 225 -> 9).
int trace_pick_R(int n_quad)
{
    int best = 1;
    double best_cost = 1e300;
    for (int R = 1; R <= 9; ++R) {
        const int pad = (n_quad + R - 1) / R * R;
        const double cost = pad * (1.0 + 0.6 / R);
        if (cost < best_cost - 1e-12) { best = R; best_cost = cost; }
    }
    return best;
}

cudaError_t launch_trace(const Program &prog, const TraceArgs &a, int R, int nvec, cudaStream_t st)
{
    switch (R) {
    case 1: return launch_trace_R<1>(prog, a, nvec, st);
    case 2: return launch_trace_R<2>(prog, a, nvec, st);
    case 3: return launch_trace_R<3>(prog, a, nvec, st);
    case 4: return launch_trace_R<4>(prog, a, nvec, st);
    case 5: return launch_trace_R<5>(prog, a, nvec, st);
    case 6: return launch_trace_R<6>(prog, a, nvec, st);
    case 7: return launch_trace_R<7>(prog, a, nvec, st);
    case 8: return launch_trace_R<8>(prog, a, nvec, st);
    case 9: return launch_trace_R<9>(prog, a, nvec, st);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace lensed
