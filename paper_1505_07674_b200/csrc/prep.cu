// prep.cu -- step a0: parameter vectors xi -> kernel-ready constants, in FP64 on the device.
//
// One thread per (parameter vector, model).  Everything the ray tracer would otherwise recompute
// per ray is evaluated once here, in double, and rounded to FP32 once:
//   * component centres as (integer pixel, fraction)
//   * SIE: cos/sin PA, q^2, q' = sqrt(1-q^2), A = b sqrt(q)/q' folded into the rotation
//     back to the image frame                                  (R2)
//   * Sersic: b_n from P(2n, b_n) = 1/2 (r_S is the half-light radius; R5),
//     log2 I_0 from the total magnitude (R6), the rotated, q-stretched,
//     r_S-scaled frame of eq. 23
//   * the domain check: outside it the vector is flagged invalid;
//   * an unrounded FP64 copy of the same constants and, per source Sersic, the squared radius
//     inside which its pixels are re-traced in FP64 (refine.cu).
#include "lensed_internal.h"
#include <math.h>

namespace lensed {
namespace {

constexpr double kPi = 3.141592653589793238462643383279502884;
constexpr double kLn2 = 0.693147180559945309417232121458176568;
constexpr double kLn10 = 2.302585092994045684017991454684364208;

// Regularised lower incomplete gamma P(a, x) by its power series
//   P = x^a e^-x / Gamma(a+1) * (1 + x/(a+1) + x^2/((a+1)(a+2)) + ...),
// which converges for every x > 0; near the root of P(2n, x) = 1/2 (x ~ 2n - 1/3 < a + 1)
// the terms decrease from the start.  Returns ln P.
__device__ double log_gamma_p_series(double a, double x, double lgam_a1)
{
    double term = 1.0, sum = 1.0;
    for (int k = 1; k < 4000; ++k) {
        term *= x / (a + k);
        sum += term;
        if (term < sum * 1e-17) break;
    }
    return a * log(x) - x - lgam_a1 + log(sum);
}

// b_n: Newton iteration in t = ln b on g(t) = ln P(2n, e^t) - ln(1/2).  ln P is close to
// linear in t for small b (P ~ b^a / Gamma(a+1)), so the iteration also converges quickly
// for n << 1 where Newton in b itself crawls.  Start: Ciotti & Bertin's asymptotic series
// for n >= 0.36, the small-b solution (Gamma(a+1)/2)^(1/a) below.
__device__ double sersic_bn(double n)
{
    const double a = 2.0 * n;
    const double lgam_a1 = lgamma(a + 1.0);
    double t;
    if (n >= 0.36)
        t = log(a - 1.0 / 3.0 + 4.0 / (405.0 * n) + 46.0 / (25515.0 * n * n));
    else
        t = (lgam_a1 - kLn2) / a;
    for (int it = 0; it < 60; ++it) {
        const double b = exp(t);
        const double lp = log_gamma_p_series(a, b, lgam_a1);
        // d ln P / dt = b * P'(b) / P,   b P'(b) = b^a e^-b / Gamma(a)
        const double lden = a * t - b - (lgam_a1 - log(a));
        const double dt = (lp + kLn2) * exp(lp - lden);
        t -= dt;
        // quadratic convergence: a step below 1e-9 leaves an error below 1e-17, so the check that
        // would only confirm it (one more evaluation of the series) is not made
        if (fabs(dt) < 1e-9 * fmax(1.0, fabs(t))) break;
    }
    return exp(t);
}

__device__ inline void put_centre(float *d, double x_arcsec, double y_arcsec, const PrepArgs &a)
{
    const double cx = x_arcsec / a.scale + a.cxh, cy = y_arcsec / a.scale + a.cyh;
    const double ix = rint(cx), iy = rint(cy);
    d[0] = (float)ix; d[1] = (float)(cx - ix);
    d[2] = (float)iy; d[3] = (float)(cy - iy);
}

// frame of eq. 23 scaled by 1/len: (u', v') = (sqrt(q) u, v / sqrt(q)) / len
__device__ inline void put_frame(float *d, double pa_deg, double q, double len_px)
{
    double s, c;
    sincos(pa_deg * (kPi / 180.0), &s, &c);
    const double sq = sqrt(q);
    d[0] = (float)(c * sq / len_px);
    d[1] = (float)(s * sq / len_px);
    d[2] = (float)(-s / (sq * len_px));
    d[3] = (float)(c / (sq * len_px));
}

// FP64 copy of a model's constants for the refinement pass (refine.cu), lengths in pixels
__device__ inline void put64(double *e, double a0 = 0, double a1 = 0, double a2 = 0, double a3 = 0, double a4 = 0,
                             double a5 = 0, double a6 = 0, double a7 = 0, double a8 = 0)
{
    e[0] = a0; e[1] = a1; e[2] = a2; e[3] = a3; e[4] = a4; e[5] = a5; e[6] = a6; e[7] = a7; e[8] = a8;
}

constexpr int kPrepVec = 8;            // vectors per block; threadIdx.x = model slot (kMaxModels = 32)

// One thread per (vector, model): the b_n solves of a vector's Sersic components run side by
// side.  Per vector, shared memory collects validity, the SIE mode and the deflection scale.
__global__ void __launch_bounds__(kMaxModels * kPrepVec) prep_kernel(Program prog, PrepArgs a)
{
    __shared__ int s_valid[kPrepVec], s_mode[kPrepVec];
    __shared__ float s_defl[kPrepVec][kMaxModels];   // deflection scale of each lens, pixels
    const int m = threadIdx.x, lv = threadIdx.y;
    const int b = blockIdx.x * kPrepVec + lv;
    const bool active = b < a.B && m < prog.n_models;
    if (m == 0) { s_valid[lv] = 1; s_mode[lv] = 0; }
    s_defl[lv][m] = 0.0f;
    __syncthreads();

    float *d = nullptr;
    double *e = nullptr;
    int kind = -1;
    double p[7];
    bool valid = true;
    double sersic_c = 0.0, sersic_n = 0.0, sersic_b = 0.0;   // source Sersic: threshold constants (below)
    if (active) {
        kind = prog.kind[m];
        const float *pf = a.params + (size_t)b * prog.P + prog.par_off[m];
        d = a.derived + (size_t)b * prog.D + prog.der_off[m];
        e = a.derived64 + ((size_t)b * prog.n_models + m) * kD64PerModel;
        const int np = kind_num_params(kind), nd = kind_num_derived(kind);
        for (int i = 0; i < nd; ++i) d[i] = 0.0f;
        put64(e);
        for (int i = 0; i < np; ++i) {
            p[i] = (double)pf[i];
            if (!isfinite(p[i])) valid = false;
        }
    }
    if (active && valid) {
        switch (kind) {
        case K_SIS:
            valid = p[2] >= 0.0;
            put_centre(d, p[0], p[1], a);
            d[4] = (float)(p[2] / a.scale);
            put64(e, p[0] / a.scale + a.cxh, p[1] / a.scale + a.cyh, p[2] / a.scale);
            s_defl[lv][m] = (float)(p[2] / a.scale);
            break;
        case K_POINT:
            valid = p[2] >= 0.0;
            put_centre(d, p[0], p[1], a);
            d[4] = (float)((p[2] / a.scale) * (p[2] / a.scale));
            put64(e, p[0] / a.scale + a.cxh, p[1] / a.scale + a.cyh, (p[2] / a.scale) * (p[2] / a.scale));
            s_defl[lv][m] = (float)(p[2] / a.scale);
            break;
        case K_SHEAR:
            d[0] = (float)p[0]; d[1] = (float)p[1];
            put64(e, p[0], p[1]);
            s_defl[lv][m] = (float)(sqrt(p[0] * p[0] + p[1] * p[1]) * sqrt(a.cxh * a.cxh + a.cyh * a.cyh));
            break;
        case K_SIE: {
            const double q = p[3];
            valid = p[2] >= 0.0 && q > 0.0 && q <= 1.0;
            if (!valid) break;
            put_centre(d, p[0], p[1], a);
            atomicMax(&s_mode[lv], sie_mode(q));
            double s, c;
            sincos(p[4] * (kPi / 180.0), &s, &c);
            d[4] = (float)c; d[5] = (float)s;
            d[6] = (float)(q * q);
            // q' floored: A atan(q' u/psi) -> b sqrt(q) u/psi as q' -> 0 with relative
            // deviation q'^2/3, so the floor changes nothing above 3e-9 and A stays finite
            const double qp = fmax(sqrt((1.0 - q) * (1.0 + q)), 1e-4);
            const double A = p[2] / a.scale * sqrt(q) / qp;
            d[7] = (float)qp;
            d[8] = (float)(c * A); d[9] = (float)(s * A);
            d[10] = (float)(c * A * (0.5 * kLn2)); d[11] = (float)(-s * A * (0.5 * kLn2));
            put64(e, p[0] / a.scale + a.cxh, p[1] / a.scale + a.cyh, c, s, q, p[2] / a.scale);
            s_defl[lv][m] = (float)(p[2] / a.scale);
            break;
        }
        case K_SRC_SERSIC: case K_FG_SERSIC: {
            const double rs = p[2] / a.scale, mag = p[3], n = p[4], q = p[5];
            valid = p[2] > 0.0 && n >= 0.02 && n <= 20.0 && q > 0.0 && q <= 1.0;
            if (!valid) break;
            put_centre(d, p[0], p[1], a);
            put_frame(d + 4, p[6], q, rs);
            const double bn = sersic_bn(n);
            // I_0 = F b_n^(2n) / (2 pi n r_S^2 Gamma(2n)), r_S in pixels (R6)
            const double ln_i0 = -0.4 * (mag - a.zp) * kLn10 + 2.0 * n * log(bn) - lgamma(2.0 * n)
                                 - log(2.0 * kPi * n * rs * rs);
            d[8] = (float)(ln_i0 / kLn2);
            d[9] = (float)(bn / kLn2);
            d[10] = (float)(0.5 / n);
            double s, c;
            sincos(p[6] * (kPi / 180.0), &s, &c);
            put64(e, p[0] / a.scale + a.cxh, p[1] / a.scale + a.cyh, c, s, q, rs, 1.0 / n, bn, ln_i0);
            if (kind == K_SRC_SERSIC && n > 1.0) { sersic_c = n * sqrt(q) * rs / bn; sersic_n = n; sersic_b = bn; }
            // Foreground expansion (trace_static.cuh): the pixel integral of exp(h(s)), s = (R/r_S)^2,
            // from its Taylor expansion to fourth order in the rule offsets is accurate to
            // 0.016 tau^6 (measured over n in [0.5, 8], q in [0.2, 1], r_S in [2, 60] px for the sub4,
            // Gauss-Legendre and Gauss-Kronrod rules) with
            //   tau = max((b_n/n) R'^(1/n), 1) eta / R',   eta = rule radius / (sqrt(q) r_S),
            // the offset of the farthest rule point in units of the pixel's scaled radius R', times
            // the logarithmic slope of the profile.  tau <= fgx_tau gives R' >= eta / fgx_tau and
            // (b_n/n) R'^(1/n - 1) <= fgx_tau / eta: a lower bound for n > 1, an upper one for n < 1.
            // Second-order terms alone are accurate to 0.04 tau^4, i.e. the same 2e-7 for tau <= fgx_tau / 3:
            // d[12..13] = range of the fourth-order form, d[14..15] = of the second-order form.
            d[12] = 3e38f; d[13] = 0.0f; d[14] = 3e38f; d[15] = 0.0f;      // empty ranges: per-ray sum
            if (kind == K_FG_SERSIC && a.fgx_tau > 0.0) {
                const double eta = a.rule_radius / (sqrt(q) * rs);
                for (int tier = 0; tier < 2; ++tier) {
                    const double t = tier ? a.fgx_tau / 3.0 : a.fgx_tau;
                    double r_lo = eta / t, r_hi = 1e18;
                    const double g = bn / n * eta / t;                     // needs g R'^(1/n - 1) <= 1
                    if (n > 1.0 + 1e-6) r_lo = fmax(r_lo, pow(g, n / (n - 1.0)));
                    else if (n < 1.0 - 1e-6) r_hi = pow(g, -n / (1.0 - n));
                    else if (g > 1.0) r_hi = 0.0;
                    if (r_hi > r_lo) {
                        d[12 + 2 * tier] = (float)fmin(r_lo * r_lo * (1.0 + 1e-6), 3e38);
                        d[13 + 2 * tier] = (float)fmin(r_hi * r_hi * (1.0 - 1e-6), 3e38);
                    }
                }
            }
            break;
        }
        case K_SRC_GAUSS: case K_FG_GAUSS: {
            const double sg = p[2] / a.scale, mag = p[3], q = p[4];
            valid = p[2] > 0.0 && q > 0.0 && q <= 1.0;
            if (!valid) break;
            put_centre(d, p[0], p[1], a);
            put_frame(d + 4, p[5], q, sg);
            const double ln_i0 = -0.4 * (mag - a.zp) * kLn10 - log(2.0 * kPi * sg * sg);
            d[8] = (float)(ln_i0 / kLn2);
            d[9] = (float)(0.5 / kLn2);
            double s, c;
            sincos(p[5] * (kPi / 180.0), &s, &c);
            put64(e, p[0] / a.scale + a.cxh, p[1] / a.scale + a.cyh, c, s, q, sg, ln_i0);
            break;
        }
        case K_SKY:
            d[0] = (float)p[0];
            put64(e, p[0]);
            break;
        default:
            valid = false;
        }
    }
    if (active && !valid) atomicAnd(&s_valid[lv], 0);
    __syncthreads();
    if (!active) return;
    // Refinement threshold of a source Sersic with n > 1 (refine.cu; DESIGN.md "FP32 and the
    // cusp"): a ray position carries ~eps |alpha| of FP32 rounding noise, and the profile turns a
    // displacement dx (pixels) into  d ln I = (b_n/n) R'^(1/n-1) / (sqrt(q) r_S) dx  at most,
    // R' = R/r_S.  Pixels with a ray where that slope exceeds G = 200 / max(deflection scale, 25 px)
    // per pixel are re-traced in FP64:  R'^2 < T2 = (G n sqrt(q) r_S / b_n)^(-2n/(n-1)).
    if (sersic_c > 0.0 && s_valid[lv]) {
        float defl = 0.0f;
        for (int i = 0; i < prog.n_models; ++i) defl += s_defl[lv][i];     // list order: deterministic
        const double G = a.refine_gain * 200.0 / fmax((double)defl, 25.0);
        const double cc = G * sersic_c;
        // ... and never beyond the scaled radius where the profile has fallen to exp(-24) of its centre,
        // b_n R'^(1/n) = 24: just above n = 1 the exponent runs away, and with cc < 1 (a compact source,
        // r_S below ~0.3 px) T2 would reach the clamp and EVERY traced pixel of the vector be re-traced in
        // FP64 -- one such prior draw then dominates the step.  Out there the component is below FP32
        // resolution of its own peak, so its rounding noise cannot be seen in any pixel that counts.
        const double cap = pow(24.0 / sersic_b, 2.0 * sersic_n);
        d[11] = (float)fmin(fmin(pow(cc, -2.0 * sersic_n / (sersic_n - 1.0)), cap), 1e30);
    }
    if (m == 0) {
        float *der = a.derived + (size_t)b * prog.D;
        der[0] = s_valid[lv] ? 1.0f : 0.0f;
        der[1] = (float)s_mode[lv];
        der[2] = 0.0f; der[3] = 0.0f;
    }
}


// Block order of the ray tracer: the vectors of each batch chunk sorted by (SIE mode, index),
// vectors outside the model domain last.  The specialised tracers hold one straight-line copy of
// the ray loop per mode (trace_static.cuh); with the vectors of a launch in arbitrary order the
// blocks resident at one time run all six copies and miss the instruction cache (HST config:
// `no_instruction` 2.8 stall cycles per issue, profiles/r2b.md).  Stable counting sort, one block
// per chunk: the order is a function of the inputs.  It only changes which block works on which
// vector -- every vector's result is what it was.
constexpr int kOrderKeys = 7;                   // SIE modes 0..5, 6 = invalid
__global__ void __launch_bounds__(256) order_kernel(const float *derived, int D, int B, int Bc, int *order)
{
    __shared__ int s_run[kOrderKeys + 1];       // next free slot per key
    __shared__ int s_warp[8][kOrderKeys];       // per warp, per key: count within the current tile
    const int b0 = blockIdx.x * Bc, n = min(Bc, B - b0);
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    auto key_of = [&](int i) {
        const float *hdr = derived + (size_t)(b0 + i) * D;
        return hdr[0] != 0.0f ? min(max((int)hdr[1], 0), kOrderKeys - 2) : kOrderKeys - 1;
    };
    if (t <= kOrderKeys) s_run[t] = 0;
    __syncthreads();
    for (int i = t; i < n; i += 256) atomicAdd(&s_run[key_of(i) + 1], 1);      // totals (integers: order-free)
    __syncthreads();
    if (t == 0)
        for (int k = 1; k <= kOrderKeys; ++k) s_run[k] += s_run[k - 1];        // s_run[k] = first slot of key k
    __syncthreads();
    for (int base = 0; base < n; base += 256) {
        const int i = base + t;
        const int key = i < n ? key_of(i) : kOrderKeys;
        int rank = 0;
#pragma unroll
        for (int k = 0; k < kOrderKeys; ++k) {
            const unsigned m = __ballot_sync(0xffffffffu, key == k);
            if (key == k) rank = __popc(m & ((1u << lane) - 1u));
            if (lane == 0) s_warp[warp][k] = __popc(m);
        }
        __syncthreads();
        if (key < kOrderKeys) {
            int off = s_run[key] + rank;
            for (int w = 0; w < warp; ++w) off += s_warp[w][key];
            order[b0 + off] = i;
        }
        __syncthreads();
        if (t < kOrderKeys) {
            int c = 0;
            for (int w = 0; w < 8; ++w) c += s_warp[w][t];
            s_run[t] += c;
        }
        __syncthreads();
    }
}

}  // namespace

cudaError_t launch_prep(const Program &prog, const PrepArgs &a, cudaStream_t st)
{
    const dim3 block(kMaxModels, kPrepVec);
    prep_kernel<<<(a.B + kPrepVec - 1) / kPrepVec, block, 0, st>>>(prog, a);
    return cudaGetLastError();
}

cudaError_t launch_order(const float *derived, int D, int B, int Bc, int *order, cudaStream_t st)
{
    order_kernel<<<(B + Bc - 1) / Bc, 256, 0, st>>>(derived, D, B, Bc, order);
    return cudaGetLastError();
}

}  // namespace lensed
