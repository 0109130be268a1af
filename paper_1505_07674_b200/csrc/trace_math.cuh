// trace_math.cuh -- per-model arithmetic of the ray tracer on packed FP32 pairs (f32x2.cuh).
//
//   y = x - sum_lenses alpha(x)                               PAPER.md:53-57  eq. 1
//   I = sum_src I_S(y) + sum_fg I_L(x) + sky                  PAPER.md:59-63  eq. 2
//   Sersic / elliptical radius                                PAPER.md:244-250 eqs. 22-23
//
// Every component works in its own linear frame (u, v) = M (x - c); a ray enters it as
//   (u, v) = (u0, v0) + table[k],   (u0, v0) = M (pixel - c) per pixel,  table = M (xi_k, eta_k)
// per (vector, rule point) in shared memory (trace.cu).  Arithmetic: FFMA2 / FMUL2 / FADD2 on
// the FMA pipe, MUFU rsqrt / rcp / lg2 / ex2 on the XU pipe.  The SIE's atan and atanh are
// polynomials whose degree is picked per parameter vector from its axis ratio (SieMode), so
// that for q >= 1/2 the only MUFU of the lens is the rsqrt of psi^2.
#pragma once
#include "lensed_internal.h"
#include "f32x2.cuh"

namespace lensed {

__device__ __forceinline__ float mufu_rsq(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_rcp(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_lg2(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_ex2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float min3(float a, float b, float c) { float y; asm("min.f32 %0, %1, %2, %3;" : "=f"(y) : "f"(a), "f"(b), "f"(c)); return y; }   // FMNMX3

constexpr float kTiny = 1e-30f;            // floor of squared radii: rsqrt / rcp stay finite, 0 * finite = 0
constexpr float kHalfPi = 1.5707963267948966f;

template <int NP>
struct Rays {
    f2 ax[NP], ay[NP];   // summed deflection, pixels
    f2 I[NP];            // summed brightness
};

// NP consecutive pairs of one table row
template <int NP>
__device__ __forceinline__ void load_pairs(const float *row, f2 (&out)[NP])
{
    if constexpr (NP % 2 == 0) {
#pragma unroll
        for (int i = 0; i < NP; i += 2) {
            const float4 t = *reinterpret_cast<const float4 *>(row + 2 * i);
            out[i] = mk2(t.x, t.y);
            out[i + 1] = mk2(t.z, t.w);
        }
    } else {
#pragma unroll
        for (int i = 0; i < NP; ++i) {
            const float2 t = *reinterpret_cast<const float2 *>(row + 2 * i);
            out[i] = mk2(t.x, t.y);
        }
    }
}

// NP consecutive scalars of one table row (16-byte aligned start)
template <int NP>
__device__ __forceinline__ void load_scalars(const float *row, float (&out)[NP])
{
    static_assert(NP <= 8, "at most eight points per pass");
    const float4 t = *reinterpret_cast<const float4 *>(row);
    const float v[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
    for (int i = 0; i < NP && i < 4; ++i) out[i] = v[i];
    if constexpr (NP > 4) {
        const float4 t2 = *reinterpret_cast<const float4 *>(row + 4);
        const float v2[4] = {t2.x, t2.y, t2.z, t2.w};
#pragma unroll
        for (int i = 4; i < NP; ++i) out[i] = v2[i - 4];
    }
}

// Two ways to fill a packed pair, chosen by the type of the frame origin:
//   float origin  "ray pairs":   the pair = two consecutive rule points of ONE pixel
//                 (interpreting tracer): table entries come as pairs, the origin is broadcast;
//   f2 origin     "pixel pairs": the pair = the SAME rule point of TWO pixels (specialised
//                 tracers): the table entry is broadcast, the origins come as a pair.  No rule is
//                 padded to an even length, per-pixel arithmetic is packed too, and a table row is
//                 read once for both pixels.
template <int NP>
__device__ __forceinline__ void enter(const float *row, float origin, f2 (&out)[NP])
{
    f2 p[NP];
    load_pairs<NP>(row, p);
#pragma unroll
    for (int k = 0; k < NP; ++k) out[k] = add2(p[k], bc(origin));
}
template <int NP>
__device__ __forceinline__ void enter(const float *row, f2 origin, f2 (&out)[NP])
{
    float t[NP];
    load_scalars<NP>(row, t);
#pragma unroll
    for (int k = 0; k < NP; ++k) out[k] = add2(bc(t[k]), origin);
}
// rule weights of a pass, as the multiplicand of the pixel sum
template <int NP>
__device__ __forceinline__ void pass_weights(const float *row, float, f2 (&out)[NP]) { load_pairs<NP>(row, out); }
template <int NP>
__device__ __forceinline__ void pass_weights(const float *row, f2, f2 (&out)[NP])
{
    float t[NP];
    load_scalars<NP>(row, t);
#pragma unroll
    for (int k = 0; k < NP; ++k) out[k] = bc(t[k]);
}
// running minimum of a squared radius: per pixel
__device__ __forceinline__ void min_radius(float &rmin, f2 r2) { rmin = min3(rmin, lo2(r2), hi2(r2)); }
__device__ __forceinline__ void min_radius(float2 &rmin, f2 r2) { rmin.x = fminf(rmin.x, lo2(r2)); rmin.y = fminf(rmin.y, hi2(r2)); }

// ---- minimax tables (gen_poly.py beside this file prints them with their errors) ---------
// atan(z)/z and (2/ln 2) atanh(z)/z in t = z^2 on [0, T]; highest degree first.  The tables
// marked "in s" are monomials in s = (2/T) t - 1: FP32 Horner in t itself loses up to 1e-5
// to cancellation for T >~ 1.  Relative error, fit / FP32 Horner:
//   kAtan019  T = 4/21  deg  4 in t   2.9e-8 / 1.0e-7      kAtanh016  T = 0.16  deg  4 in t   2.8e-8 / 1.2e-7
//   kAtan056  T = 9/16  deg  6 in t   3.0e-8 / 1.1e-7      kAtanh036  T = 0.36  deg  6 in t   2.6e-8 / 1.2e-7
//   kAtan1    T = 1     deg  8 in t   1.5e-8 / 0.9e-7      kAtanh050  T = 0.50  deg  8 in t   1.3e-8 / 0.9e-7
//   kAtan2    T = 2     deg 10 in s   5.5e-8 / 1.4e-7      kAtanh067  T = 2/3   deg 10 in s   4.0e-8 / 1.5e-7
//   kAtan3    T = 3     deg 12 in s   6.1e-8 / 1.4e-7      kAtanh075  T = 0.75  deg 12 in s   4.1e-8 / 1.5e-7
__device__ constexpr float kAtan019[5] = {7.7191768884e-02f, -1.3767447193e-01f, 1.9966269114e-01f, -3.3332551885e-01f, 9.9999997081e-01f};
__device__ constexpr float kAtan056[7] = {1.8452358884e-02f, -5.8612542189e-02f, 1.0069710760e-01f, -1.4100846142e-01f, 1.9983821868e-01f, -3.3332792361e-01f, 9.9999997016e-01f};
__device__ constexpr float kAtan1[9] = {2.8498055468e-03f, -1.6068293304e-02f, 4.2690975050e-02f, -7.5042486123e-02f, 1.0640912567e-01f, -1.4203639026e-01f, 1.9992618715e-01f, -3.3333073313e-01f, 9.9999998476e-01f};
__device__ constexpr float kAtan2[11] = {9.1487060309e-05f, -1.8564391925e-04f, 1.5699309251e-04f, -3.9463378275e-04f, 1.1686782180e-03f, -2.7031232426e-03f, 6.4149697350e-03f, -1.6261596296e-02f, 4.4525141523e-02f, -1.4269952760e-01f, 7.8539815093e-01f};
__device__ constexpr float kAtan3[13] = {3.0422385513e-04f, -4.8443279783e-04f, -1.2014446101e-04f, 2.3235041340e-05f, 1.2300481067e-03f, -2.0805755083e-03f, 3.1809357122e-03f, -6.3178359761e-03f, 1.2922699920e-02f, -2.7101507477e-02f, 6.1303160862e-02f, -1.6173893999e-01f, 7.2347895789e-01f};
__device__ constexpr float kAtanh016[5] = {4.5452240586e-01f, 3.9193689016e-01f, 5.7828276164e-01f, 9.6177198571e-01f, 2.8853901623e+00f};
__device__ constexpr float kAtanh036[7] = {7.9859918538e-01f, -9.8292821592e-02f, 4.2027748616e-01f, 3.9866639322e-01f, 5.7793389114e-01f, 9.6177664003e-01f, 2.8853901580e+00f};
__device__ constexpr float kAtanh050[9] = {2.1876451735e+00f, -2.5781934840e+00f, 1.9242353758e+00f, -3.0531906864e-01f, 4.2784923043e-01f, 4.0105080738e-01f, 5.7765090270e-01f, 9.6178545527e-01f, 2.8853901179e+00f};
__device__ constexpr float kAtanh067[11] = {2.7909708512e-04f, 5.6547031726e-04f, 4.8361299614e-04f, 1.2329644873e-03f, 3.6610617060e-03f, 8.5636712306e-03f, 2.0668864871e-02f, 5.3606889406e-02f, 1.5204721478e-01f, 5.1862281330e-01f, 3.2908421537e+00f};
__device__ constexpr float kAtanh075[13] = {9.3871416073e-04f, 1.4826418351e-03f, -3.7924017826e-04f, -2.8540519880e-05f, 3.8816269518e-03f, 6.5758985577e-03f, 1.0253188210e-02f, 2.0702484489e-02f, 4.3176660471e-02f, 9.3234500434e-02f, 2.2056315283e-01f, 6.2923262188e-01f, 3.3581557041e+00f};

// z * P(z^2) for a pair; N = number of coefficients, CENTRED: P is in s = two_over_T z^2 - 1
template <int N, bool CENTRED>
__device__ __forceinline__ f2 odd_poly2(f2 z, const float (&c)[N], float two_over_T)
{
    f2 x = mul2(z, z);
    if (CENTRED) x = fma2(x, bc(two_over_T), bc(-1.0f));
    f2 p = fma2(bc(c[0]), x, bc(c[1]));
#pragma unroll
    for (int k = 2; k < N; ++k) p = fma2(p, x, bc(c[k]));
    return mul2(z, p);
}

// ---- SIE ----------------------------------------------------------------------------------
// Kormann et al. 1994 (cited PAPER.md:220; reading R2):
//   alpha_u = A atan(q' u/psi), alpha_v = A atanh(q' v/psi), A = b sqrt(q)/q',
//   psi = sqrt(q^2 u^2 + v^2), (u, v) in the lens frame (major axis along u).
// The arguments are bounded by the axis ratio:  z_u^2 <= q'^2/q^2,  z_v^2 <= q'^2 = 1 - q^2.
// prep.cu stores the mode of a vector (the most general one any of its SIEs needs) in the
// header of its derived block; it is block-uniform in the tracer.
//   mode   q^2 >=   atan               atanh
//   0      0.84     kAtan019           kAtanh016
//   1      0.64     kAtan056           kAtanh036
//   2      0.50     kAtan1             kAtanh050
//   3      1/3      kAtan2             kAtanh067  (or log, kAtanhLogFrom)
//   4      0.25     kAtan3             kAtanh075  (or log)
//   5      -        pi/2 - atan(1/z)   log:  lg2((1 + z)/(1 - z)) with MUFU rcp + lg2
// The log form is only used where q' >= 0.58, i.e. A <= 1.7 b: lg2's absolute error 2^-22
// then moves a ray by < 1e-6 b.  (Near q = 1, where A is large, modes 0-2 are polynomials in
// relative error.)  prep.cu floors q' at 1e-4 in both A and the arguments (relative change
// <= q'^2/3 ~ 3e-9), so q -> 1 needs no special case.
// Block: [c0][cs, sn, q^2, q'][cs A, sn A, cs A l, -sn A l], l = ln 2 / 2 (atanh in lg2 units).
constexpr int kSieModes = 6;
constexpr int kAtanhLogFrom = 5;           // modes >= this take the log form of atanh

template <int MODE>
__device__ __forceinline__ f2 sie_atan2x(f2 z)
{
    if constexpr (MODE == 0) return odd_poly2<5, false>(z, kAtan019, 0.0f);
    else if constexpr (MODE == 1) return odd_poly2<7, false>(z, kAtan056, 0.0f);
    else if constexpr (MODE == 2) return odd_poly2<9, false>(z, kAtan1, 0.0f);
    else if constexpr (MODE == 3) return odd_poly2<11, true>(z, kAtan2, 1.0f);
    else if constexpr (MODE == 4) return odd_poly2<13, true>(z, kAtan3, 2.0f / 3.0f);
    else {
        // |z| > 1: atan|z| = pi/2 - atan(1/|z|), through a = -1/|z|
        float z0, z1;
        un2(z, z0, z1);
        const float i0 = mufu_rcp(fmaxf(fabsf(z0), 1.0f)), i1 = mufu_rcp(fmaxf(fabsf(z1), 1.0f));
        const bool b0 = fabsf(z0) > 1.0f, b1 = fabsf(z1) > 1.0f;
        const f2 a = mk2(b0 ? -i0 : fabsf(z0), b1 ? -i1 : fabsf(z1));
        const f2 hp = mk2(b0 ? kHalfPi : 0.0f, b1 ? kHalfPi : 0.0f);
        const f2 r = add2(odd_poly2<9, false>(a, kAtan1, 0.0f), hp);
        return map2(r, z, [](float x, float s) { return copysignf(x, s); });
    }
}

// (2/ln 2) atanh(q' v / psi) for a pair, from v and s = q'/psi; qp = q' of THIS lens.
// The mode is per vector (the most general one any of its SIEs needs), so in mode 5 a second,
// rounder SIE of the same vector arrives here too: its A = b sqrt(q)/q' is large and the log
// form's absolute error would be multiplied by it.  The branch on its own q' (block-uniform)
// keeps the invariant "log form only where q' >= 0.6, A <= 1.7 b".
template <int MODE>
__device__ __forceinline__ f2 sie_atanh2x(f2 v, f2 s, float qp)
{
    if constexpr (MODE >= kAtanhLogFrom) {
        if (qp < 0.6f) return odd_poly2<7, false>(mul2(v, s), kAtanh036, 0.0f);    // z^2 <= q'^2 < 0.36
        const f2 num = fma2(v, s, bc(1.0f));
        f2 den = fma2(v, mul2(s, bc(-1.0f)), bc(1.0f));
        if (MODE >= 5) den = map2(den, [](float x) { return fmaxf(x, 1e-7f); });   // q' -> 1 on the v axis
        const f2 ratio = mul2(num, map2(den, [](float x) { return mufu_rcp(x); }));
        return map2(ratio, [](float x) { return mufu_lg2(x); });
    } else {
        const f2 z = mul2(v, s);
        if constexpr (MODE == 0) return odd_poly2<5, false>(z, kAtanh016, 0.0f);
        else if constexpr (MODE == 1) return odd_poly2<7, false>(z, kAtanh036, 0.0f);
        else if constexpr (MODE == 2) return odd_poly2<9, false>(z, kAtanh050, 0.0f);
        else if constexpr (MODE == 3) return odd_poly2<11, true>(z, kAtanh067, 3.0f);
        else return odd_poly2<13, true>(z, kAtanh075, 8.0f / 3.0f);
    }
}

// frame origin of a positioned component for pixel (jf, rf): d[0] = (cxi, cxf, cyi, cyf),
// offsets formed as (integer difference) - fraction (lensed_internal.h)
__device__ __forceinline__ void centre_offset(const float4 &c0, float jf, float rf, float &dx, float &dy)
{
    dx = (jf - c0.x) - c0.y;
    dy = (rf - c0.z) - c0.w;
}

__device__ __forceinline__ void sie_origin(const float4 *d, float jf, float rf, float &u0, float &v0)
{
    float dx, dy;
    centre_offset(d[0], jf, rf, dx, dy);
    const float4 c1 = d[1];
    u0 = fmaf(c1.x, dx, c1.y * dy);
    v0 = fmaf(c1.x, dy, -c1.y * dx);
}

// the same origins for two pixels at once (pixel pairs): jf, rf = (column, row) of both
__device__ __forceinline__ void centre_offset(const float4 &c0, f2 jf, f2 rf, f2 &dx, f2 &dy)
{
    dx = add2(add2(jf, bc(-c0.x)), bc(-c0.y));
    dy = add2(add2(rf, bc(-c0.z)), bc(-c0.w));
}
__device__ __forceinline__ void sie_origin(const float4 *d, f2 jf, f2 rf, f2 &u0, f2 &v0)
{
    f2 dx, dy;
    centre_offset(d[0], jf, rf, dx, dy);
    const float4 c1 = d[1];
    u0 = fma2(bc(c1.x), dx, mul2(bc(c1.y), dy));
    v0 = fma2(bc(c1.x), dy, mul2(bc(-c1.y), dx));
}

// RAW: leave (atan, atanh-in-lg2-units) themselves in (r.ax, r.ay) instead of accumulating the
// deflection: the sources then subtract B (atan, atanh), B = M_source x [amplitudes, rotation]
// (trace_static.cuh "direct frames").
template <int NP, int MODE, bool RAW = false, class O = float>
__device__ __forceinline__ void lens_sie(const float4 *d, const float *tu, const float *tv, O u0, O v0,
                                         Rays<NP> &r)
{
    const float4 c1 = d[1], c2 = d[2];
    f2 pu[NP], pv[NP];
    enter<NP>(tu, u0, pu);
    enter<NP>(tv, v0, pv);
#pragma unroll
    for (int k = 0; k < NP; ++k) {
        const f2 u = pu[k], v = pv[k];
        const f2 psi2 = fma2(mul2(u, bc(c1.z)), u, mul2(v, v));
#ifdef LENSED_RSQ_NEWTON            // tuning build: the SIE's rsqrt off the XU pipe (integer seed + packed Newton steps)
        f2 ipsi = map2(psi2, [](float x) { return __uint_as_float(0x5f375a86u - (__float_as_uint(fmaxf(x, kTiny)) >> 1)); });
        {
            const f2 hx = mul2(map2(psi2, [](float x) { return fmaxf(x, kTiny); }), bc(0.5f));
#pragma unroll
            for (int it = 0; it < LENSED_RSQ_NEWTON; ++it) ipsi = mul2(ipsi, fma2(mul2(hx, ipsi), mul2(ipsi, bc(-1.0f)), bc(1.5f)));
        }
#else
        const f2 ipsi = map2(psi2, [](float x) { return mufu_rsq(fmaxf(x, kTiny)); });
#endif
        const f2 s = mul2(ipsi, bc(c1.w));
        const f2 at = sie_atan2x<MODE>(mul2(u, s));
        const f2 lv = sie_atanh2x<MODE>(v, s, c1.w);
        if (RAW) {
            r.ax[k] = at;
            r.ay[k] = lv;
        } else {
            r.ax[k] = fma2(lv, bc(c2.w), fma2(at, bc(c2.x), r.ax[k]));
            r.ay[k] = fma2(lv, bc(c2.z), fma2(at, bc(c2.y), r.ay[k]));
        }
    }
}

// ---- SIS / point mass (R3) ------------------------------------------------------------------
// SIS: alpha = b (u, v)/r; point mass: alpha = thetaE^2 (u, v)/r^2; both 0 at r = 0.
// Block: [c0][b or thetaE^2, 0, 0, 0]; identity frame = the raw rule offsets.
__device__ __forceinline__ void circular_origin(const float4 *d, float jf, float rf, float &u0, float &v0)
{
    centre_offset(d[0], jf, rf, u0, v0);
}

__device__ __forceinline__ void circular_origin(const float4 *d, f2 jf, f2 rf, f2 &u0, f2 &v0)
{
    centre_offset(d[0], jf, rf, u0, v0);
}

template <int NP, bool POINT, class O = float>
__device__ __forceinline__ void lens_circular(const float4 *d, const float *tu, const float *tv, O u0, O v0,
                                              Rays<NP> &r)
{
    const float amp = d[1].x;
    f2 pu[NP], pv[NP];
    enter<NP>(tu, u0, pu);
    enter<NP>(tv, v0, pv);
#pragma unroll
    for (int k = 0; k < NP; ++k) {
        const f2 u = pu[k], v = pv[k];
        const f2 r2 = fma2(u, u, mul2(v, v));
        const f2 inv = map2(r2, [](float x) { return POINT ? mufu_rcp(fmaxf(x, kTiny)) : mufu_rsq(fmaxf(x, kTiny)); });
        const f2 s = mul2(inv, bc(amp));
        r.ax[k] = fma2(s, u, r.ax[k]);
        r.ay[k] = fma2(s, v, r.ay[k]);
    }
}

// ---- external shear about the image centre (R4) ---------------------------------------------
// alpha = (g1 x + g2 y, g2 x - g1 y): linear, so alpha = (per pixel) + (table).
// INIT: first lens of the list, alpha starts here.
__device__ __forceinline__ void shear_origin(const float4 *d, float jf, float rf, float cxh, float cyh, float &u0,
                                             float &v0)
{
    const float4 c0 = d[0];
    const float x0 = jf - cxh, y0 = rf - cyh;
    u0 = fmaf(c0.x, x0, c0.y * y0);
    v0 = fmaf(c0.y, x0, -c0.x * y0);
}

__device__ __forceinline__ void shear_origin(const float4 *d, f2 jf, f2 rf, float cxh, float cyh, f2 &u0, f2 &v0)
{
    const float4 c0 = d[0];
    const f2 x0 = add2(jf, bc(-cxh)), y0 = add2(rf, bc(-cyh));
    u0 = fma2(bc(c0.x), x0, mul2(bc(c0.y), y0));
    v0 = fma2(bc(c0.y), x0, mul2(bc(-c0.x), y0));
}

template <int NP, bool INIT, class O = float>
__device__ __forceinline__ void lens_shear(const float *tu, const float *tv, O u0, O v0, Rays<NP> &r)
{
    f2 pu[NP], pv[NP];
    enter<NP>(tu, u0, pu);
    enter<NP>(tv, v0, pv);
#pragma unroll
    for (int k = 0; k < NP; ++k) {
        const f2 a = pu[k], b = pv[k];
        r.ax[k] = INIT ? a : add2(r.ax[k], a);
        r.ay[k] = INIT ? b : add2(r.ay[k], b);
    }
}

// ---- Sersic / Gaussian light ------------------------------------------------------------------
// Sersic, eqs. 22-23:  I = I0 exp(-b_n (R/r_S)^(1/n))
//   = 2^(log2 I0 - (b_n log2 e) 2^(lg2((R/r_S)^2) / (2n))).   R = 0: lg2 = -inf, 2^-inf = 0, I = I0.
// Gaussian (R7):  I = I0 exp(-R^2 / (2 sigma^2)) = 2^(log2 I0 - (log2 e / 2) (R/sigma)^2).
// Block: [c0][a1, a2, a3, a4][log2 I0, b_n log2 e | log2 e / 2, 1/(2n), 0], frame scaled by
// 1/r_S | 1/sigma so that u^2 + v^2 = (R/r_S)^2 with R of eq. 23.
__device__ __forceinline__ void light_origin(const float4 *d, float jf, float rf, float &u0, float &v0)
{
    float dx, dy;
    centre_offset(d[0], jf, rf, dx, dy);
    const float4 c1 = d[1];
    u0 = fmaf(c1.x, dx, c1.y * dy);
    v0 = fmaf(c1.z, dx, c1.w * dy);
}

__device__ __forceinline__ void light_origin(const float4 *d, f2 jf, f2 rf, f2 &u0, f2 &v0)
{
    f2 dx, dy;
    centre_offset(d[0], jf, rf, dx, dy);
    const float4 c1 = d[1];
    u0 = fma2(bc(c1.x), dx, mul2(bc(c1.y), dy));
    v0 = fma2(bc(c1.z), dx, mul2(bc(c1.w), dy));
}

// cm: the 2 x 2 matrix applied to (r.ax, r.ay) of a source -- the frame M itself (d[1]) when
// they hold the deflection, B when they hold the SIE's raw functions.
// rmin (source Sersic only): running minimum of (R/r_S)^2 over the rays of the pixel; the caller
// compares it with the block's T2 (lensed_internal.h) to flag the pixel for the FP64 refinement.
template <int NP, bool SRC, bool GAUSS, bool INIT, class O = float, class RM = float>
__device__ __forceinline__ void light_profile(const float4 *d, const float *tu, const float *tv, O u0, O v0,
                                              Rays<NP> &r, const float4 *cm, RM &rmin)
{
    const float4 c1 = cm ? cm[0] : d[1], c2 = d[2];
    const float nk = -c2.y;
    f2 pu[NP], pv[NP];
    enter<NP>(tu, u0, pu);
    enter<NP>(tv, v0, pv);
#pragma unroll
    for (int k = 0; k < NP; ++k) {
        f2 u = pu[k], v = pv[k];
        if (SRC) {
            u = fma2(r.ay[k], bc(-c1.y), fma2(r.ax[k], bc(-c1.x), u));
            v = fma2(r.ay[k], bc(-c1.w), fma2(r.ax[k], bc(-c1.z), v));
        }
        const f2 r2 = fma2(u, u, mul2(v, v));
        f2 x;
        if (GAUSS) {
            x = fma2(r2, bc(nk), bc(c2.x));
        } else {
#ifndef LENSED_NO_FLAG                  // tuning builds: what the flagging costs
            if (SRC) min_radius(rmin, r2);
#endif
            const f2 lg = map2(r2, [](float a) { return mufu_lg2(a); });
            const f2 e = map2(mul2(lg, bc(c2.z)), [](float a) { return mufu_ex2(a); });
            x = fma2(e, bc(nk), bc(c2.x));
        }
        const f2 val = map2(x, [](float a) { return mufu_ex2(a); });
        r.I[k] = INIT ? val : add2(r.I[k], val);
    }
}

}  // namespace lensed
