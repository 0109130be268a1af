// trace.cu -- steps a1-a4: ray generation, deflection summed over lenses, surface
// brightness, pixel quadrature, fused; one launch covers (pixel chunk) x (parameter vector).
//
//   x_k = pixel centre + (xi_k, eta_k)                       PAPER.md:155-159 eq. 14
//   y_k = x_k - sum_lenses alpha(x_k)                        PAPER.md:53-57  eq. 1
//   I   = sum_src I_S(y_k) + sum_fg I_L(x_k) + sky           PAPER.md:59-63  eq. 2
//   L_i = sum_k w_k I                                        PAPER.md:155-157 eq. 14
//
// Layout.  blockIdx.y = parameter vector, blockIdx.x = chunk of the traced-pixel list.  A
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
// (frames x rule points) once in its prologue.  Sources see the deflected position:
//     (u, v) = M (x - c) - M alpha,   two packed FMAs per coordinate.
// The shear is linear, so its whole deflection is "per pixel + table"; it is sorted to the
// front of the lens list (api.cu) and initialises alpha.  Sky is added once per pixel (the
// rule weights sum to one).
//
// Arithmetic: FP32, packed FFMA2 / FMUL2 / FADD2 on the FMA pipe, MUFU rsqrt / rcp / lg2 /
// ex2 on the XU pipe (the bound: DESIGN.md 5.2), selects and clamps on the ALU pipe.
#include "lensed_internal.h"
#include "f32x2.cuh"

namespace lensed {
namespace {

constexpr int kThreads = 256;

__device__ __forceinline__ float mufu_rsq(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_rcp(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_lg2(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_ex2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

constexpr float kTiny = 1e-30f;            // floor of squared radii: rsqrt / rcp stay finite, 0 * finite = 0
constexpr float kHalfPi = 1.5707963267948966f;

template <int NP>
struct Rays {
    f2 ax[NP], ay[NP];   // summed deflection, pixels
    f2 I[NP];            // summed brightness
};

// NP consecutive pairs of one table row, starting at rule point q0 (a multiple of 2 NP)
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

// atan(z) for a pair.  BIG = the block's vector can have |z| > 1 (q'/q > 1): then
// atan|z| = pi/2 - atan(1/|z|) through a = -1/|z|.  P: minimax of atan(a)/a in a^2 on [0, 1],
// relative error 1.5e-8.
template <bool BIG>
__device__ __forceinline__ f2 atan2x(f2 z)
{
    f2 a = z, hp;
    if (BIG) {
        float z0, z1;
        un2(z, z0, z1);
        const float i0 = mufu_rcp(fmaxf(fabsf(z0), 1.0f)), i1 = mufu_rcp(fmaxf(fabsf(z1), 1.0f));
        const bool b0 = fabsf(z0) > 1.0f, b1 = fabsf(z1) > 1.0f;
        a = mk2(b0 ? -i0 : fabsf(z0), b1 ? -i1 : fabsf(z1));
        hp = mk2(b0 ? kHalfPi : 0.0f, b1 ? kHalfPi : 0.0f);
    }
    const f2 t = mul2(a, a);
    f2 p = fma2(bc(2.8498720241e-03f), t, bc(-1.6068558782e-02f));
    p = fma2(p, t, bc(4.2691405628e-02f));
    p = fma2(p, t, bc(-7.5042849627e-02f));
    p = fma2(p, t, bc(1.0640929559e-01f));
    p = fma2(p, t, bc(-1.4203643337e-01f));
    p = fma2(p, t, bc(1.9992619252e-01f));
    p = fma2(p, t, bc(-3.3333073338e-01f));
    p = fma2(p, t, bc(9.9999998477e-01f));
    if (!BIG) return mul2(a, p);
    const f2 r = fma2(a, p, hp);
    return map2(r, z, [](float x, float s) { return copysignf(x, s); });
}

// 2 atanh(z) / ln 2 = lg2((1+z)/(1-z)) for a pair, |z| < 1.  Below z^2 = 0.16 a polynomial
// of atanh(z)/z in z^2 (relative error 2.8e-8, coefficients pre-multiplied by 2/ln 2);
// above, MUFU rcp + lg2, where lg2's absolute error (2^-22) is harmless.  LARGE = the
// block's vector can reach z^2 >= 0.16 at all (q' >= 0.4).
template <bool LARGE>
__device__ __forceinline__ f2 lg2_ratio2x(f2 z)
{
    const f2 t = mul2(z, z);
    f2 p = fma2(bc(4.5452297837e-01f), t, bc(3.9193670683e-01f));
    p = fma2(p, t, bc(5.7828278000e-01f));
    p = fma2(p, t, bc(9.6177198511e-01f));
    p = fma2(p, t, bc(2.8853901623e+00f));
    const f2 small = mul2(z, p);
    if (!LARGE) return small;
    const f2 zc = map2(z, [](float x) { return fminf(fabsf(x), 0.99999994f); });
    const f2 num = add2(zc, bc(1.0f)), den = fma2(zc, bc(-1.0f), bc(1.0f));
    const f2 ratio = mul2(num, map2(den, [](float x) { return mufu_rcp(x); }));
    const f2 lg = map2(ratio, [](float x) { return mufu_lg2(x); });
    float s0, s1, l0, l1, t0, t1, z0, z1;
    un2(small, s0, s1); un2(lg, l0, l1); un2(t, t0, t1); un2(z, z0, z1);
    return mk2(t0 < 0.16f ? s0 : copysignf(l0, z0), t1 < 0.16f ? s1 : copysignf(l1, z1));
}

// SIE (Kormann et al. 1994; R2):  alpha_u = A atan(q' u/psi), alpha_v = A atanh(q' v/psi),
// A = b sqrt(q)/q', psi = sqrt(q^2 u^2 + v^2), (u, v) in the lens frame (major axis along u).
// prep.cu floors q' at 1e-4 in both A and the arguments (relative change <= q'^2/3 ~ 3e-9),
// so q -> 1 needs no special case.  Block: [c0][cs, sn, q^2, q'][cs A, sn A, cs A l, -sn A l],
// l = ln 2 / 2 (the atanh comes back in lg2 units).
template <int NP, bool BIG, bool LARGE>
__device__ __forceinline__ void lens_sie(const float4 *d, const float *tu, const float *tv, float jf, float rf,
                                         Rays<NP> &r)
{
    const float4 c0 = d[0], c1 = d[1], c2 = d[2];
    const float dx0 = (jf - c0.x) - c0.y, dy0 = (rf - c0.z) - c0.w;
    const float u0 = fmaf(c1.x, dx0, c1.y * dy0), v0 = fmaf(c1.x, dy0, -c1.y * dx0);
    f2 pu[NP], pv[NP];
    load_pairs<NP>(tu, pu);
    load_pairs<NP>(tv, pv);
#pragma unroll
    for (int k = 0; k < NP; ++k) {
        const f2 u = add2(pu[k], bc(u0)), v = add2(pv[k], bc(v0));
        const f2 psi2 = fma2(mul2(u, bc(c1.z)), u, mul2(v, v));
        const f2 ipsi = map2(psi2, [](float x) { return mufu_rsq(fmaxf(x, kTiny)); });
        const f2 s = mul2(ipsi, bc(c1.w));
        const f2 at = atan2x<BIG>(mul2(u, s));
        const f2 lv = lg2_ratio2x<LARGE>(mul2(v, s));
        r.ax[k] = fma2(lv, bc(c2.w), fma2(at, bc(c2.x), r.ax[k]));
        r.ay[k] = fma2(lv, bc(c2.z), fma2(at, bc(c2.y), r.ay[k]));
    }
}

// SIS: alpha = b (u, v)/r; point mass: alpha = thetaE^2 (u, v)/r^2; both 0 at r = 0 (R3).
// Block: [c0][b or thetaE^2, 0, 0, 0]; identity frame = the raw rule offsets.
template <int NP, bool POINT>
__device__ __forceinline__ void lens_circular(const float4 *d, const float *tu, const float *tv, float jf, float rf,
                                              Rays<NP> &r)
{
    const float4 c0 = d[0], c1 = d[1];
    const float dx0 = (jf - c0.x) - c0.y, dy0 = (rf - c0.z) - c0.w;
    f2 pu[NP], pv[NP];
    load_pairs<NP>(tu, pu);
    load_pairs<NP>(tv, pv);
#pragma unroll
    for (int k = 0; k < NP; ++k) {
        const f2 u = add2(pu[k], bc(dx0)), v = add2(pv[k], bc(dy0));
        const f2 r2 = fma2(u, u, mul2(v, v));
        const f2 inv = map2(r2, [](float x) { return POINT ? mufu_rcp(fmaxf(x, kTiny)) : mufu_rsq(fmaxf(x, kTiny)); });
        const f2 s = mul2(inv, bc(c1.x));
        r.ax[k] = fma2(s, u, r.ax[k]);
        r.ay[k] = fma2(s, v, r.ay[k]);
    }
}

// External shear about the image centre (R4): alpha = (g1 x + g2 y, g2 x - g1 y); linear,
// so alpha = (per pixel) + (table).  INIT: first lens of the list, alpha starts here.
template <int NP, bool INIT>
__device__ __forceinline__ void lens_shear(const float4 *d, const float *tu, const float *tv, float jf, float rf,
                                           float cxh, float cyh, Rays<NP> &r)
{
    const float4 c0 = d[0];
    const float x0 = jf - cxh, y0 = rf - cyh;
    const float sx = fmaf(c0.x, x0, c0.y * y0), sy = fmaf(c0.y, x0, -c0.x * y0);
    f2 pu[NP], pv[NP];
    load_pairs<NP>(tu, pu);
    load_pairs<NP>(tv, pv);
#pragma unroll
    for (int k = 0; k < NP; ++k) {
        const f2 a = add2(pu[k], bc(sx)), b = add2(pv[k], bc(sy));
        r.ax[k] = INIT ? a : add2(r.ax[k], a);
        r.ay[k] = INIT ? b : add2(r.ay[k], b);
    }
}

// Sersic, eqs. 22-23:  I = I0 exp(-b_n (R/r_S)^(1/n))
//   = 2^(log2 I0 - (b_n log2 e) 2^(lg2((R/r_S)^2) / (2n))).   R = 0: lg2 = -inf, 2^-inf = 0, I = I0.
// Gaussian (R7):  I = I0 exp(-R^2 / (2 sigma^2)) = 2^(log2 I0 - (log2 e / 2) (R/sigma)^2).
// Block: [c0][a1, a2, a3, a4][log2 I0, b_n log2 e | log2 e / 2, 1/(2n), 0], frame scaled by
// 1/r_S | 1/sigma so that u^2 + v^2 = (R/r_S)^2 with R of eq. 23.
template <int NP, bool SRC, bool GAUSS>
__device__ __forceinline__ void light_profile(const float4 *d, const float *tu, const float *tv, float jf, float rf,
                                              Rays<NP> &r)
{
    const float4 c0 = d[0], c1 = d[1], c2 = d[2];
    const float dx0 = (jf - c0.x) - c0.y, dy0 = (rf - c0.z) - c0.w;
    const float u0 = fmaf(c1.x, dx0, c1.y * dy0), v0 = fmaf(c1.z, dx0, c1.w * dy0);
    const float nk = -c2.y;
    f2 pu[NP], pv[NP];
    load_pairs<NP>(tu, pu);
    load_pairs<NP>(tv, pv);
#pragma unroll
    for (int k = 0; k < NP; ++k) {
        f2 u = add2(pu[k], bc(u0)), v = add2(pv[k], bc(v0));
        if (SRC) {
            u = fma2(r.ay[k], bc(-c1.y), fma2(r.ax[k], bc(-c1.x), u));
            v = fma2(r.ay[k], bc(-c1.w), fma2(r.ax[k], bc(-c1.z), v));
        }
        const f2 r2 = fma2(u, u, mul2(v, v));
        f2 x;
        if (GAUSS) {
            x = fma2(r2, bc(nk), bc(c2.x));
        } else {
            const f2 lg = map2(r2, [](float a) { return mufu_lg2(a); });
            const f2 e = map2(mul2(lg, bc(c2.z)), [](float a) { return mufu_ex2(a); });
            x = fma2(e, bc(nk), bc(c2.x));
        }
        r.I[k] = add2(r.I[k], map2(x, [](float a) { return mufu_ex2(a); }));
    }
}

// Shared memory of a block: [D/4] float4 derived constants of its vector, then the frame
// tables  tab[slot][2][nq_pad]  (slot 0 = identity, 1 + m = lens m, 1 + n_lens + m = light
// m), then the rule weights [nq_pad].
template <int NP>
__global__ void __launch_bounds__(kThreads, 2) trace_kernel(Program prog, TraceArgs a)
{
    constexpr int R = 2 * NP;
    extern __shared__ float4 smem4[];
    float4 *sder = smem4;
    float *stab = reinterpret_cast<float *>(smem4 + prog.D / 4);
    const int nq = a.nq_pad;
    const int n_slots = 1 + prog.n_lens + prog.n_light;
    float *sw = stab + (size_t)n_slots * 2 * nq;
    const int bvec = blockIdx.y;
    {
        const float4 *g = reinterpret_cast<const float4 *>(a.derived + (size_t)bvec * prog.D);
        for (int i = threadIdx.x; i < prog.D / 4; i += kThreads) sder[i] = g[i];
    }
    __syncthreads();
    if (sder[0].x == 0.0f) return;                // vector outside the model domain: skipped
    float sky = 0.0f;
    for (int m = 0; m < prog.n_light; ++m)
        if (prog.light_kind[m] == K_SKY) sky += sder[prog.light_off[m] >> 2].x;
    for (int i = threadIdx.x; i < n_slots * nq; i += kThreads) {
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
        if (slot == 0) sw[k] = qk.z;
    }
    __syncthreads();
    float *Lb = a.L + (size_t)bvec * a.l_stride;

    const int base = blockIdx.x * a.pix_per_block;
    const int end = min(base + a.pix_per_block, a.npix);
#pragma unroll 1
    for (int ip = base + threadIdx.x; ip < end; ip += kThreads) {
        const uint32_t rc = a.pix[ip];
        const int row = (int)(rc >> 16), col = (int)(rc & 0xffffu);
        const float jf = (float)col, rf = (float)row;
        f2 acc = bc(0.0f);
#pragma unroll 1
        for (int q0 = 0; q0 < nq; q0 += R) {
            Rays<NP> r;
#pragma unroll
            for (int k = 0; k < NP; ++k) r.I[k] = bc(0.0f);
            int m = 0;
            if (prog.n_lens > 0 && prog.lens_kind[0] == K_SHEAR) {
                lens_shear<NP, true>(sder + (prog.lens_off[0] >> 2), stab + 2 * nq + q0, stab + 3 * nq + q0, jf, rf,
                                     a.cxh, a.cyh, r);
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
                case K_SIE: {
                    // q^2 < 1/2: q'/q > 1, the atan needs its range reduction; q' >= 0.4: the
                    // atanh can leave the polynomial's range.  Both block-uniform.
                    const bool big = d[1].z < 0.5f, large = d[1].w >= 0.4f;
                    if (big) lens_sie<NP, true, true>(d, tu, tv, jf, rf, r);
                    else if (large) lens_sie<NP, false, true>(d, tu, tv, jf, rf, r);
                    else lens_sie<NP, false, false>(d, tu, tv, jf, rf, r);
                    break;
                }
                case K_SIS:   lens_circular<NP, false>(d, stab + q0, stab + nq + q0, jf, rf, r); break;
                case K_POINT: lens_circular<NP, true>(d, stab + q0, stab + nq + q0, jf, rf, r); break;
                default:      lens_shear<NP, false>(d, tu, tv, jf, rf, a.cxh, a.cyh, r); break;
                }
            }
#pragma unroll 1
            for (m = 0; m < prog.n_light; ++m) {
                const float4 *d = sder + (prog.light_off[m] >> 2);
                const float *tu = stab + (size_t)(2 * (1 + prog.n_lens + m)) * nq + q0, *tv = tu + nq;
                switch (prog.light_kind[m]) {
                case K_SRC_SERSIC: light_profile<NP, true, false>(d, tu, tv, jf, rf, r); break;
                case K_FG_SERSIC:  light_profile<NP, false, false>(d, tu, tv, jf, rf, r); break;
                case K_SRC_GAUSS:  light_profile<NP, true, true>(d, tu, tv, jf, rf, r); break;
                case K_FG_GAUSS:   light_profile<NP, false, true>(d, tu, tv, jf, rf, r); break;
                default: break;                   // sky: added once per pixel below
                }
            }
            f2 w[NP];
            load_pairs<NP>(sw + q0, w);
#pragma unroll
            for (int k = 0; k < NP; ++k) acc = fma2(w[k], r.I[k], acc);
        }
        Lb[row * a.W + col] = (lo2(acc) + hi2(acc)) + sky;
    }
}

template <int NP>
cudaError_t launch_trace_NP(const Program &prog, const TraceArgs &a, int nvec, cudaStream_t st)
{
    const size_t smem = trace_smem_bytes(prog, a.nq_pad);
    static size_t s_attr = 48 * 1024;             // raise the dynamic shared memory limit on demand
    if (smem > s_attr) {
        cudaError_t e = cudaFuncSetAttribute(trace_kernel<NP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        s_attr = smem;
    }
    dim3 grid((a.npix + a.pix_per_block - 1) / a.pix_per_block, nvec);
    trace_kernel<NP><<<grid, kThreads, smem, st>>>(prog, a);
    return cudaGetLastError();
}

}  // namespace

size_t trace_smem_bytes(const Program &prog, int nq_pad)
{
    const size_t n_slots = 1 + prog.n_lens + prog.n_light;
    return (size_t)prog.D * sizeof(float) + (n_slots * 2 + 1) * (size_t)nq_pad * sizeof(float);
}

// Rays carried per thread, R = 2 NP in {2, 4, 6, 8, 10}: least padded rule length, weighted
// by a per-block overhead that shrinks with R (4 -> 4, 9 -> 10, 16 -> 8, 25 -> 10, 49 -> 10).
int trace_pick_R(int n_quad)
{
    int best = 2;
    double best_cost = 1e300;
    for (int R = 2; R <= 10; R += 2) {
        const int pad = (n_quad + R - 1) / R * R;
        const double cost = pad * (1.0 + 0.6 / R);
        if (cost < best_cost - 1e-12) { best = R; best_cost = cost; }
    }
    return best;
}

cudaError_t launch_trace(const Program &prog, const TraceArgs &a, int R, int nvec, cudaStream_t st)
{
    switch (R) {
    case 2: return launch_trace_NP<1>(prog, a, nvec, st);
    case 4: return launch_trace_NP<2>(prog, a, nvec, st);
    case 6: return launch_trace_NP<3>(prog, a, nvec, st);
    case 8: return launch_trace_NP<4>(prog, a, nvec, st);
    case 10: return launch_trace_NP<5>(prog, a, nvec, st);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace lensed
