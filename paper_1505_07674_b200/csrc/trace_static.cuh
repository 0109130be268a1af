// trace_static.cuh -- the ray tracer with the model list fixed at compile time.
//
// Same computation and layout as trace.cu (steps a1-a4, eqs. 1-2
// eq. 14), but the lens / light lists are a template signature, so one pass over R rays is
// straight-line code: no switch per model, no list indexing, and ptxas interleaves the
// MUFU-heavy light profiles with the FMA-heavy SIE polynomials inside one warp (the
// interpreted kernel serialises them: profiles/r1c).  Per-pixel frame origins are computed
// once per pixel, not once per pass.  api.cu sorts the lists into the canonical order
//   lenses: shear, SIE, SIS, point mass        lights: source Sersic, source Gaussian,
//                                                      foreground Sersic, foreground Gaussian, sky
// and trace.cu picks the static kernel whose signature matches, else the interpreted one.
#pragma once
#include "trace_block.cuh"

namespace lensed {

template <int NSHEAR, int NSIE, int NSIS, int NPOINT, int NSS, int NSG, int NFS, int NFG>
struct TraceSig {
    static_assert(NSHEAR <= 1, "at most one shear in a static signature");
    static constexpr int n_shear = NSHEAR, n_sie = NSIE, n_sis = NSIS, n_point = NPOINT;
    static constexpr int n_ss = NSS, n_sg = NSG, n_fs = NFS, n_fg = NFG;
    static constexpr int n_lens = NSHEAR + NSIE + NSIS + NPOINT;
    static constexpr int n_pos = NSS + NSG + NFS + NFG;          // positioned lights (sky excluded)
    static constexpr int n_src = NSS + NSG;
    // "Direct frames": with one SIE and no other non-linear lens, the deflection is never
    // formed.  alpha = Gamma (x - x_c) + R diag(A, A l) (atan, atanh), so in a source frame
    //   M (x - c - alpha) = [M (x - c) - M Gamma (x - x_c)]  -  B (atan, atanh),   B = M R diag(A, A l):
    // the bracket is linear in x -- the source's table and per-pixel origin absorb the shear --
    // and the SIE leaves its two raw functions in (ax, ay).  Saves the two packed adds of the
    // shear and the four packed FMAs of the SIE's accumulation per pair of rays.
    static constexpr bool direct = NSIE == 1 && NSIS == 0 && NPOINT == 0 && NSS + NSG >= 1;
    // float4 index of the derived block of lens / light m (canonical order) in the vector's derived
    // constants: api.cu lays them out header, lenses, lights in that order, so for a signature the
    // offsets are compile-time constants (blocks: shear 1, SIE 3, SIS / point 2 | Sersic 4, Gaussian 3)
    __host__ __device__ static constexpr int lens_off4(int m)
    {
        return 1 + (m < NSHEAR ? m : NSHEAR + (m < NSHEAR + NSIE ? 3 * (m - NSHEAR) : 3 * NSIE + 2 * (m - NSHEAR - NSIE)));
    }
    __host__ __device__ static constexpr int light_off4(int m)
    {
        return lens_off4(n_lens) +
               (m < NSS ? 4 * m
                        : 4 * NSS + (m < NSS + NSG ? 3 * (m - NSS)
                                                   : 3 * NSG + (m < NSS + NSG + NFS ? 4 * (m - NSS - NSG)
                                                                                    : 4 * NFS + 3 * (m - NSS - NSG - NFS))));
    }
#ifndef __CUDACC_RTC__
    static bool matches(const int (&c)[K_COUNT])
    {
        return c[K_SHEAR] == NSHEAR && c[K_SIE] == NSIE && c[K_SIS] == NSIS && c[K_POINT] == NPOINT &&
               c[K_SRC_SERSIC] == NSS && c[K_SRC_GAUSS] == NSG && c[K_FG_SERSIC] == NFS && c[K_FG_GAUSS] == NFG;
    }
#endif
};

// ---- foreground expansion ------------------------------------------------------------------
// A foreground Sersic (eqs. 22-23) is evaluated at the image-plane point
// itself (eq. 2), so over one pixel its argument moves over a known patch of its own frame:
// y = y0 + M delta_k with y0 = M (pixel centre - c) and delta_k the rule offsets.  Away from
// its centre the profile I = exp(h(s)), s = |y|^2, h = ln I0 - b_n s^(1/2n), is smooth on that
// scale, and the rule sum of eq. 14 follows from its Taylor series in
// Delta = s - s0 = L + Q,  L = 2 y0 . M delta,  Q = |M delta|^2,  to fourth order in delta:
//   sum_k w_k I(y0 + M delta_k) = F0 + F1 E[Q] + F2/2 (E[L^2] + E[Q^2]) + F3/2 E[L^2 Q] + F4/24 E[L^4],
// Fj = d^j exp(h)/ds^j at s0, where E[.] = sum_k w_k (.) are second and fourth moments of the
// rule in the light's frame (the odd ones vanish for a symmetric rule; api.cu checks).  The
// block prologue sums them from the SAME frame table the per-ray path reads, so the expansion
// reproduces the rule's own sum -- not the exact integral -- to 0.016 tau^6 (prep.cu
// "foreground expansion" derives the range of s0 where tau <= fgx_tau; default 0.15: 2e-7).
// Cost: 4 MUFU + ~70 flops per PIXEL instead of 3 MUFU + 17 flops per RAY; pixels outside the
// range (the few around the profile's centre) take the per-ray sum.
struct FgMoments { float S11, S12, S22, T0, T1, T2, T3, T4; };       // E[d_i d_j], E[d1^(4-i) d2^i]

// full: fourth-order form; else the second-order terms only (valid on the narrower range d[3].zw)
__device__ __forceinline__ float fg_expansion(const float4 *d, const FgMoments &m, float a, float b, float s0, bool full)
{
    const float4 c2 = d[2];                              // log2 I0, b_n log2 e, 1/(2n)
    const float c = c2.z;
    const float e = mufu_ex2(c * mufu_lg2(s0));          // s0^c
    const float F = mufu_ex2(fmaf(-c2.y, e, c2.x));
    const float is = mufu_rcp(s0);
    const float h1 = -(c2.y * 0.69314718056f) * c * e * is;           // dh/ds = -b_n c s^(c-1)
    const float h2 = h1 * (c - 1.0f) * is;
    const float h11 = h1 * h1;
    if (!full) {
        const float el2 = 4.0f * (a * a * m.S11 + 2.0f * a * b * m.S12 + b * b * m.S22);
        return fmaf(F, fmaf(h1, m.S11 + m.S22, 0.5f * (h11 + h2) * el2), F);
    }
    const float h3 = h2 * (c - 2.0f) * is, h4 = h3 * (c - 3.0f) * is;
    const float F1 = h1, F2 = h11 + h2, F3 = h1 * (h11 + 3.0f * h2) + h3;
    const float F4 = h11 * (h11 + 6.0f * h2) + 3.0f * h2 * h2 + 4.0f * h1 * h3 + h4;
    const float aa = a * a, ab = a * b, bb = b * b;
    const float EQ = m.S11 + m.S22;
    const float EL2 = 4.0f * (aa * m.S11 + 2.0f * ab * m.S12 + bb * m.S22);
    const float EQ2 = m.T0 + 2.0f * m.T2 + m.T4;
    const float EL2Q = 4.0f * (aa * (m.T0 + m.T2) + 2.0f * ab * (m.T1 + m.T3) + bb * (m.T2 + m.T4));
    const float EL4 = 16.0f * (aa * (aa * m.T0 + 4.0f * ab * m.T1 + 6.0f * bb * m.T2) + bb * (4.0f * ab * m.T3 + bb * m.T4));
    const float corr = F1 * EQ + 0.5f * F2 * (EL2 + EQ2) + 0.5f * F3 * EL2Q + (1.0f / 24.0f) * F4 * EL4;
    return fmaf(F, corr, F);
}

template <int NP, class S, int MODE>
__device__ __forceinline__ void trace_pixels(const Program &prog, const TraceArgs &a, const TraceBlock &tb, float *Lb, int vec)
{
    constexpr int R = 2 * NP;
    constexpr int NL = S::n_lens, NPOS = S::n_pos;
    constexpr int L_SIE = S::n_shear, L_SIS = L_SIE + S::n_sie, L_PT = L_SIS + S::n_sis;
    constexpr int G_SG = S::n_ss, G_FS = G_SG + S::n_sg, G_FG = G_FS + S::n_fs;
    const int nq = a.nq_pad;
    const float4 *sder = tb.sder;
    const float *ltab = tb.stab + 2 * nq;                     // lens m: rows 2m, 2m+1
    const float *gtab = tb.stab + (size_t)(2 * (1 + NL)) * nq; // light m

    const int base = blockIdx.x * a.pix_per_block;
    const int end = min(base + a.pix_per_block, a.npix);
    // this thread's flags: bit i = its i-th pixel has a ray inside a source Sersic's cusp zone,
    // (R/r_S)^2 < T2 of lensed_internal.h (refine.cu)
    uint32_t flags = 0, bit = 1;
#pragma unroll 1
    for (int ip = base + threadIdx.x; ip < end; ip += kTraceThreads, bit += bit) {
        const uint32_t rc = a.pix[ip];
        const int row = (int)(rc >> 16), col = (int)(rc & 0xffffu);
        const float jf = (float)col, rf = (float)row;
        float rmin[S::n_ss > 0 ? S::n_ss : 1];
#pragma unroll
        for (int i = 0; i < S::n_ss; ++i) rmin[i] = 3e38f;
        float rdummy = 0.0f;

        // frame origins of this pixel
        float lu[NL > 0 ? NL : 1], lv[NL > 0 ? NL : 1], gu[NPOS > 0 ? NPOS : 1], gv[NPOS > 0 ? NPOS : 1];
        if (S::n_shear) shear_origin(sder + S::lens_off4(0), jf, rf, a.cxh, a.cyh, lu[0], lv[0]);
#pragma unroll
        for (int i = 0; i < S::n_sie; ++i)
            sie_origin(sder + S::lens_off4(L_SIE + i), jf, rf, lu[L_SIE + i], lv[L_SIE + i]);
#pragma unroll
        for (int i = 0; i < S::n_sis + S::n_point; ++i)
            circular_origin(sder + S::lens_off4(L_SIS + i), jf, rf, lu[L_SIS + i], lv[L_SIS + i]);
#pragma unroll
        for (int i = 0; i < NPOS; ++i) light_origin(sder + S::light_off4(i), jf, rf, gu[i], gv[i]);
        if (S::direct && S::n_shear) {
#pragma unroll
            for (int i = 0; i < S::n_src; ++i) {              // sources come first among the lights
                const float4 M = sder[S::light_off4(i) + 1];
                gu[i] -= fmaf(M.x, lu[0], M.y * lv[0]);
                gv[i] -= fmaf(M.z, lu[0], M.w * lv[0]);
            }
        }

        // the origins are per-pixel values: an empty asm that "writes" them keeps ptxas from
        // recomputing them inside the ray loop to save registers (it did: +13 instructions per pass)
#pragma unroll
        for (int i = 0; i < NL; ++i) { asm volatile("" : "+f"(lu[i]), "+f"(lv[i])); }
#pragma unroll
        for (int i = 0; i < S::n_src; ++i) { asm volatile("" : "+f"(gu[i]), "+f"(gv[i])); }

        // foreground Sersics: moment expansion where it holds, else their own per-ray sum
        float fg = 0.0f;
#pragma unroll
        for (int i = 0; i < S::n_fs; ++i) {
            const float4 *d = sder + S::light_off4(G_FS + i);
            const float s0 = fmaf(gu[G_FS + i], gu[G_FS + i], gv[G_FS + i] * gv[G_FS + i]);
            const float4 rng = d[3];
            if (s0 >= rng.x && s0 <= rng.y) {
                fg += fg_expansion(d, tb.sfgx[i], gu[G_FS + i], gv[G_FS + i], s0, !(s0 >= rng.z && s0 <= rng.w));
            } else {
                f2 accf = bc(0.0f);
#pragma unroll 1
                for (int q0 = 0; q0 < nq; q0 += R) {
                    Rays<NP> rf_;
                    light_profile<NP, false, false, true>(d, gtab + (size_t)(2 * (G_FS + i)) * nq + q0,
                                                          gtab + (size_t)(2 * (G_FS + i) + 1) * nq + q0, gu[G_FS + i],
                                                          gv[G_FS + i], rf_, nullptr, rdummy);
                    f2 w[NP];
                    load_pairs<NP>(tb.sw + q0, w);
#pragma unroll
                    for (int k = 0; k < NP; ++k) accf = fma2(w[k], rf_.I[k], accf);
                }
                fg += lo2(accf) + hi2(accf);
            }
        }

        f2 acc = bc(0.0f);
#pragma unroll 1
        for (int q0 = 0; q0 < nq; q0 += R) {
            Rays<NP> r;
            if (S::direct) {
                // (ax, ay) are set by the SIE below
            } else if (S::n_shear) {
                lens_shear<NP, true>(ltab + q0, ltab + nq + q0, lu[0], lv[0], r);
            } else {
#pragma unroll
                for (int k = 0; k < NP; ++k) { r.ax[k] = bc(0.0f); r.ay[k] = bc(0.0f); }
            }
#pragma unroll
            for (int i = 0; i < S::n_sie; ++i) {
                const int m = L_SIE + i;
                lens_sie<NP, MODE, S::direct>(sder + S::lens_off4(m), ltab + (size_t)(2 * m) * nq + q0,
                                              ltab + (size_t)(2 * m + 1) * nq + q0, lu[m], lv[m], r);
            }
            // SIS / point mass: identity frame = slot 0
#pragma unroll
            for (int i = 0; i < S::n_sis; ++i) {
                const int m = L_SIS + i;
                lens_circular<NP, false>(sder + S::lens_off4(m), tb.stab + q0, tb.stab + nq + q0, lu[m], lv[m], r);
            }
#pragma unroll
            for (int i = 0; i < S::n_point; ++i) {
                const int m = L_PT + i;
                lens_circular<NP, true>(sder + S::lens_off4(m), tb.stab + q0, tb.stab + nq + q0, lu[m], lv[m], r);
            }
            if (NPOS - S::n_fs == 0) {                    // no light left in the ray loop
#pragma unroll
                for (int k = 0; k < NP; ++k) r.I[k] = bc(0.0f);
            }
            // foreground lights first: they do not wait for the deflection (foreground Sersics
            // are not in this loop: "foreground expansion" above)
#define LENSED_LIGHT(m, SRC, GAUSS, INIT)                                                                     \
    light_profile<NP, SRC, GAUSS, INIT>(sder + S::light_off4(m), gtab + (size_t)(2 * (m)) * nq + q0, \
                                        gtab + (size_t)(2 * (m) + 1) * nq + q0, gu[m], gv[m], r,              \
                                        (SRC) && S::direct ? tb.smat + (m) : nullptr,                         \
                                        (SRC) && !(GAUSS) ? rmin[(m) < S::n_ss ? (m) : 0] : rdummy)
            constexpr bool fg_first = S::n_fg > 0;
#pragma unroll
            for (int i = 0; i < S::n_fg; ++i) {
                if (i == 0) LENSED_LIGHT(G_FG + i, false, true, true);
                else LENSED_LIGHT(G_FG + i, false, true, false);
            }
#pragma unroll
            for (int i = 0; i < S::n_ss; ++i) {
                if (i == 0 && !fg_first) LENSED_LIGHT(i, true, false, true);
                else LENSED_LIGHT(i, true, false, false);
            }
#pragma unroll
            for (int i = 0; i < S::n_sg; ++i) {
                if (i == 0 && !fg_first && S::n_ss == 0) LENSED_LIGHT(G_SG + i, true, true, true);
                else LENSED_LIGHT(G_SG + i, true, true, false);
            }
#undef LENSED_LIGHT
            f2 w[NP];
            load_pairs<NP>(tb.sw + q0, w);
#pragma unroll
            for (int k = 0; k < NP; ++k) acc = fma2(w[k], r.I[k], acc);
        }
        store_pixel(a, Lb, row, col, ((lo2(acc) + hi2(acc)) + fg) + tb.sky);
#pragma unroll
        for (int i = 0; i < S::n_ss; ++i)
            if (rmin[i] < sder[S::light_off4(i) + 2].w) flags |= bit;
    }
    if (a.fixmask) a.fixmask[((size_t)vec * gridDim.x + blockIdx.x) * kTraceThreads + threadIdx.x] = flags;
}

// ---- pixel pairs ------------------------------------------------------------------------------
// The specialised tracers work on PAIRS OF PIXELS: a thread takes its list entries two at a time
// (ip, ip + 256) and a packed register pair holds the same rule point of both (trace_math.cuh
// "enter").  Against pairs of rule points of one pixel: (1) no rule is padded to an even number of
// points -- 9-, 25- and 49-point rules lose 10 %, 12 % and 2 % of padding; (2) the per-pixel
// arithmetic (frame origins, the foreground expansion, the final sums) is packed as well; (3) a
// table row is read once for two pixels, as scalars that enter as broadcast operands.  NP = rule
// points per pass, each pass a 16-byte-aligned stretch of NPP = 4 (NP <= 4) or 8 table entries
// (api.cu lays the rule out that way for these kernels: TraceArgs::quad / nq_pad as the static
// launcher sets them).
#ifndef LENSED_PIXEL_PAIRS
#define LENSED_PIXEL_PAIRS 1
#endif
#ifndef LENSED_PIPELINE
#define LENSED_PIPELINE 0          // tuning builds: deflection of the next pass beside the brightness of this one
#endif

__device__ __forceinline__ void keep(f2 &x) { asm volatile("" : "+l"(x.v)); }

// fg_expansion for two pixels at once (same expressions, packed; MUFU per half)
__device__ __forceinline__ f2 fg_expansion(const float4 *d, const FgMoments &m, f2 a, f2 b, f2 s0, bool full)
{
    const float4 c2 = d[2];                              // log2 I0, b_n log2 e, 1/(2n)
    const float c = c2.z;
    const f2 e = map2(mul2(map2(s0, [](float x) { return mufu_lg2(x); }), bc(c)), [](float x) { return mufu_ex2(x); });
    const f2 F = map2(fma2(e, bc(-c2.y), bc(c2.x)), [](float x) { return mufu_ex2(x); });
    const f2 is = map2(s0, [](float x) { return mufu_rcp(x); });
    const f2 h1 = mul2(mul2(e, bc(-(c2.y * 0.69314718056f) * c)), is);            // dh/ds = -b_n c s^(c-1)
    const f2 h2 = mul2(mul2(h1, bc(c - 1.0f)), is);
    const f2 h11 = mul2(h1, h1);
    const f2 aa = mul2(a, a), ab = mul2(a, b), bb = mul2(b, b);
    const f2 EL2 = mul2(fma2(aa, bc(m.S11), fma2(ab, bc(2.0f * m.S12), mul2(bb, bc(m.S22)))), bc(4.0f));
    if (!full) return fma2(F, fma2(h1, bc(m.S11 + m.S22), mul2(mul2(add2(h11, h2), bc(0.5f)), EL2)), F);
    const f2 h3 = mul2(mul2(h2, bc(c - 2.0f)), is), h4 = mul2(mul2(h3, bc(c - 3.0f)), is);
    const f2 F2 = add2(h11, h2);
    const f2 F3 = add2(mul2(h1, fma2(h2, bc(3.0f), h11)), h3);
    const f2 F4 = add2(fma2(h11, fma2(h2, bc(6.0f), h11), mul2(mul2(h2, h2), bc(3.0f))), fma2(mul2(h1, h3), bc(4.0f), h4));
    const float EQ = m.S11 + m.S22, EQ2 = m.T0 + 2.0f * m.T2 + m.T4;
    const f2 EL2Q = mul2(fma2(aa, bc(m.T0 + m.T2), fma2(ab, bc(2.0f * (m.T1 + m.T3)), mul2(bb, bc(m.T2 + m.T4)))), bc(4.0f));
    const f2 q1 = fma2(aa, bc(m.T0), fma2(ab, bc(4.0f * m.T1), mul2(bb, bc(6.0f * m.T2))));
    const f2 q2 = fma2(ab, bc(4.0f * m.T3), mul2(bb, bc(m.T4)));
    const f2 EL4 = mul2(fma2(aa, q1, mul2(bb, q2)), bc(16.0f));
    f2 corr = mul2(h1, bc(EQ));
    corr = fma2(mul2(F2, bc(0.5f)), add2(EL2, bc(EQ2)), corr);
    corr = fma2(mul2(F3, bc(0.5f)), EL2Q, corr);
    corr = fma2(mul2(F4, bc(1.0f / 24.0f)), EL4, corr);
    return fma2(F, corr, F);
}

template <int NP, class S, int MODE>
__device__ __forceinline__ void trace_pixel_pairs(const Program &prog, const TraceArgs &a, const TraceBlock &tb, float *Lb, int vec)
{
    constexpr int NPP = NP <= 4 ? 4 : 8;
    constexpr int NL = S::n_lens, NPOS = S::n_pos;
    constexpr int L_SIE = S::n_shear, L_SIS = L_SIE + S::n_sie, L_PT = L_SIS + S::n_sis;
    constexpr int G_SG = S::n_ss, G_FS = G_SG + S::n_sg, G_FG = G_FS + S::n_fs;
    const int nq = a.nq_pad;
    const float4 *sder = tb.sder;
    const float *ltab = tb.stab + 2 * nq;
    const float *gtab = tb.stab + (size_t)(2 * (1 + NL)) * nq;

    const int base = blockIdx.x * a.pix_per_block;
    const int end = min(base + a.pix_per_block, a.npix);
    // this thread's flags: bit i = its i-th pixel (list index base + 256 i + thread) has a ray inside a
    // source Sersic's cusp zone (refine.cu); one loop pass takes pixels 2n and 2n + 1
    uint32_t flags = 0, bit = 1;
#pragma unroll 1
    for (int ip = base + threadIdx.x; ip < end; ip += 2 * kTraceThreads, bit <<= 2) {
        const bool two = ip + kTraceThreads < end;           // the list is odd for this thread: second pixel = the first again
        const uint32_t rcA = a.pix[ip], rcB = a.pix[two ? ip + kTraceThreads : ip];
        const int rowA = (int)(rcA >> 16), colA = (int)(rcA & 0xffffu), rowB = (int)(rcB >> 16), colB = (int)(rcB & 0xffffu);
        const f2 jf = mk2((float)colA, (float)colB), rf = mk2((float)rowA, (float)rowB);
        float2 rmin[S::n_ss > 0 ? S::n_ss : 1];
#pragma unroll
        for (int i = 0; i < S::n_ss; ++i) rmin[i] = make_float2(3e38f, 3e38f);
        float2 rdummy = make_float2(0.0f, 0.0f);

        f2 lu[NL > 0 ? NL : 1], lv[NL > 0 ? NL : 1], gu[NPOS > 0 ? NPOS : 1], gv[NPOS > 0 ? NPOS : 1];
        if (S::n_shear) shear_origin(sder + S::lens_off4(0), jf, rf, a.cxh, a.cyh, lu[0], lv[0]);
#pragma unroll
        for (int i = 0; i < S::n_sie; ++i) sie_origin(sder + S::lens_off4(L_SIE + i), jf, rf, lu[L_SIE + i], lv[L_SIE + i]);
#pragma unroll
        for (int i = 0; i < S::n_sis + S::n_point; ++i)
            circular_origin(sder + S::lens_off4(L_SIS + i), jf, rf, lu[L_SIS + i], lv[L_SIS + i]);
#pragma unroll
        for (int i = 0; i < NPOS; ++i) light_origin(sder + S::light_off4(i), jf, rf, gu[i], gv[i]);
        if (S::direct && S::n_shear) {
#pragma unroll
            for (int i = 0; i < S::n_src; ++i) {              // sources come first among the lights
                const float4 M = sder[S::light_off4(i) + 1];
                gu[i] = fma2(lu[0], bc(-M.x), fma2(lv[0], bc(-M.y), gu[i]));
                gv[i] = fma2(lu[0], bc(-M.z), fma2(lv[0], bc(-M.w), gv[i]));
            }
        }
        // per-pixel values: keep ptxas from recomputing them inside the ray loop to save registers
#pragma unroll
        for (int i = 0; i < NL; ++i) { keep(lu[i]); keep(lv[i]); }
#pragma unroll
        for (int i = 0; i < S::n_src; ++i) { keep(gu[i]); keep(gv[i]); }

        // foreground Sersics: moment expansion where it holds for both pixels, else the per-ray sum
        f2 fg = bc(0.0f);
#pragma unroll
        for (int i = 0; i < S::n_fs; ++i) {
            const float4 *d = sder + S::light_off4(G_FS + i);
            const f2 s0 = fma2(gu[G_FS + i], gu[G_FS + i], mul2(gv[G_FS + i], gv[G_FS + i]));
            const float4 rng = d[3];
            const float sA = lo2(s0), sB = hi2(s0);
            if (sA >= rng.x && sA <= rng.y && sB >= rng.x && sB <= rng.y) {
                const bool full = !(sA >= rng.z && sA <= rng.w && sB >= rng.z && sB <= rng.w);
                fg = add2(fg, fg_expansion(d, tb.sfgx[i], gu[G_FS + i], gv[G_FS + i], s0, full));
            } else {
                f2 accf = bc(0.0f);
#pragma unroll 1
                for (int q0 = 0; q0 < nq; q0 += NPP) {
                    Rays<NP> rf_;
                    light_profile<NP, false, false, true>(d, gtab + (size_t)(2 * (G_FS + i)) * nq + q0,
                                                          gtab + (size_t)(2 * (G_FS + i) + 1) * nq + q0, gu[G_FS + i],
                                                          gv[G_FS + i], rf_, nullptr, rdummy);
                    f2 w[NP];
                    pass_weights<NP>(tb.sw + q0, s0, w);
#pragma unroll
                    for (int k = 0; k < NP; ++k) accf = fma2(w[k], rf_.I[k], accf);
                }
                fg = add2(fg, accf);
            }
        }

        f2 acc = bc(0.0f);
        // the two stages of a pass: deflection (FP32-pipe heavy) and brightness + rule sum (MUFU heavy)
        auto lenses = [&](int q0, Rays<NP> &r) {
            if (S::direct) {
                // (ax, ay) are set by the SIE below
            } else if (S::n_shear) {
                lens_shear<NP, true>(ltab + q0, ltab + nq + q0, lu[0], lv[0], r);
            } else {
#pragma unroll
                for (int k = 0; k < NP; ++k) { r.ax[k] = bc(0.0f); r.ay[k] = bc(0.0f); }
            }
#pragma unroll
            for (int i = 0; i < S::n_sie; ++i) {
                const int m = L_SIE + i;
                lens_sie<NP, MODE, S::direct>(sder + S::lens_off4(m), ltab + (size_t)(2 * m) * nq + q0,
                                              ltab + (size_t)(2 * m + 1) * nq + q0, lu[m], lv[m], r);
            }
#pragma unroll
            for (int i = 0; i < S::n_sis; ++i) {
                const int m = L_SIS + i;
                lens_circular<NP, false>(sder + S::lens_off4(m), tb.stab + q0, tb.stab + nq + q0, lu[m], lv[m], r);
            }
#pragma unroll
            for (int i = 0; i < S::n_point; ++i) {
                const int m = L_PT + i;
                lens_circular<NP, true>(sder + S::lens_off4(m), tb.stab + q0, tb.stab + nq + q0, lu[m], lv[m], r);
            }
        };
        auto lights = [&](int q0, Rays<NP> &r) {
            if (NPOS - S::n_fs == 0) {
#pragma unroll
                for (int k = 0; k < NP; ++k) r.I[k] = bc(0.0f);
            }
#define LENSED_LIGHT(m, SRC, GAUSS, INIT)                                                                 \
    do {                                                                                                  \
        if constexpr ((SRC) && !(GAUSS))                                                                  \
            light_profile<NP, SRC, GAUSS, INIT>(sder + S::light_off4(m), gtab + (size_t)(2 * (m)) * nq + q0,      \
                                                gtab + (size_t)(2 * (m) + 1) * nq + q0, gu[m], gv[m], r,          \
                                                S::direct ? tb.smat + (m) : nullptr, rmin[(m) < S::n_ss ? (m) : 0]); \
        else                                                                                              \
            light_profile<NP, SRC, GAUSS, INIT>(sder + S::light_off4(m), gtab + (size_t)(2 * (m)) * nq + q0,      \
                                                gtab + (size_t)(2 * (m) + 1) * nq + q0, gu[m], gv[m], r,          \
                                                (SRC) && S::direct ? tb.smat + (m) : nullptr, rdummy);    \
    } while (0)
            constexpr bool fg_first = S::n_fg > 0;
#pragma unroll
            for (int i = 0; i < S::n_fg; ++i) {
                if (i == 0) LENSED_LIGHT(G_FG + i, false, true, true);
                else LENSED_LIGHT(G_FG + i, false, true, false);
            }
#pragma unroll
            for (int i = 0; i < S::n_ss; ++i) {
                if (i == 0 && !fg_first) LENSED_LIGHT(i, true, false, true);
                else LENSED_LIGHT(i, true, false, false);
            }
#pragma unroll
            for (int i = 0; i < S::n_sg; ++i) {
                if (i == 0 && !fg_first && S::n_ss == 0) LENSED_LIGHT(G_SG + i, true, true, true);
                else LENSED_LIGHT(G_SG + i, true, true, false);
            }
#undef LENSED_LIGHT
            f2 w[NP];
            pass_weights<NP>(tb.sw + q0, acc, w);
#pragma unroll
            for (int k = 0; k < NP; ++k) acc = fma2(w[k], r.I[k], acc);
        };
#if LENSED_PIPELINE
        if constexpr (S::direct) {
            // software pipeline: the SIE of pass p + 1 sits in the same loop body as the light profiles
            // of pass p, so every warp issues a steady mix for both pipes instead of alternating
            // between an FP32-heavy and a MUFU-heavy phase
            Rays<NP> r, n;
            lenses(0, n);
#pragma unroll 1
            for (int q0 = 0; q0 + NPP < nq; q0 += NPP) {
#pragma unroll
                for (int k = 0; k < NP; ++k) { r.ax[k] = n.ax[k]; r.ay[k] = n.ay[k]; }
                lenses(q0 + NPP, n);
                lights(q0, r);
            }
#pragma unroll
            for (int k = 0; k < NP; ++k) { r.ax[k] = n.ax[k]; r.ay[k] = n.ay[k]; }
            lights(nq - NPP, r);
        } else
#endif
        {
#pragma unroll 1
            for (int q0 = 0; q0 < nq; q0 += NPP) {
                Rays<NP> r;
                lenses(q0, r);
                lights(q0, r);
            }
        }
        const f2 total = add2(add2(acc, fg), bc(tb.sky));
        store_pixel(a, Lb, rowA, colA, lo2(total));
        if (two) store_pixel(a, Lb, rowB, colB, hi2(total));
#pragma unroll
        for (int i = 0; i < S::n_ss; ++i) {
            const float T2 = sder[S::light_off4(i) + 2].w;
            if (rmin[i].x < T2) flags |= bit;
            if (two && rmin[i].y < T2) flags |= bit << 1;
        }
    }
    if (a.fixmask) a.fixmask[((size_t)vec * gridDim.x + blockIdx.x) * kTraceThreads + threadIdx.x] = flags;
}

// MINB = resident blocks per SM the register budget is cut for (3 -> 80 registers, 2 -> 128):
// chosen per signature where it was measured (profiles/r1f.md)
template <int NP, class S, int MINB>
__global__ void __launch_bounds__(kTraceThreads, MINB * (256 / kTraceThreads)) trace_static_kernel(Program prog, TraceArgs a)
{
    extern __shared__ float4 smem4[];
    const int vec = trace_vector(a);
    const TraceBlock tb = trace_prologue(prog, a, smem4, vec);
    if (!tb.valid) {
        if (a.fixmask) a.fixmask[((size_t)vec * gridDim.x + blockIdx.x) * kTraceThreads + threadIdx.x] = 0;
        return;
    }
    if constexpr (S::direct || S::n_fs > 0) {
        const int nq = a.nq_pad;
        if constexpr (S::n_fs > 0) {
            // rule moments in the frame of every foreground Sersic ("foreground expansion"), from the
            // table the per-ray path reads (padding entries have zero weight): one warp per component,
            // the rule points across its lanes, a fixed shuffle tree
            const int lane = threadIdx.x & 31;
            for (int i = threadIdx.x >> 5; i < S::n_fs; i += kTraceThreads / 32) {
                const int m = S::n_ss + S::n_sg + i;
                const float *tu = tb.stab + (size_t)(2 * (1 + S::n_lens + m)) * nq, *tv = tu + nq;
                float v[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
                for (int k = lane; k < nq; k += 32) {
                    const float w = tb.sw[k], d1 = tu[k], d2 = tv[k], w11 = w * d1 * d1, w12 = w * d1 * d2, w22 = w * d2 * d2;
                    v[0] += w11; v[1] += w12; v[2] += w22;
                    v[3] += w11 * d1 * d1; v[4] += w11 * d1 * d2; v[5] += w11 * d2 * d2; v[6] += w12 * d2 * d2; v[7] += w22 * d2 * d2;
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1)
#pragma unroll
                    for (int e = 0; e < 8; ++e) v[e] += __shfl_xor_sync(0xffffffffu, v[e], o);
                if (lane == 0) tb.sfgx[i] = FgMoments{v[0], v[1], v[2], v[3], v[4], v[5], v[6], v[7]};
            }
        }
        if constexpr (S::direct) {
            // source tables lose M Gamma (rule offset); B per source (TraceSig "direct frames").  The
            // moments above read foreground tables only, so both share one barrier.
            float *stab = const_cast<float *>(tb.stab);
            float *gtab = stab + (size_t)(2 * (1 + S::n_lens)) * nq;
            if (S::n_shear) {
                for (int i = threadIdx.x; i < S::n_src * nq; i += kTraceThreads) {
                    const int m = i / nq, k = i - m * nq;
                    const float4 M = tb.sder[S::light_off4(m) + 1];
                    const float su = stab[2 * nq + k], sv = stab[3 * nq + k];     // shear = lens 0
                    gtab[(size_t)(2 * m) * nq + k] -= fmaf(M.x, su, M.y * sv);
                    gtab[(size_t)(2 * m + 1) * nq + k] -= fmaf(M.z, su, M.w * sv);
                }
            }
            if (threadIdx.x < S::n_src) {
                const float4 M = tb.sder[S::light_off4(threadIdx.x) + 1];
                const float4 c2 = tb.sder[S::lens_off4(S::n_shear) + 2];          // (cs A, sn A, cs A l, -sn A l)
                tb.smat[threadIdx.x] = make_float4(fmaf(M.x, c2.x, M.y * c2.y), fmaf(M.x, c2.w, M.y * c2.z),
                                                   fmaf(M.z, c2.x, M.w * c2.y), fmaf(M.z, c2.w, M.w * c2.z));
            }
        }
        __syncthreads();
    }
    float *Lb = a.L + (size_t)vec * a.l_stride;
#if LENSED_PIXEL_PAIRS
#define LENSED_TRACE_BODY trace_pixel_pairs
#else
#define LENSED_TRACE_BODY trace_pixels
#endif
    if constexpr (S::n_sie == 0) {
        LENSED_TRACE_BODY<NP, S, 0>(prog, a, tb, Lb, vec);
    } else {
        switch ((int)tb.sder[0].y) {              // SieMode of the vector (prep.cu), block-uniform
        case 0: LENSED_TRACE_BODY<NP, S, 0>(prog, a, tb, Lb, vec); break;
        case 1: LENSED_TRACE_BODY<NP, S, 1>(prog, a, tb, Lb, vec); break;
        case 2: LENSED_TRACE_BODY<NP, S, 2>(prog, a, tb, Lb, vec); break;
        case 3: LENSED_TRACE_BODY<NP, S, 3>(prog, a, tb, Lb, vec); break;
        case 4: LENSED_TRACE_BODY<NP, S, 4>(prog, a, tb, Lb, vec); break;
        default: LENSED_TRACE_BODY<NP, S, 5>(prog, a, tb, Lb, vec); break;
        }
    }
#undef LENSED_TRACE_BODY
}

#ifndef __CUDACC_RTC__
// Pixel pairs: NP = rule points per pass (TraceArgs::np_pp, from trace_pick_np), on the rule laid out
// in passes (quad_pp, nq_pp).  Ray pairs (LENSED_PIXEL_PAIRS=0): R = 2 NP rays per register block.
template <class S, int MINB>
cudaError_t launch_trace_static(const Program &prog, const TraceArgs &a0, int R, int nvec, cudaStream_t st)
{
#if LENSED_PIXEL_PAIRS
    TraceArgs a = a0;
    a.quad = a0.quad_pp;
    a.nq_pad = a0.nq_pp;
    switch (a0.np_pp) {
    case 2: return launch_trace_kernel(trace_static_kernel<2, S, MINB>, prog, a, nvec, st);
    case 3: return launch_trace_kernel(trace_static_kernel<3, S, MINB>, prog, a, nvec, st);
    case 4: return launch_trace_kernel(trace_static_kernel<4, S, MINB>, prog, a, nvec, st);
    case 5: return launch_trace_kernel(trace_static_kernel<5, S, MINB>, prog, a, nvec, st);
    default: return cudaErrorInvalidValue;
    }
#else
    const TraceArgs &a = a0;
    switch (R) {
    case 2: return launch_trace_kernel(trace_static_kernel<1, S, MINB>, prog, a, nvec, st);
    case 4: return launch_trace_kernel(trace_static_kernel<2, S, MINB>, prog, a, nvec, st);
    case 6: return launch_trace_kernel(trace_static_kernel<3, S, MINB>, prog, a, nvec, st);
    case 8: return launch_trace_kernel(trace_static_kernel<4, S, MINB>, prog, a, nvec, st);
    case 10: return launch_trace_kernel(trace_static_kernel<5, S, MINB>, prog, a, nvec, st);
    default: return cudaErrorInvalidValue;
    }
#endif
}

// Defines  bool NAME(counts, prog, args, R, nvec, stream, &err): false if the signature does
// not match the list's per-kind counts, else launches and sets err (a NULL err only asks).
// One per .cu file, so that the signatures compile in parallel (build.py).
#define LENSED_DEFINE_STATIC_TRACER(NAME, MINB, ...)                                                         \
    bool NAME(const int (&counts)[K_COUNT], const Program &prog, const TraceArgs &a, int R, int nvec,   \
              cudaStream_t st, cudaError_t *err)                                                        \
    {                                                                                                   \
        using S = TraceSig<__VA_ARGS__>;                                                                \
        if (!S::matches(counts)) return false;                                                          \
        if (err) *err = launch_trace_static<S, MINB>(prog, a, R, nvec, st);                             \
        return true;                                                                                    \
    }

#endif  // !__CUDACC_RTC__

}  // namespace lensed
