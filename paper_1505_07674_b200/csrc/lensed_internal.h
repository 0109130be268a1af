// lensed_internal.h -- shared declarations of the CUDA path (host side + kernels).
// Not part of the public ABI (include/lensed.h is); shares nothing with oracle/.
//
// Units inside the kernels: PIXELS.  The prep kernel divides every length by the pixel
// scale, so the ray tracer never multiplies by s; deflections are linear in that scaling
// for every lens here (SIS, SIE, point mass: alpha(lambda x; lambda b) = lambda alpha(x; b);
// shear is linear in x).
#pragma once
#ifdef __CUDACC_RTC__              // compiled at run time by NVRTC (jit.cu): no host headers, kernels only
typedef unsigned char uint8_t;
typedef unsigned short uint16_t;
typedef unsigned int uint32_t;
#else
#include <cuda_runtime.h>
#include <stdint.h>
#endif

struct lensed_handle;

namespace lensed {

// ---- derived-constant blocks (floats per model, each a multiple of 4 for LDS.128) ------
// Every positioned component starts with its centre split as (integer pixel, fraction):
//   c0 = (cxi, cxf, cyi, cyf),   pixel-frame centre = cxi + cxf, |cxf| <= 1/2,
// so that the thread forms (float(j) - cxi) - cxf: an exact integer difference followed
// by ONE rounding at the magnitude of the component-relative offset.
//
//  SIS    [c0][b, 0, 0, 0]                                              8
//  SIE    [c0][cos, sin, q^2, q'][cos A, sin A, cos A l, -sin A l]      12
//         A = b sqrt(q)/q' with q' floored at 1e-4, l = ln(2)/2 (trace.cu lens_sie)
//  POINT  [c0][thetaE^2, 0, 0, 0]                                       8
//  SHEAR  [g1, g2, 0, 0]                                                4
//  SERSIC [c0][a1, a2, a3, a4][log2 I0, b_n*log2(e), 1/(2n), T2][s_lo, s_hi, s_lo2, s_hi2]   16
//         T2 = squared scaled radius inside which a source's pixels are refined in FP64
//         (prep.cu "refinement threshold"; 0 for foregrounds and n <= 1);
//         [s_lo, s_hi] (foregrounds): range of the squared scaled radius of a pixel centre in
//         which the pixel integral of the profile is taken from its moment expansion instead
//         of the per-ray sum (trace_static.cuh "foreground expansion"; empty range = never);
//         inside [s_lo2, s_hi2] its second-order terms are enough
//         (u', v') = (a1 dx + a2 dy, a3 dx + a4 dy) = rotated, q-stretched offset / r_S,
//         so that u'^2 + v'^2 = (R / r_S)^2 with R of PAPER.md:250 eq. 23
//  GAUSS  [c0][a1, a2, a3, a4][log2 I0, log2(e)/2, 0, 0]                12   (offset / sigma)
//  SKY    [level, 0, 0, 0]                                              4
//
// derived64 [B][n_models][kD64PerModel] doubles, LIST order, lengths in pixels, centres in
// pixel-index coordinates (column, row) -- the unrounded constants refine.cu re-traces with:
//  SIS cx, cy, b | SIE cx, cy, cos, sin, q, b | POINT cx, cy, thetaE^2 | SHEAR g1, g2
//  SERSIC cx, cy, cos, sin, q, r_S, 1/n, b_n, ln I0 | GAUSS cx, cy, cos, sin, q, sigma, ln I0 | SKY level
//
// Block 0 of every vector is the header [valid, SIE mode, 0, 0]; the mode (trace_math.cuh
// "SIE") is the most general one any SIE of the vector needs, 0 without an SIE.
enum Kind : int {
    K_SIS = 0, K_SIE = 1, K_POINT = 2, K_SHEAR = 3,
    K_SRC_SERSIC = 4, K_SRC_GAUSS = 5, K_FG_SERSIC = 6, K_FG_GAUSS = 7, K_SKY = 8,
    K_COUNT = 9
};

// SIE mode from the axis ratio (thresholds on q^2; table in trace_math.cuh)
__host__ __device__ inline int sie_mode(double q)
{
    const double q2 = q * q;
    return q2 >= 0.84 ? 0 : q2 >= 0.64 ? 1 : q2 >= 0.5 ? 2 : q2 >= 1.0 / 3.0 ? 3 : q2 >= 0.25 ? 4 : 5;
}

constexpr int kMaxModels = 32;
constexpr int kMaxQuad = 256;
constexpr int kMaxPsf = 63;
constexpr int kHeaderFloats = 4;
constexpr int kD64PerModel = 12;
constexpr int kTapPoolPairs = 7680;   // conv.cu c_taps: 60 KB of constant bank shared by the live handles

__host__ __device__ constexpr int kind_num_params(int k) {
    return k == K_SIS ? 3 : k == K_SIE ? 5 : k == K_POINT ? 3 : k == K_SHEAR ? 2
         : (k == K_SRC_SERSIC || k == K_FG_SERSIC) ? 7
         : (k == K_SRC_GAUSS || k == K_FG_GAUSS) ? 6 : k == K_SKY ? 1 : -1;
}
__host__ __device__ constexpr int kind_num_derived(int k) {
    return k == K_SIS ? 8 : k == K_SIE ? 12 : k == K_POINT ? 8 : k == K_SHEAR ? 4
         : (k == K_SRC_SERSIC || k == K_FG_SERSIC) ? 16 : (k == K_SRC_GAUSS || k == K_FG_GAUSS) ? 12
         : k == K_SKY ? 4 : -1;
}

// The model list compiled to two flat programs (lenses first, then lights); passed to the
// kernels by value, i.e. it sits in the constant bank and is read with uniform loads.
struct Program {
    int n_models;                  // list order (prep kernel)
    int n_lens, n_light;
    int P, D;                      // floats per parameter vector / per derived vector
    uint8_t kind[kMaxModels];      // list order
    uint16_t par_off[kMaxModels];  // list order: offset into the parameter vector
    uint16_t der_off[kMaxModels];  // list order: offset into the derived vector
    uint8_t lens_kind[kMaxModels];
    uint16_t lens_off[kMaxModels];
    uint8_t light_kind[kMaxModels];   // K_SRC_* / K_FG_* / K_SKY
    uint16_t light_off[kMaxModels];
};

struct PrepArgs {
    const float *params;   // [B][P]
    float *derived;        // [B][D]
    double *derived64;     // [B][n_models][kD64PerModel]
    int B;
    double refine_gain;    // scales the refinement threshold G (1 = default; prep.cu)
    double fgx_tau;        // foreground expansion: largest expansion parameter tau (0 = off; prep.cu)
    double rule_radius;    // largest distance of a rule point from the pixel centre, pixels
    double scale, zp;      // arcsec per pixel, magnitude zero point
    double cxh, cyh;       // (W-1)/2, (H-1)/2
};

struct TraceArgs {
    const float *derived;  // [.][D], already offset to the chunk's first vector
    const int *order;      // [nvec] or NULL: block row y works on vector order[y] of the chunk -- the chunk's
                           // vectors sorted by SIE mode (prep.cu order_kernel), so that the blocks resident at
                           // one time run the same specialised code path (instruction cache)
    const uint32_t *pix;   // [npix] packed (row << 16) | column
    const float4 *quad;    // [nq_pad] (xi, eta, w, w - w'), zero-weight padding up to a multiple of R (even);
                           // w' = embedded rule of lensed_set_error_rule (0 before it is set)
    const float4 *quad_pp; // the same rule laid out for the specialised tracers' pixel pairs: passes of np_pp
                           // points, each padded with zero-weight entries to 4 (np_pp <= 4) or 8 entries
    int nq_pp, np_pp;      // entries of quad_pp; rule points per pass (trace_pick_np)
    float *err;            // [.][H*W] quadrature error estimates instead of L (trace.cu ERR), or NULL
    uint32_t *fixmask;     // [nvec][blocks per vector][256] or NULL: per tracer thread, bit i = its i-th
                           // pixel (list index block base + 256 i + thread) wants the FP64 refinement (refine.cu)
    float *L;              // [.][Hp*Wp], chunk-local PADDED frames: pixel (i, j) at (i + py, j + px),
                           // border pixels replicated into the pad (conv.cu "Input")
    long long l_stride;    // Hp*Wp
    int npix, nq_pad;
    int H, W, Wp, px, py;
    int pix_per_block;     // pixels of the list one block walks (a multiple of 256, at most 8192)
    float cxh, cyh;
};

struct RefineArgs {
    TraceArgs t;               // the launch whose flags are refined (pix, quad, L, fixmask, geometry)
    const double *derived64;   // [nvec][n_models][kD64PerModel], offset to the chunk's first vector
    const float *derived;      // [nvec][D] (validity is not needed: invalid vectors have no flags)
    unsigned long long *count; // refined pixels, accumulated (statistic) or NULL
    uint2 *queue;              // [queue_cap] (vector, pixel-list index) between the two passes
    unsigned *queue_count;     // entries requested (may exceed queue_cap)
    int queue_cap;
    int nvec, n_blocks;        // grid of that launch: vectors, blocks per vector
    int n_quad;                // unpadded rule length
};

struct ConvArgs {
    const float *Lp;       // [nb][Hp*Wp] chunk-local padded unconvolved images (TraceArgs::L)
    const float *image;    // [H*W] d
    const float *wmask;    // [H*W] w_i, 0 where masked
    const uint32_t *tiles; // [n_tiles] packed (tile row << 16) | tile column of the active tiles; for the strip shape
                           // (first pixel row << 16) | first pixel column of each strip (api.cu strip_list)
    double *partial;       // [nb][n_tiles] chunk-local chi-square partials   (loglike)
    float *model;          // [nb][H*W] chunk-local output                    (render)
    const float *derived;  // [nb][D] chunk-local (valid flag)                (render)
    long long lp_stride;   // Hp*Wp
    int D;
    int H, W, Wp, KH, KW, NC, n_tiles;
    int ox, oy;            // image coordinates of tile (0, 0); ox is a multiple of 4
    int nb;                // vectors in this launch
    const unsigned long long *gtaps;   // the handle's tap pairs in global memory when the constant pool was
                           // full (then tap_off = 0), else NULL
    int shape;             // 1 = 256 threads, 64 x 128 tiles; 0 = 128 threads, 64 x 64 tiles; 2 = independent
                           // warps on 16 x 64 strips (conv.cu)
    int tap_off;           // first tap pair of this handle in c_taps: Q[j][c][k] at tap_off + (j NC + c) 4 + k,
                           // Q[j][c][k] = (G[j][4c+k], G[j-1][4c+k]), j = 0..KH, G = flipped normalised PSF
    int n_stages;          // input-tile buffers in shared memory (set by launch_conv)
};

struct FinalArgs {
    const double *partial; // [B][n_tiles]
    const float *derived;  // [B][D]
    float *logl;           // [B]
    int B, n_tiles, D;
};

#ifndef __CUDACC_RTC__
// launchers (each returns the cudaGetLastError of its launch)
cudaError_t launch_prep(const Program &prog, const PrepArgs &a, cudaStream_t st);
// order[c * Bc + i] = index within chunk c of its i-th vector by (SIE mode, index); invalid vectors last
cudaError_t launch_order(const float *derived, int D, int B, int Bc, int *order, cudaStream_t st);
// allow_static: use the compile-time-specialised kernel when the list has one (trace.cu)
struct JitTracer;
// jit: the run-time compiled tracer of a list without a built-in signature (jit.cu) or NULL
cudaError_t launch_trace(const Program &prog, const TraceArgs &a, int R, int nvec, bool allow_static, const JitTracer *jit,
                         cudaStream_t st);
inline int trace_blocks_per_vector(const TraceArgs &a) { return (a.npix + a.pix_per_block - 1) / a.pix_per_block; }
cudaError_t launch_refine(const Program &prog, const RefineArgs &a, int n_sm, cudaStream_t st);
bool trace_has_static(const Program &prog);
cudaError_t launch_conv(ConvArgs a, const void *tensor_map, bool render, int n_sm, cudaStream_t st);
cudaError_t conv_make_tensor_map(void *out, const float *L, int Wp, int Hp, long long n_frames, int KH, int NC, int shape);
cudaError_t conv_upload_taps(const float *pairs, int n_pairs, int pool_offset);
void conv_padded_shape(int rows, int cols, int KH, int NC, int *Hp, int *Wp);
cudaError_t launch_final(const FinalArgs &a, cudaStream_t st);
// deflect.cu: y = x - sum alpha for K points per vector / in place for the listed sources' (x, y)
cudaError_t launch_deflect(const Program &prog, const float *params, int B, const float *xy, int K, float *out,
                           cudaStream_t st);
cudaError_t launch_image_plane_prior(const Program &prog, const int *par_offs, int n_src, float *params, int B,
                                     cudaStream_t st);
cudaError_t conv_setup();                 // one-time function attributes
int trace_pick_R(int n_quad);             // rays per register block for an n_quad-point rule (ray pairs)
int trace_pick_np(int n_quad);            // rule points per pass for the pixel-pair tracers
size_t trace_smem_bytes(const Program &prog, int nq_pad);
// shape: 0 narrow (128 threads, 64 x 64 tiles, 2 blocks per SM), 1 wide (256 threads, 64 x 128), 2 strip
// (8 independent warps, 16 x 64 strips)
void conv_tile_shape(int shape, int *tile_w, int *tile_h);
size_t conv_smem_bytes(int KH, int NC, bool render, int shape);
bool conv_shape_fits(int KH, int NC, int shape);
int conv_num_stages(int KH, int NC, bool render, int shape);   // input-tile buffers per block (2 = double buffered)
cudaError_t run_fma_peak(int iters, double *tflops);
cudaError_t run_issue_probe(int kind, int n_extra, int warps, double *cycles_per_body);

// for the clients of the handle outside api.cu (nested.cu): error text on the handle, its device
int handle_fail(::lensed_handle *h, int status, const char *fmt, ...);
int handle_device(const ::lensed_handle *h);
#endif  // !__CUDACC_RTC__

}  // namespace lensed
