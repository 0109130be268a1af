/*
 * lensed_tune.h -- measurement, tuning and test hooks of liblensed_b200.so.
 *
 * include/lensed.h is the method: the calls that follow the paper's statement of the problem.
 * This header holds everything else the library exports: per-kernel timing for bench.py, the
 * knobs behind the design decisions recorded in DESIGN.md (refinement gain, foreground expansion,
 * chunk size, convolution shape, tracer selection), the hooks the tests use to force the rarely
 * taken paths, and two micro-benchmarks.  None of them changes what the method computes beyond
 * rounding (the tests compare the variants); a sampler never needs this header.
 *
 * Environment variables the library reads (all optional, all read at lensed_create or at the
 * first call; they select between kernels that compute the same thing):
 *   LENSED_JIT=0            do not specialise the tracer at run time: lists without a built-in
 *                           signature run the interpreting tracer
 *   LENSED_NO_BUILTIN=1     ignore the built-in signatures (every list goes through the run-time
 *                           specialisation: bench.py's comparison of the two)
 *   LENSED_STRIP_WARPS=n    independent warps per SM of the strip convolution (default 8)
 * The remaining LENSED_* names in csrc/ are compile-time defines of tuning builds
 * (paper_1505_07674_b200/build.py `defines=`), not environment variables.
 */
#ifndef LENSED_TUNE_H
#define LENSED_TUNE_H

#include "lensed.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * Instrumentation (measurement only; never changes results).
 * lensed_set_profiling(h, 1) brackets every kernel the library launches with CUDA
 * events on the launching stream.  lensed_get_profile synchronises those events and
 * returns, since the last lensed_reset_profile: milliseconds and launch counts of the
 * parameter-prep, ray-trace, FP64-refinement, convolution(+chi-square) and final-reduction
 * kernels as ms[5] / launches[5] (host arrays, either may be NULL).  Launch counts are kept
 * even with profiling off (ms are then 0).  lensed_reset_profile synchronises the device.  */
lensed_status lensed_set_profiling(lensed_handle *h, int on);
lensed_status lensed_get_profile(lensed_handle *h, double *ms, long long *launches);
lensed_status lensed_reset_profile(lensed_handle *h);

/*
 * FP64 refinement of cusp pixels.  FP32 ray positions carry ~1e-6 pixel of rounding noise
 * (y = x - alpha with |alpha| of tens of pixels, eq. 1); near the centre of a
 * compact Sersic source of high index (the paper's prior reaches n = 8) the
 * profile's logarithmic slope per pixel is large enough to turn that into more than 1e-5 in the
 * pixel -- and, those being the brightest pixels, in logL.  The ray tracer therefore flags the
 * pixels that have a ray where a source Sersic's slope  d ln I / dx  exceeds
 *   G = gain * 200 / max(deflection scale in pixels, 25)      per pixel
 * (deflection scale = sum of the lenses' Einstein radii + shear * image half-diagonal), and a
 * second kernel re-traces those pixels -- all rule points, all components -- in double
 * precision before the convolution.  Typically 1-20 pixels per vector.
 * lensed_set_refine: gain = 1 is the default; larger = fewer pixels refined; gain <= 0 turns
 * the refinement off (plain FP32 everywhere).  EINVAL for NaN.
 * lensed_get_refined: pixels refined since the last lensed_reset_profile (synchronises).    */
lensed_status lensed_set_refine(lensed_handle *h, double gain);
lensed_status lensed_get_refined(lensed_handle *h, long long *pixels);

/* Test hook standing in for an uninitialised-read checker.  The unconvolved images live in padded
 * frames of handle-owned scratch: cells of the pad that no border pixel
 * clamps to, and pixels outside the traced set of a masked image, are never written by the
 * tracer; the convolution reads some of them, but only under structurally zero taps or for
 * outputs it discards.  lensed_debug_fill_frames overwrites EVERY cell of the frames the handle
 * holds now with `value` (finite: 0 x value must stay 0); a later call on the same batch size must
 * return bitwise what it returned before -- if it does not, a never-written cell reaches a result.
 * Synchronises the device.  EINVAL for NULL or a non-finite value.                              */
lensed_status lensed_debug_fill_frames(lensed_handle *h, float value);

/*
 * Foreground expansion.  A foreground Sersic component is evaluated at the image-plane points
 * themselves (eq. 2), where it is smooth on the scale of a pixel except around its
 * centre.  The specialised tracers therefore take its pixel integral (eq. 14: the
 * rule sum over the pixel's points) from the Taylor expansion of the profile about the pixel
 * centre to fourth order in the rule offsets, with the rule's own second and fourth moments -- it
 * reproduces the rule sum, not the exact integral -- wherever the expansion parameter
 *   tau = max((b_n/n) (R/r_S)^(1/n), 1) * (rule radius) / (sqrt(q) R)
 * is at most `tau`; the error is below 0.016 tau^6 (2e-7 at the default 0.15), two orders under
 * the FP32 noise of a pixel sum.  Pixels closer to the component's centre take the per-ray sum,
 * as do all pixels when the rule is not symmetric (odd moments), with the interpreting tracer,
 * and with tau = 0.  lensed_set_fg_expansion: 0 <= tau <= 0.5, EINVAL otherwise.             */
lensed_status lensed_set_fg_expansion(lensed_handle *h, double tau);

/* Tuning knob: bytes of device scratch the unconvolved images L[b] of one batch chunk
 * may take (default 1 GiB: the buffer costs ~3.5 bytes of traffic per 3500 flops, so
 * launches are made long rather than L2-resident).  One vector
 * takes lensed_frame_bytes(h): its image in a frame padded by the PSF half-widths and
 * rounded up to whole convolution tiles.  EINVAL if bytes < one frame.
 * lensed_frame_bytes: -1 for NULL.                                                      */
lensed_status lensed_set_chunk_bytes(lensed_handle *h, long long bytes);
long long lensed_frame_bytes(const lensed_handle *h);

/* Convolution shape.  The convolution exists in four shapes (same per-pixel arithmetic):
 *   3 "half"    as "strip", on 16 x 32 strips with each half-warp on its own parameter vector:
 *               hugs a mask closer still and moves two vectors per tensor copy: the strip shape
 *               lensed_create picks
 *   2 "strip"   one block of 8 INDEPENDENT warps per SM, each on its own 16 x 64 output strip with
 *               its own shared-memory stage: nothing is lost at block barriers, masked images skip
 *               whole strips; needs 8 stages of (16 + psf_h - 1) x (64 + 4 ceil(psf_w / 4)) floats
 *               (PSFs up to about 37 rows)
 *   1 "wide"    256 threads on 64 x 128 output tiles, one block per SM: any PSF
 *   0 "narrow"  128 threads on 64 x 64 tiles, two blocks per SM: small or masked images
 * lensed_create picks one (strips for PSFs up to 23 x 23, and where a mask makes the strip list
 * compute at least 15 % fewer pixels; else wide, or narrow on the same 15 % rule); lensed_set_conv_shape(h, shape) forces one (it
 * rebuilds the tile lists and the frame layout and synchronises the device; EINVAL for another
 * value, LENSED_EUNSUPPORTED if the PSF is too large for that shape's shared memory).
 * lensed_get_conv_shape: 3 / 2 / 1 / 0, -1 for NULL.  Rendered pixels do not depend on the shape at
 * all; logL only through the order in which the per-tile chi-square partials are summed.
 *
 * PSF taps.  The taps of a handle normally sit in a 60 KB pool of constant memory shared by
 * the live handles of a device ((psf_h + 1) * 4 ceil(psf_w / 4) * 8 bytes each: 8 KB for 31 x 31,
 * 32 KB for 63 x 63).  A handle created when the pool is full keeps its taps in global memory
 * and runs a variant of the convolution that reads them from there (same results, somewhat
 * slower); lensed_uses_global_taps tells (1 / 0, -1 for NULL).
 * lensed_debug_force_global_taps(1) makes every later lensed_create take that path (tests).   */
lensed_status lensed_set_conv_shape(lensed_handle *h, int shape);
int lensed_get_conv_shape(const lensed_handle *h);
int lensed_uses_global_taps(const lensed_handle *h);
void lensed_debug_force_global_taps(int on);

/* Tracer selection.  The ray tracer exists as one kernel that interprets any model list and as
 * kernels SPECIALISED for one list each (same arithmetic, straight-line code; a list matches by
 * its per-kind counts, sky components aside).  Nine signatures are built in (SIS + Gaussian
 * source; SIE + shear + 1 or 2 Sersic sources + Sersic lens light; 2 SIE + point mass + shear + 2
 * Sersic + 1 Gaussian source + Sersic lens light; SIE + Sersic source with / without Sersic lens
 * light; SIE + shear + Sersic source; SIS + Sersic source; 2 SIE + 2 Sersic sources + 3 Sersic
 * foregrounds).  For any other list lensed_create compiles the specialised kernel at run time
 * (NVRTC, a few seconds once per process; the paper compiles its kernel at run time as well,
 * PAPER.md:149) -- lists with at most one shear, three SIEs, six lenses and eight positioned light
 * components; beyond that, without libnvrtc, or with LENSED_JIT=0 in the environment, the
 * interpreting kernel runs.
 * lensed_set_static_tracer(h, 0) forces the interpreting kernel (tests compare the two); (h, 1)
 * re-enables the specialised one and returns LENSED_EUNSUPPORTED if the list has none.
 * lensed_get_static_tracer: which one the next call runs: 1 = built-in specialised, 2 = specialised
 * at run time, 0 = interpreting; -1 for NULL.                                              */
lensed_status lensed_set_static_tracer(lensed_handle *h, int on);
int lensed_get_static_tracer(const lensed_handle *h);
/* Test hook: only the compilation step of that run-time specialisation, for a model list (host
 * array of lensed_kind) and an n_quad-point rule; needs NVRTC but no device.  Returns the size of
 * the cubin in bytes, or -1 with the reason (the compiler's log) in log[log_len] (may be NULL).  */
int lensed_debug_jit_compile(const int *models, int n_models, int n_quad, char *log, int log_len);

/* The sampler's random number generator, Philox4x32-10 (Salmon et al. 2011), for tests:
 * counter[4], key[2] -> out[4], host arrays.                                                  */
void lensed_ns_philox(const unsigned *counter, const unsigned *key, unsigned *out);

/*
 * lensed_fma_peak -- FP32 FFMA micro-benchmark used as the measured roofline
 * denominator: runs `iters` dependent-chain FFMAs per thread on a full grid and returns
 * the achieved TFLOP/s (2 flops per FFMA) in *tflops.  Synchronous.                     */
lensed_status lensed_fma_peak(int device, int iters, double *tflops);

/* lensed_issue_probe -- a second micro-benchmark behind the kernel design (DESIGN.md section 5,
 * profiles/r2b.md): FP32-pipe time of a loop body of 64 packed FFMA2 with n_extra in {0, 8, 16, 32,
 * 64} instructions of another kind among them (kind 0 none, 1 LOP3 on the ALU pipe, 2 MUFU.EX2,
 * 3 scalar FFMA, 4 IMAD), `warps` in {1, 2, 4} warps per scheduler on every SM.  *cycles_per_body:
 * SM cycles per body and warp (128 = the pipe's full rate).  Synchronous.  EINVAL / ECUDA.      */
lensed_status lensed_issue_probe(int device, int kind, int n_extra, int warps, double *cycles_per_body);

#ifdef __cplusplus
}
#endif
#endif /* LENSED_TUNE_H */
