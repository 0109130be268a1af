/*
 * lensed.h -- C ABI of the B200-native batched lens likelihood.
 *
 * The hot path of Lensed (Tessore, Bellagamba & Metcalf, arXiv:1505.07674): for a batch
 * of parameter vectors, ray-trace every pixel's quadrature points through the lens
 * models, evaluate source / foreground surface brightness, integrate to pixel
 * luminosities, convolve with the PSF and reduce the weighted chi-square to one
 * log-likelihood per vector.  Citations are "PAPER.md:<line>" of the paper text plus the
 * section / equation; "R<n>" is a reading listed in DESIGN.md where the paper is silent.
 *
 * Every step runs in hand-written CUDA kernels for sm_100a (paper_1505_07674_b200/csrc).
 * There is no CPU fallback and no other backend: without a CUDA device lensed_create
 * fails with LENSED_ECUDA.  Plain pointers and sizes only; "host" / "device" is stated
 * for every pointer.  All device work of a call is enqueued on the given CUDA stream
 * (a cudaStream_t passed as void*, NULL = the legacy default stream) and is asynchronous
 * with respect to the host unless stated otherwise.
 *
 * Thread-safety: the problem data of a handle (image, weights, mask, pixel lists, PSF) is
 * immutable after lensed_create; its scratch buffers and options are not, so calls on ONE
 * handle must not overlap in time.  For several streams or threads on one problem use
 * lensed_clone: clones share the immutable device arrays and own their scratch.
 */
#ifndef LENSED_H
#define LENSED_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lensed_handle lensed_handle;   /* opaque; owns device copies of all inputs */

typedef enum {
    LENSED_OK = 0,
    LENSED_EINVAL = 1,        /* bad argument (see each call)                             */
    LENSED_ENOMEM = 2,        /* host or device allocation failed                         */
    LENSED_ECUDA = 3,         /* CUDA error; text in lensed_last_error                    */
    LENSED_EUNSUPPORTED = 4   /* valid request outside the built limits (see LENSED_MAX_*)*/
} lensed_status;

/* Model kinds.  Lenses deflect (eq. 1, deflections add over lenses,
 * PAPER.md:37, 357); SRC objects are evaluated at the source-plane point y(x), FG
 * objects at the image-plane point x (eq. 2).
 * Parameter layout per kind, in the paper's order:
 *   SIS    x, y, r                   r = Einstein radius                       (R3)
 *   SIE    x, y, r, q, pa            Kormann et al. 1994        (R2)
 *   POINT  x, y, r                   r = Einstein radius of the point mass     (R3)
 *   SHEAR  g1, g2                    about the image centre                    (R4)
 *   SERSIC x, y, r, mag, n, q, pa    PAPER.md:244-252 eqs. 22-23; r = half-light (R5, R6)
 *   GAUSS  x, y, sigma, mag, q, pa                                             (R7)
 *   SKY    level                     per-pixel constant
 * Positions and radii in arcsec relative to the image centre (+x = columns, +y = rows,
 * R1), pa in degrees counter-clockwise from +x to the major axis.  A
 * vector is the concatenation over the model list, in list order.                       */
typedef enum {
    LENSED_LENS_SIS = 0,
    LENSED_LENS_SIE = 1,
    LENSED_LENS_POINT = 2,
    LENSED_LENS_SHEAR = 3,
    LENSED_SRC_SERSIC = 4,
    LENSED_SRC_GAUSS = 5,
    LENSED_FG_SERSIC = 6,
    LENSED_FG_GAUSS = 7,
    LENSED_FG_SKY = 8
} lensed_kind;

#define LENSED_MAX_MODELS 32      /* objects in one model list                            */
#define LENSED_MAX_QUAD   256     /* points of the pixel quadrature rule (g7k15 = 225)    */
#define LENSED_MAX_PSF    63      /* PSF rows / columns                                   */

/*
 * lensed_create -- set up one reconstruction problem (PAPER.md:132-133 steps i-ii,
 * 159, 182): copies every array to the device; the handle is immutable afterwards.
 *   H, W        image rows / columns; pixel (i, j) = (row, column) has centre
 *               x_j = (j-(W-1)/2) s, y_i = (i-(H-1)/2) s                         (R1)
 *   pixel_scale s, arcsec per pixel, > 0
 *   image       [H*W] host f32, row-major: observed d_i
 *   weight      [H*W] host f32, w_i = 1/s_i^2 >= 0 (eq. 17)
 *   mask        [H*W] host u8 or NULL; 0 = masked => w_i := 0
 *   psf         [psf_h*psf_w] host f32, odd dims <= LENSED_MAX_PSF, element
 *               [p+a][q+b] = F_{a,b}, first index = row (R10); divided
 *               by its sum in double (L159).  NULL or 1x1 = no PSF.  Even dims, a
 *               non-finite value or a zero sum: LENSED_EINVAL (R11).
 *   quad        [n_quad][3] host f32 = (xi_k, eta_k, w_k): abscissae as offsets from
 *               the pixel centre in pixel units, weights renormalised to sum 1
 *               (eq. 14, R6).  1 <= n_quad <= LENSED_MAX_QUAD.
 *   models      [n_models] host, 1 <= n_models <= LENSED_MAX_MODELS
 *   mag_zero_point  zp of F = 10^(-0.4 (mag - zp))                               (R6)
 *   device      CUDA device ordinal
 *   out         receives the handle (NULL on failure)
 * Errors: EINVAL for null pointers, non-positive sizes, negative or non-finite weights,
 * non-finite image values at unmasked pixels, bad PSF / rule / kind; ECUDA if there is
 * no usable device; ENOMEM for a failed allocation.  Synchronous.                       */
lensed_status lensed_create(int H, int W, double pixel_scale,
                            const float *image, const float *weight,
                            const unsigned char *mask,
                            const float *psf, int psf_h, int psf_w,
                            const float *quad, int n_quad,
                            const int *models, int n_models,
                            double mag_zero_point, int device,
                            lensed_handle **out);

/*
 * lensed_clone -- a second handle on the same problem, for another stream or thread.  The
 * large immutable device arrays (image, weights, pixel lists, PSF taps) are shared and
 * reference-counted; the clone has its own scratch, options and profile, so calls on the two
 * handles may overlap in time (one handle per stream).  Either may be destroyed first.
 * Synchronous.  EINVAL for NULL; ENOMEM / ECUDA.                                          */
lensed_status lensed_clone(const lensed_handle *h, lensed_handle **out);

/* P, the length of one parameter vector for the handle's model list; -1 for NULL.       */
int lensed_num_params(const lensed_handle *h);

/* Pixels lensed_loglike ray-traces per vector: the unmasked set dilated by the PSF
 * window with border clamping (R8) plus one guard row above and below every window
 * (an implementation margin; the result does not depend on it); H*W without a mask.
 * -1 for NULL.                                                                           */
int lensed_num_traced(const lensed_handle *h);

/* H * W, the pixels of one model image (the stride of lensed_render's output); -1 for NULL. */
int lensed_num_pixels(const lensed_handle *h);

/*
 * lensed_render -- model images L* (PAPER.md:136 step iv; eqs. 14, 15), mask ignored.
 *   params_dev  [B][P] device f32
 *   model_dev   [B][H][W] device f32, receives the PSF-convolved pixel luminosities; a
 *               vector outside the model domain gets NaN everywhere
 * Errors: EINVAL for null pointers or B < 1; ENOMEM / ECUDA.                            */
lensed_status lensed_render(lensed_handle *h, const float *params_dev, int B,
                            float *model_dev, void *cuda_stream);

/*
 * lensed_loglike -- loglike = -1/2 sum_i w_i (d_i - L*_i)^2 per vector
 * (PAPER.md:137 step v, 172-182 eqs. 16-17; the normalisation term is dropped as in
 * the paper).
 *   params_dev  [B][P] device f32
 *   logl_dev    [B] device f32; -INFINITY for a vector outside the model domain
 * Deterministic: the same inputs give bitwise the same output on every call.            */
lensed_status lensed_loglike(lensed_handle *h, const float *params_dev, int B,
                             float *logl_dev, void *cuda_stream);

/*
 * Image-plane priors (section 5): "Instead of defining the prior
 * distribution on the source plane, one can define a prior on the image plane for the position
 * at which one of the images of the source is required to appear.  Drawing from such a
 * distribution is done ... by first sampling a position on the image plane, mapping it to the
 * source plane, and assigning it to the source."
 *
 * lensed_deflect -- the map itself, y = x - sum_lenses alpha(x) (eq. 1), for K
 * image-plane points per parameter vector through that vector's own lens list.
 *   params_dev  [B][P] device f32 (light components of the list are ignored)
 *   xy_dev      [B][K][2] device f32: image-plane (x, y), arcsec (R1)
 *   out_dev     [B][K][2] device f32: source-plane (x, y), arcsec; NaN where a lens parameter of
 *               the vector is outside its domain or the point is not finite
 * Double-precision arithmetic on the device.  Asynchronous.  EINVAL for null pointers, B < 1, K < 1.
 *
 * lensed_image_plane_prior -- the assignment, in place: for every vector and every listed
 * source component, its (x, y) parameters hold an image-plane position on entry (what the
 * sampler drew from the image-plane prior) and the source-plane position y(x) on return.
 *   params_dev     [B][P] device f32, read and written (only those (x, y) entries change)
 *   source_models  [n_sources] HOST: indices into the model list given to lensed_create; each
 *                  must be a LENSED_SRC_* component, none twice
 * Asynchronous.  EINVAL for null pointers, B < 1, a bad or repeated index, a non-source.        */
lensed_status lensed_deflect(lensed_handle *h, const float *params_dev, int B, const float *xy_dev, int K,
                             float *out_dev, void *cuda_stream);
lensed_status lensed_image_plane_prior(lensed_handle *h, float *params_dev, int B, const int *source_models,
                                       int n_sources, void *cuda_stream);

/* The same two calls with HOST buffers: the parameters are copied to the device, the
 * result is copied back and the stream is synchronised before returning.  Pinned host
 * memory makes the copies asynchronous until that final synchronisation.                */
lensed_status lensed_render_host(lensed_handle *h, const float *params_host, int B,
                                 float *model_host, void *cuda_stream);
lensed_status lensed_loglike_host(lensed_handle *h, const float *params_host, int B,
                                  float *logl_host, void *cuda_stream);

/*
 * lensed_estimate_weights -- create-time variance estimation from the data (PAPER.md:190-212
 * eqs. 18-21), for observations without an independent variance map: photon counts
 * k_i = g_i (d_i + b_i) are Poisson, so  s_i^2 = (d_i + b_i) / g_i  and
 *   w_i = x_i / s_i^2 = x_i g_i / (d_i + b_i).
 *   image   [n] host f32, d_i
 *   gain    [n] host f32 or NULL (then gain0 for every pixel): effective gain g_i > 0 (eq. 19)
 *   offset  [n] host f32 or NULL (then offset0): b_i, what was subtracted from the data
 *   extra   [n] host f32 or NULL (then 1): the multiplicative extra weight factor x_i >= 0
 *   weight  [n] host f32, receives w_i, ready for lensed_create
 * Pixels whose estimated counts are not positive (d_i + b_i <= 0) cannot be given a Poisson
 * variance and get w_i = 0, i.e. they are masked (reading R15).  Host arithmetic in
 * double; no device is touched.  EINVAL for NULL image / weight, n < 1, a gain <= 0, a
 * negative extra factor or a non-finite input.                                            */
lensed_status lensed_estimate_weights(long long n, const float *image, const float *gain, double gain0,
                                      const float *offset, double offset0, const float *extra,
                                      float *weight);

/*
 * Quadrature error estimate ("an embedded three-point rule estimates the error
 * of the integration for each pixel, which is saved with the output").
 * lensed_set_error_rule: w_embedded [n_quad] host f32 = weights of the embedded lower-order
 * rule at the abscissae given to lensed_create (0 at the points it does not use; for the
 * Cartesian square of a Gauss-Kronrod rule: the products of the embedded Gauss weights),
 * renormalised to sum 1.  EINVAL for NULL, non-finite values or a zero sum.  Synchronises
 * the device.
 * lensed_render_error: err_dev [B][H*W] device f32 receives, for every pixel (mask ignored),
 *   | sum_k w_k I(x_k) - sum_k w'_k I(x_k) |
 * of the UNCONVOLVED pixel luminosity (eq. 14, before the PSF); NaN for parameter vectors
 * outside the model domain.  Asynchronous on `stream`.  EINVAL before an embedded rule is set.
 * A diagnostic, not on the likelihood path: it runs the interpreting tracer.              */
lensed_status lensed_set_error_rule(lensed_handle *h, const float *w_embedded);
lensed_status lensed_render_error(lensed_handle *h, const float *params_dev, int B, float *err_dev, void *stream);

/*
 * lensed_ns_run -- device-resident nested sampling with the batched likelihood.
 * PAPER.md:134-139 steps (iii)-(vii): draw parameters from the prior, compute their likelihood,
 * accumulate the posterior, repeat until the parameter space is sufficiently sampled;
 * the sampler is Nested Sampling (Skilling 2004, 2006), which also gives
 * the evidence (eq. 13).  The paper delegates this to the MultiNest library;
 * this call is the base algorithm with MultiNest's ellipsoidal bound (a single ellipsoid), run
 * with everything on the device: live points, proposal batches, evidence accumulators and dead
 * points.  Each round proposes `batch` vectors inside the current likelihood contour, evaluates
 * them with ONE lensed_loglike call and consumes them in order against the rising threshold.
 *   prior_lo, prior_hi  [P] HOST: uniform priors; lo == hi fixes a parameter (PAPER.md:133 step ii)
 *   image_plane_sources [n_image_plane] HOST or NULL: model-list indices of source components
 *                       whose (x, y) prior box is an IMAGE-plane box: every drawn vector goes
 *                       through lensed_image_plane_prior before its likelihood
 *   opt                 n_live in [free parameters + 1, 4096]; batch >= 1; tol: stop when
 *                       max live L * X < tol * Z; enlarge >= 1: linear enlargement of the ellipsoid
 *                       that bounds the live points; seed of the counter-based generator;
 *                       tied_to [P] HOST or NULL: parameter p with tied_to[p] = q >= 0 is not drawn but takes
 *                       the value drawn for parameter q ("the centre of the mass distribution
 *                       [forced] to coincide with the centre of the surface brightness distribution"); it
 *                       needs lo[p] == hi[p], q untied and q != p (EINVAL otherwise); -1 = not tied
 *   res                 HOST, receives ln Z, its error sqrt(H/n_live), the information H, counts
 *   samples_dev [capacity][P], logl_dev [capacity], logw_dev [capacity]: device f32 or NULL with
 *                       capacity 0: the dead points in order of death, then the live points; logw =
 *                       ln(L w / Z), i.e. posterior weights summing to 1.  Points beyond capacity are
 *                       dropped (res->n_samples = written, res->n_dead = all deaths before the live set).
 * Synchronous: returns when the run has converged or max_rounds is reached.  At most 48 free
 * parameters (LENSED_EUNSUPPORTED beyond).  EINVAL for null pointers, hi < lo, no free parameter,
 * bad options.  The handle's one-call-at-a-time rule applies for the whole run.               */
typedef struct {
    int n_live, batch, max_rounds;
    double tol, enlarge;
    unsigned long long seed;
    const int *tied_to;       /* HOST [P] or NULL: see above */
} lensed_ns_options;
typedef struct {
    double ln_z, ln_z_err, information;
    long long n_rounds, n_likelihood, n_dead, n_samples;
    int converged;
} lensed_ns_result;
lensed_status lensed_ns_run(lensed_handle *h, const float *prior_lo, const float *prior_hi,
                            const int *image_plane_sources, int n_image_plane,
                            const lensed_ns_options *opt, lensed_ns_result *res,
                            float *samples_dev, float *logl_dev, float *logw_dev, long long capacity,
                            void *cuda_stream);
/*
 * lensed_chisq_static -- the likelihood of model images that are already on the device, from a
 * call that allocates NOTHING: no cudaMalloc, no cudaMallocAsync, no cudaFree, no handle.
 *   loglike[b] = -1/2 sum_i w_i (d_i - model[b][i])^2       (eqs. 16-17)
 *
 * Why it exists.  lensed_create allocates the problem's arrays and lensed_loglike / lensed_render
 * grow their scratch whenever a batch is larger than any they have seen.  That is wrong for a
 * caller that may not allocate once it is running: a sampler inside a process whose deep-learning
 * framework has already taken the device memory for its own pool (a later cudaMalloc then fails);
 * workers on several streams (lensed_clone), where one worker's cudaMalloc / cudaFree synchronises
 * the device under all the others; a job on a fixed memory budget (MIG slice, MPS memory limit)
 * whose budget is checked once at start-up.  Such a caller scores images held in ITS OWN buffers
 * -- written by lensed_render at a batch size warmed up during set-up, or by its own forward model,
 * or lensed_render's plus a term this library does not model -- with this call.
 *
 *   device      CUDA device ordinal the pointers belong to (made current by the call)
 *   image_dev   [n_pix] device f32, the data d_i
 *   weight_dev  [n_pix] device f32, w_i = 1 / s_i^2 >= 0 with 0 at masked pixels;
 *               pixels with w_i = 0 are skipped, so the model may hold anything (NaN too) there
 *   model_dev   [B][n_pix] device f32, the PSF-convolved model images L* (lensed_render's layout)
 *   logl_dev    [B] device f32; -INFINITY for an image with a non-finite pixel under a non-zero
 *               weight (lensed_render's NaN image of a vector outside the model domain gives the
 *               -INFINITY lensed_loglike gives that vector)
 * All four are caller-owned; nothing is retained.  Asynchronous on `cuda_stream`.  Deterministic:
 * FP32 differences, FP64 sums in a fixed order, bitwise the same on every call.
 *
 * Scratch and its limit.  The per-block partial sums live in one fixed array inside the library's
 * device image: 1 040 KB that every GPU loading the library holds until the process exits.  It
 * serves at most LENSED_CHISQ_STATIC_MAX_VECTORS images per call (n_pix up to 2^30); a larger B is
 * refused with LENSED_EINVAL and a message saying so -- split the batch.  EVERY call on a device,
 * from any thread or stream, uses that same array: two calls that may run on the GPU at the same
 * time (different streams with no ordering between them) race on it and both results are garbage;
 * order them with an event, or keep this call on one stream.  The array keeps what the last call
 * left; each call clears the part that has to start at zero, on its stream, before its kernel.
 *
 * First call on a device.  It looks up the array's device address (cudaGetSymbolAddress, which may
 * load the library's kernels onto that device) and caches it; make that first call during set-up,
 * before any stream capture begins.  Later calls issue one memset and one kernel, nothing else.
 *
 * Errors: EINVAL for null pointers, B < 1, n_pix < 1, B or n_pix beyond the limits, a bad device
 * ordinal (checked in that order, before CUDA is touched); ECUDA with the CUDA error text.  The
 * text is read with lensed_last_error(NULL).                                                    */
#define LENSED_CHISQ_STATIC_MAX_VECTORS 4096
lensed_status lensed_chisq_static(int device, const float *image_dev, const float *weight_dev, long long n_pix,
                                  const float *model_dev, int B, float *logl_dev, void *cuda_stream);

/* Text of the last error on this handle (valid until the next call on the handle); for
 * a failed lensed_create or lensed_fma_peak pass NULL to read the thread-local text.  After a
 * successful lensed_create it is empty, or says why the list's tracer could not be specialised at
 * run time (the interpreting tracer is then in use; see "Tracer selection").               */
const char *lensed_last_error(const lensed_handle *h);

/* Frees the handle and its device memory (synchronises the device).  NULL is a no-op.   */
void lensed_destroy(lensed_handle *h);

#ifdef __cplusplus
}
#endif
#endif /* LENSED_H */
