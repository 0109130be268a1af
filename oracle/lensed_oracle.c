/*
 * lensed_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, double-precision CPU statement of what the hot path computes:
 * the batched Lensed likelihood (Tessore, Bellagamba & Metcalf, arXiv:1505.07674).
 * It exists only to check the CUDA library; only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or constant with paper_1505_07674_b200/csrc.
 *
 * Each function cites the passage of /root/reference/PAPER.md it follows
 * ("PAPER.md:<line>", section / equation) or the reading of DESIGN.md
 * ("R<n>", taken from SURVEY.md section 8(c.2)) where the paper is silent.
 *
 * Loop order is the paper's: parameter vector -> pixel -> rule point -> object
 * (PAPER.md:136-137 steps iv-v, 155-159 eq. 14), then the direct PSF
 * convolution (eq. 15), then the weighted chi-square
 * (eq. 17).  No blocking, fusion or reordering.
 *
 * Pins (tests/test_oracle_pins.py, all "-m 'not gpu'"): SIS ring and image
 * positions, SIE -> SIS for q -> 1, alpha = grad(psi) by finite differences,
 * div(alpha) = 2 kappa = b/R, the SIE spot value of tests/golden, b_n against
 * the textbook values and scipy's inverse incomplete gamma, half-light flux by
 * brute-force integration, total Sersic / Gaussian flux, Gaussian == Sersic
 * n=1/2, quadrature exactness and brute-force supersampling, one-hot PSF shift,
 * delta PSF identity, PSF auto-normalisation, logL closed forms, rotation /
 * mirror symmetry of the whole pipeline; oracle_render_raw with a one-point
 * rule against oracle_brightness and its summed flux against F for Sersic
 * indices 0.5 .. 8 (both are built from the same two static functions
 * light_constants / light_profile); oracle_source_position against the lens
 * equation solved by inspection (SIS image positions), the additivity of
 * deflections and grad(psi); oracle_estimate_weights against hand values and
 * the unit mean of w (d - mu)^2 on seeded Poisson counts; params_valid bound
 * by bound against the hand-written table of tests/cases.py (domain_cases:
 * every kind, one vector just inside and one just outside every bound, NaN /
 * inf in every slot).  Parity unpinned:
 * absolute pixel values of any figure of the paper (it prints none).
 *
 * Build: gcc -O2 -std=c99 -fopenmp -fPIC -shared lensed_oracle.c -o liblensed_oracle.so -lm
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_PI 3.14159265358979323846264338327950288

/* Model kinds: the order of the paper's object list.
 * Lenses deflect; "SRC" objects are evaluated at the source-plane point y(x),
 * "FG" objects at the image-plane point x (eq. 2). */
enum {
    ORACLE_LENS_SIS = 0,   /* x, y, r                     (R3)                  */
    ORACLE_LENS_SIE = 1,   /* x, y, r, q, pa   */
    ORACLE_LENS_POINT = 2, /* x, y, r (its Einstein radius) (R3)                */
    ORACLE_LENS_SHEAR = 3, /* g1, g2                      (R4)                  */
    ORACLE_SRC_SERSIC = 4, /* x, y, r, mag, n, q, pa*/
    ORACLE_SRC_GAUSS = 5,  /* x, y, sigma, mag, q, pa     (R7)                  */
    ORACLE_FG_SERSIC = 6,
    ORACLE_FG_GAUSS = 7,
    ORACLE_FG_SKY = 8      /* level    */
};

int oracle_kind_num_params(int kind)
{
    switch (kind) {
    case ORACLE_LENS_SIS: return 3;
    case ORACLE_LENS_SIE: return 5;
    case ORACLE_LENS_POINT: return 3;
    case ORACLE_LENS_SHEAR: return 2;
    case ORACLE_SRC_SERSIC: case ORACLE_FG_SERSIC: return 7;
    case ORACLE_SRC_GAUSS: case ORACLE_FG_GAUSS: return 6;
    case ORACLE_FG_SKY: return 1;
    default: return -1;
    }
}

int oracle_num_params(const int *kinds, int n_models)
{
    int P = 0;
    for (int m = 0; m < n_models; ++m) {
        int k = oracle_kind_num_params(kinds[m]);
        if (k < 0) return -1;
        P += k;
    }
    return P;
}

static int is_lens(int kind) { return kind <= ORACLE_LENS_SHEAR; }
static int is_source(int kind) { return kind == ORACLE_SRC_SERSIC || kind == ORACLE_SRC_GAUSS; }

/* ------------------------------------------------------------------------ */
/* Sersic b_n (R5): r_S is the half-light radius, so b_n is the
 * root of P(2n, b) = 1/2 with P the regularised lower incomplete gamma.      */

/* P(a, x) by its power series  x^a e^-x / Gamma(a+1) * sum_k x^k / (a+1)_k
 * (converges for every x > 0; used for x < a + 1), else 1 - Q by the
 * Legendre continued fraction evaluated with the modified Lentz recurrence.  */
double oracle_gamma_p(double a, double x)
{
    if (!(a > 0.0) || !(x >= 0.0)) return NAN;
    if (x == 0.0) return 0.0;
    double lead = exp(a * log(x) - x - lgamma(a));
    if (x < a + 1.0) {
        double term = 1.0 / a, sum = term;
        for (int k = 1; k < 100000; ++k) {
            term *= x / (a + k);
            sum += term;
            if (term < sum * 1e-17) break;
        }
        return lead * sum;
    }
    const double tiny = 1e-300;
    double bq = x + 1.0 - a, c = 1.0 / tiny, d = 1.0 / bq, h = d;
    for (int k = 1; k < 100000; ++k) {
        double an = -k * (k - a);
        bq += 2.0;
        d = an * d + bq; if (fabs(d) < tiny) d = tiny;
        c = bq + an / c; if (fabs(c) < tiny) c = tiny;
        d = 1.0 / d;
        double del = d * c;
        h *= del;
        if (fabs(del - 1.0) < 1e-16) break;
    }
    return 1.0 - lead * h;
}

double oracle_sersic_bn(double n)
{
    double a = 2.0 * n;
    double lo = 0.0, hi = 2.0 * n + 10.0;   /* P(a, a+10) > 1/2 for every a > 0 */
    for (int it = 0; it < 200; ++it) {
        double mid = 0.5 * (lo + hi);
        if (oracle_gamma_p(a, mid) < 0.5) lo = mid; else hi = mid;
        if (hi - lo <= 1e-16 * hi) break;
    }
    return 0.5 * (lo + hi);
}

/* ------------------------------------------------------------------------ */
/* Parameter domain: outside it the vector is invalid,
 * logL = -inf and the rendered image is NaN; it is not a call error.        */
static int params_valid(int kind, const double *p)
{
    int np = oracle_kind_num_params(kind);
    for (int i = 0; i < np; ++i) if (!isfinite(p[i])) return 0;
    switch (kind) {
    case ORACLE_LENS_SIS: case ORACLE_LENS_POINT: return p[2] >= 0.0;
    case ORACLE_LENS_SIE: return p[2] >= 0.0 && p[3] > 0.0 && p[3] <= 1.0;
    case ORACLE_LENS_SHEAR: return 1;
    case ORACLE_SRC_SERSIC: case ORACLE_FG_SERSIC:
        return p[2] > 0.0 && p[4] >= 0.02 && p[4] <= 20.0 && p[5] > 0.0 && p[5] <= 1.0;
    case ORACLE_SRC_GAUSS: case ORACLE_FG_GAUSS:
        return p[2] > 0.0 && p[4] > 0.0 && p[4] <= 1.0;
    case ORACLE_FG_SKY: return 1;
    default: return 0;
    }
}

/* ------------------------------------------------------------------------ */
/* Deflection angle of one lens at (x, y), arcsec (eq. 1).
 * (u, v) = offset from the lens centre rotated by -PA into the lens frame,
 * major axis along u, PA counter-clockwise from +x.           */
void oracle_deflection(int kind, const double *p, double x, double y,
                       double *ax, double *ay)
{
    *ax = 0.0; *ay = 0.0;
    switch (kind) {
    case ORACLE_LENS_SIS: {                       /* R3: alpha = b (u,v)/r     */
        double u = x - p[0], v = y - p[1], r = sqrt(u * u + v * v);
        if (r > 0.0) { *ax = p[2] * u / r; *ay = p[2] * v / r; }
        break;
    }
    case ORACLE_LENS_POINT: {                     /* R3: alpha = tE^2 (u,v)/r^2 */
        double u = x - p[0], v = y - p[1], r2 = u * u + v * v;
        if (r2 > 0.0) { *ax = p[2] * p[2] * u / r2; *ay = p[2] * p[2] * v / r2; }
        break;
    }
    case ORACLE_LENS_SHEAR:                       /* R4: about the image centre */
        *ax = p[0] * x + p[1] * y;
        *ay = p[1] * x - p[0] * y;
        break;
    case ORACLE_LENS_SIE: {                       /* R2: Kormann et al. 1994    */
        double b = p[2], q = p[3], pa = p[4] * (ORACLE_PI / 180.0);
        double c = cos(pa), s = sin(pa);
        double dx = x - p[0], dy = y - p[1];
        double u = c * dx + s * dy, v = -s * dx + c * dy;
        double au, av;
        if (1.0 - q < 1e-9) {                     /* SIS form in the q->1 limit */
            double r = sqrt(u * u + v * v);
            if (r > 0.0) { au = b * u / r; av = b * v / r; } else { au = av = 0.0; }
        } else {
            double qp = sqrt(1.0 - q * q);
            double psi = sqrt(q * q * u * u + v * v);
            if (psi > 0.0) {
                double A = b * sqrt(q) / qp;
                au = A * atan(qp * u / psi);
                av = A * atanh(qp * v / psi);
            } else { au = av = 0.0; }
        }
        *ax = c * au - s * av;
        *ay = s * au + c * av;
        break;
    }
    default: break;
    }
}

/* Lensing potential of one lens (used by the pins only: alpha = grad psi).  */
double oracle_potential(int kind, const double *p, double x, double y)
{
    switch (kind) {
    case ORACLE_LENS_SIS: {
        double u = x - p[0], v = y - p[1];
        return p[2] * sqrt(u * u + v * v);
    }
    case ORACLE_LENS_POINT: {
        double u = x - p[0], v = y - p[1];
        return p[2] * p[2] * log(sqrt(u * u + v * v));
    }
    case ORACLE_LENS_SHEAR:
        return 0.5 * p[0] * (x * x - y * y) + p[1] * x * y;
    case ORACLE_LENS_SIE: {                       /* isothermal: psi = x.alpha  */
        double ax, ay;
        oracle_deflection(kind, p, x, y, &ax, &ay);
        return (x - p[0]) * ax + (y - p[1]) * ay;
    }
    default: return 0.0;
    }
}

/* ------------------------------------------------------------------------ */
/* Surface brightness of one source / foreground object at (x, y) arcsec, in
 * flux per pixel area (R6): integrating over the plane in pixel units gives
 * the total flux F = 10^(-0.4 (mag - zp)).
 *
 * The arithmetic is split in two static functions that BOTH oracle_brightness
 * (what the half-light, total-flux, profile-shape and ellipse-convention pins
 * test) and oracle_render_raw (what every GPU parity test compares against)
 * call, so that a pin on one is a pin on the other:
 *   light_constants: what depends on the parameter vector only (b_n, I_0);
 *   light_profile:   the profile at a point, given those constants.          */
static void light_constants(int kind, const double *p, double scale, double zp,
                            double *bn, double *I0)
{
    *bn = 0.0; *I0 = 0.0;
    switch (kind) {
    case ORACLE_SRC_SERSIC: case ORACLE_FG_SERSIC: { /* PAPER.md:244-252 eqs 22-23 */
        double rs = p[2], mag = p[3], n = p[4];
        double F = pow(10.0, -0.4 * (mag - zp));     /* total magnitude, L252 */
        *bn = oracle_sersic_bn(n);                    /* R5: half-light radius */
        *I0 = F * exp(2.0 * n * log(*bn) - lgamma(2.0 * n))
              / (2.0 * ORACLE_PI * n * rs * rs) * scale * scale;      /* R6   */
        break;
    }
    case ORACLE_SRC_GAUSS: case ORACLE_FG_GAUSS: {                    /* R7     */
        double sg = p[2], mag = p[3];
        double F = pow(10.0, -0.4 * (mag - zp));
        *I0 = F / (2.0 * ORACLE_PI * sg * sg) * scale * scale;
        break;
    }
    default: break;
    }
}

static double light_profile(int kind, const double *p, double bn, double I0,
                            double x, double y)
{
    switch (kind) {
    case ORACLE_SRC_SERSIC: case ORACLE_FG_SERSIC: { /* PAPER.md:244-250 eqs 22-23 */
        double rs = p[2], n = p[4], q = p[5], pa = p[6] * (ORACLE_PI / 180.0);
        double c = cos(pa), s = sin(pa);
        double dx = x - p[0], dy = y - p[1];
        double u = c * dx + s * dy, v = -s * dx + c * dy;
        double R = sqrt(u * u * q + v * v / q);                      /* eq. 23 */
        return I0 * exp(-bn * pow(R / rs, 1.0 / n));                  /* eq. 22 */
    }
    case ORACLE_SRC_GAUSS: case ORACLE_FG_GAUSS: {                    /* R7     */
        double sg = p[2], q = p[4], pa = p[5] * (ORACLE_PI / 180.0);
        double c = cos(pa), s = sin(pa);
        double dx = x - p[0], dy = y - p[1];
        double u = c * dx + s * dy, v = -s * dx + c * dy;
        double R2 = u * u * q + v * v / q;                            /* eq. 23 squared */
        return I0 * exp(-R2 / (2.0 * sg * sg));
    }
    case ORACLE_FG_SKY: return p[0];
    default: return 0.0;
    }
}

double oracle_brightness(int kind, const double *p, double x, double y,
                         double scale, double zp)
{
    double bn, I0;
    light_constants(kind, p, scale, zp, &bn, &I0);
    return light_profile(kind, p, bn, I0, x, y);
}

/* Source-plane position of the image-plane point (x, y), arcsec:
 *   y(x) = x - sum over the lenses of the list of alpha(x)    PAPER.md:53-57 eq. 1;
 * deflections of several lens objects add.  Non-lens entries
 * of the model list are skipped.  This is also the map of the image-plane
 * priors ("sampling a position on the image plane,
 * mapping it to the source plane, and assigning it to the source").
 * offs[m] = offset of model m's parameters in params.                        */
static void source_position(const int *kinds, int n_models, const int *offs,
                            const double *params, double x, double y,
                            double *sx, double *sy)
{
    double ax = 0.0, ay = 0.0;
    for (int m = 0; m < n_models; ++m) if (is_lens(kinds[m])) {
        double dax, day;
        oracle_deflection(kinds[m], params + offs[m], x, y, &dax, &day);
        ax += dax; ay += day;
    }
    *sx = x - ax; *sy = y - ay;
}

/* The same for K points of ONE parameter vector: xy[K][2] -> out[K][2].
 * Returns 0 (out = NaN) if a LENS of the vector is outside the domain; the
 * lights of the list do not enter.                                           */
int oracle_source_position(const int *kinds, int n_models, const double *params,
                           const double *xy, int K, double *out)
{
    int *offs = (int *)calloc((size_t)n_models, sizeof(int));
    int off = 0, valid = 1;
    for (int m = 0; m < n_models; ++m) {
        offs[m] = off;
        if (is_lens(kinds[m]) && !params_valid(kinds[m], params + off)) valid = 0;
        off += oracle_kind_num_params(kinds[m]);
    }
    for (int k = 0; k < K; ++k) {
        if (valid) source_position(kinds, n_models, offs, params, xy[2 * k], xy[2 * k + 1],
                                   out + 2 * k, out + 2 * k + 1);
        else out[2 * k] = out[2 * k + 1] = NAN;
    }
    free(offs);
    return valid;
}

/* ------------------------------------------------------------------------ */
/* Unconvolved pixel luminosities L_i of one parameter vector, every pixel of
 * the image (mask ignored, R8).  PAPER.md:65-69 eq. 3, 155-159 eq. 14.
 * Grid (R1): pixel (i, j) = (row, column) has centre
 *   x_j = (j - (W-1)/2) s,  y_i = (i - (H-1)/2) s.
 * quad[k] = (xi_k, eta_k, w_k), offsets in pixel units; weights are divided
 * by their sum (R6).  Returns 0 if the vector is outside the domain (L=NaN). */
int oracle_render_raw(int H, int W, double scale, const double *quad, int n_quad,
                      const int *kinds, int n_models, double zp,
                      const double *params, double *L)
{
    int valid = 1, off = 0;
    /* b_n and I_0 depend on the vector only: light_constants once per object,
     * light_profile per ray -- the two functions oracle_brightness is made of. */
    double *bn = (double *)calloc((size_t)n_models, sizeof(double));
    double *I0 = (double *)calloc((size_t)n_models, sizeof(double));
    int *offs = (int *)calloc((size_t)n_models, sizeof(int));
    for (int m = 0; m < n_models; ++m) {
        const double *p = params + off;
        offs[m] = off;
        off += oracle_kind_num_params(kinds[m]);
        if (!params_valid(kinds[m], p)) { valid = 0; continue; }
        if (!is_lens(kinds[m])) light_constants(kinds[m], p, scale, zp, &bn[m], &I0[m]);
    }
    if (!valid) {
        for (long i = 0; i < (long)H * W; ++i) L[i] = NAN;
        free(bn); free(I0); free(offs);
        return 0;
    }
    double wsum = 0.0;
    for (int k = 0; k < n_quad; ++k) wsum += quad[3 * k + 2];

#pragma omp parallel for schedule(dynamic, 4)
    for (int i = 0; i < H; ++i) {
        for (int j = 0; j < W; ++j) {
            double xc = (j - 0.5 * (W - 1)) * scale, yc = (i - 0.5 * (H - 1)) * scale;
            double Li = 0.0;
            for (int k = 0; k < n_quad; ++k) {
                double x = xc + quad[3 * k] * scale, y = yc + quad[3 * k + 1] * scale;
                double sx, sy;                               /* eq. 1: y(x) = x - sum alpha */
                source_position(kinds, n_models, offs, params, x, y, &sx, &sy);
                double I = 0.0;                              /* eq. 2           */
                for (int m = 0; m < n_models; ++m) {
                    int kd = kinds[m];
                    if (is_lens(kd)) continue;
                    if (is_source(kd)) I += light_profile(kd, params + offs[m], bn[m], I0[m], sx, sy);
                    else               I += light_profile(kd, params + offs[m], bn[m], I0[m], x, y);
                }
                Li += (quad[3 * k + 2] / wsum) * I;          /* eq. 14          */
            }
            L[(long)i * W + j] = Li;
        }
    }
    free(bn); free(I0); free(offs);
    return 1;
}

/* ------------------------------------------------------------------------ */
/* Discrete PSF convolution, eq. 15:
 *   L*_ij = sum_{k=-p..p} sum_{l=-q..q} F_{-k,-l} L_{i+k, j+l},
 * F given as (2p+1) x (2q+1) values, array element [p+a][q+b] = F_{a,b}, first
 * index = row (R10); F is divided by its sum ("normalised automatically",
 * L159); out-of-image indices repeat the closest pixel (L164).
 * psf == NULL or 1x1 means no PSF: L* = L.                                   */
void oracle_convolve(const double *L, int H, int W, const double *psf, int ph, int pw,
                     double *out)
{
    if (!psf || (ph == 1 && pw == 1)) {
        memcpy(out, L, sizeof(double) * (size_t)H * W);
        return;
    }
    int p = (ph - 1) / 2, q = (pw - 1) / 2;
    double fsum = 0.0;
    for (int t = 0; t < ph * pw; ++t) fsum += psf[t];
#pragma omp parallel for schedule(static)
    for (int i = 0; i < H; ++i) {
        for (int j = 0; j < W; ++j) {
            double acc = 0.0;
            for (int k = -p; k <= p; ++k) {
                int ii = i + k; if (ii < 0) ii = 0; if (ii > H - 1) ii = H - 1;
                for (int l = -q; l <= q; ++l) {
                    int jj = j + l; if (jj < 0) jj = 0; if (jj > W - 1) jj = W - 1;
                    acc += (psf[(p - k) * pw + (q - l)] / fsum) * L[(long)ii * W + jj];
                }
            }
            out[(long)i * W + j] = acc;
        }
    }
}

/* ------------------------------------------------------------------------ */
/* loglike = -1/2 sum_i w_i (d_i - L*_i)^2, eq. 17; a masked
 * pixel (mask[i] == 0) has w_i = 0 (L182).  Summed in double in pixel order. */
double oracle_chi2_loglike(const double *model, const double *image, const double *weight,
                           const unsigned char *mask, long m)
{
    double s = 0.0;
    for (long i = 0; i < m; ++i) {
        double w = (mask && !mask[i]) ? 0.0 : weight[i];
        double r = image[i] - model[i];
        s += w * r * r;
    }
    return -0.5 * s;
}

/* Model images L* for B parameter vectors: model[B][H][W].                  */
int oracle_render(int H, int W, double scale, const double *psf, int ph, int pw,
                  const double *quad, int n_quad, const int *kinds, int n_models,
                  double zp, const double *params, int B, double *model, int nthreads)
{
    int P = oracle_num_params(kinds, n_models);
    if (P < 0) return -1;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
    double *raw = (double *)malloc(sizeof(double) * (size_t)H * W);
    if (!raw) return -2;
    for (int b = 0; b < B; ++b) {
        oracle_render_raw(H, W, scale, quad, n_quad, kinds, n_models, zp,
                          params + (size_t)b * P, raw);
        oracle_convolve(raw, H, W, psf, ph, pw, model + (size_t)b * H * W);
    }
    free(raw);
    return 0;
}

/* logL[B]; model (optional, may be NULL) receives the B convolved images.   */
int oracle_loglike(int H, int W, double scale, const double *image, const double *weight,
                   const unsigned char *mask, const double *psf, int ph, int pw,
                   const double *quad, int n_quad, const int *kinds, int n_models,
                   double zp, const double *params, int B, double *logl, double *model,
                   int nthreads)
{
    int P = oracle_num_params(kinds, n_models);
    if (P < 0) return -1;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
    double *raw = (double *)malloc(sizeof(double) * (size_t)H * W);
    double *cv = (double *)malloc(sizeof(double) * (size_t)H * W);
    if (!raw || !cv) { free(raw); free(cv); return -2; }
    for (int b = 0; b < B; ++b) {
        int ok = oracle_render_raw(H, W, scale, quad, n_quad, kinds, n_models, zp,
                                   params + (size_t)b * P, raw);
        oracle_convolve(raw, H, W, psf, ph, pw, cv);
        logl[b] = ok ? oracle_chi2_loglike(cv, image, weight, mask, (long)H * W) : -INFINITY;
        if (model) memcpy(model + (size_t)b * H * W, cv, sizeof(double) * (size_t)H * W);
    }
    free(raw); free(cv);
    return 0;
}

/* ------------------------------------------------------------------------ */
/* Variance estimation from the data, section 3.3:
 *   k_i = g_i (d_i + b_i)                      photon counts          eq. 18
 *   Var(k_i) = k_i                             Poisson                eq. 20
 *   s_i^2 = g_i^-2 Var(k_i) = (d_i + b_i)/g_i                         eq. 21
 *   w_i = x_i / s_i^2                          weights of eq. 17 times the
 *                                              "multiplicative extra weight factor" (L212)
 * gain / offset / extra: maps [n], or NULL for the scalar gain0 / offset0 / 1.
 * R15: a pixel whose counts k_i are not positive has no Poisson variance and
 * gets w_i = 0 (masked).  variance (optional) receives s_i^2 (NaN where R15).
 * Returns the number of pixels R15 masked, or -1 for an input outside the
 * domain (g_i <= 0, x_i < 0, non-finite).                                    */
long oracle_estimate_weights(long n, const double *image, const double *gain, double gain0,
                             const double *offset, double offset0, const double *extra,
                             double *weight, double *variance)
{
    long masked = 0;
    for (long i = 0; i < n; ++i) {
        double g = gain ? gain[i] : gain0, b = offset ? offset[i] : offset0;
        double x = extra ? extra[i] : 1.0;
        if (!isfinite(image[i]) || !isfinite(g) || !isfinite(b) || !isfinite(x)) return -1;
        if (!(g > 0.0) || x < 0.0) return -1;
        double k = g * (image[i] + b);                        /* eq. 18 */
        double var_k = k;                                     /* eq. 20 */
        double s2 = var_k / (g * g);                          /* eq. 21 */
        if (k > 0.0) { weight[i] = x / s2; if (variance) variance[i] = s2; }
        else { weight[i] = 0.0; if (variance) variance[i] = NAN; ++masked; }
    }
    return masked;
}

int oracle_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
