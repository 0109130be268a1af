// deflect.cu -- the lens equation for single points: y = x - sum_lenses alpha(x)
// (eq. 1), in double precision straight from the parameter vectors, arcsec.
//
// This is the map of the paper's image-plane priors (section 5): "first
// sampling a position on the image plane, mapping it to the source plane, and assigning it to
// the source".  lensed_deflect maps K points per vector; lensed_image_plane_prior does the
// assignment in place: the (x, y) parameters of the listed source components hold image-plane
// positions on entry and the corresponding source-plane positions on return.
// The work is B x K points, nothing next to the likelihood itself, so it runs in FP64.
#include "lensed_internal.h"
#include <math.h>

namespace lensed {
namespace {

constexpr double kPiD = 3.141592653589793238462643383279502884;

// sum of the deflections of the vector's lenses at (x, y); false if a lens is outside its domain
__device__ bool deflection_sum(const Program &prog, const float *par, double x, double y, double &ax, double &ay)
{
    ax = 0.0; ay = 0.0;
    for (int m = 0; m < prog.n_models; ++m) {
        const int kind = prog.kind[m];
        if (kind > K_SHEAR) continue;
        const float *pf = par + prog.par_off[m];
        double p[5];
        const int np = kind_num_params(kind);
        for (int i = 0; i < np; ++i) {
            p[i] = (double)pf[i];
            if (!isfinite(p[i])) return false;
        }
        switch (kind) {
        case K_SIS: {                                   // R3
            if (!(p[2] >= 0.0)) return false;
            const double u = x - p[0], v = y - p[1], r = sqrt(u * u + v * v);
            if (r > 0.0) { ax += p[2] * u / r; ay += p[2] * v / r; }
            break;
        }
        case K_POINT: {                                 // R3
            if (!(p[2] >= 0.0)) return false;
            const double u = x - p[0], v = y - p[1], r2 = u * u + v * v;
            if (r2 > 0.0) { ax += p[2] * p[2] * u / r2; ay += p[2] * p[2] * v / r2; }
            break;
        }
        case K_SHEAR:                                   // R4: about the image centre
            ax += p[0] * x + p[1] * y;
            ay += p[1] * x - p[0] * y;
            break;
        default: {                                      // K_SIE, R2
            const double b = p[2], q = p[3];
            if (!(b >= 0.0) || !(q > 0.0) || !(q <= 1.0)) return false;
            double s, c;
            sincos(p[4] * (kPiD / 180.0), &s, &c);
            const double dx = x - p[0], dy = y - p[1];
            const double u = c * dx + s * dy, v = -s * dx + c * dy;
            const double psi = sqrt(q * q * u * u + v * v);
            if (psi > 0.0) {
                const double qp = sqrt((1.0 - q) * (1.0 + q)), sq = sqrt(q);
                double au, av;
                if (qp < 1e-7) { au = b * sq * u / psi; av = b * sq * v / psi; }      // q -> 1
                else { const double A = b * sq / qp; au = A * atan(qp * u / psi); av = A * atanh(qp * v / psi); }
                ax += c * au - s * av;
                ay += s * au + c * av;
            }
            break;
        }
        }
    }
    return true;
}

__global__ void deflect_kernel(Program prog, const float *params, int B, const float *xy, int K, float *out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)B * K) return;
    const int b = (int)(i / K);
    const double x = (double)xy[2 * i], y = (double)xy[2 * i + 1];
    double ax, ay;
    const bool ok = isfinite(x) && isfinite(y) && deflection_sum(prog, params + (size_t)b * prog.P, x, y, ax, ay);
    out[2 * i] = ok ? (float)(x - ax) : nanf("");
    out[2 * i + 1] = ok ? (float)(y - ay) : nanf("");
}

struct PriorList { int n; int par_off[kMaxModels]; };

// one thread per (vector, listed source): its (x, y) parameters are replaced in place; lens
// parameters are never written, so the threads of a vector do not interfere
__global__ void image_plane_prior_kernel(Program prog, PriorList list, float *params, int B)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)B * list.n) return;
    const int b = (int)(i / list.n), k = (int)(i - (long long)b * list.n);
    float *par = params + (size_t)b * prog.P;
    float *pos = par + list.par_off[k];
    const double x = (double)pos[0], y = (double)pos[1];
    double ax, ay;
    const bool ok = isfinite(x) && isfinite(y) && deflection_sum(prog, par, x, y, ax, ay);
    pos[0] = ok ? (float)(x - ax) : nanf("");
    pos[1] = ok ? (float)(y - ay) : nanf("");
}

}  // namespace

cudaError_t launch_deflect(const Program &prog, const float *params, int B, const float *xy, int K, float *out,
                           cudaStream_t st)
{
    const long long n = (long long)B * K;
    if (n < 1) return cudaSuccess;
    deflect_kernel<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(prog, params, B, xy, K, out);
    return cudaGetLastError();
}

cudaError_t launch_image_plane_prior(const Program &prog, const int *par_offs, int n_src, float *params, int B,
                                     cudaStream_t st)
{
    PriorList list;
    list.n = n_src;
    for (int i = 0; i < n_src; ++i) list.par_off[i] = par_offs[i];
    const long long n = (long long)B * n_src;
    if (n < 1) return cudaSuccess;
    image_plane_prior_kernel<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(prog, list, params, B);
    return cudaGetLastError();
}

}  // namespace lensed
