// nested.cu -- device-resident nested sampling: the consumer the batched likelihood was shaped for.
//
// PAPER.md:134-139 (section 3, steps iii-vii): pick parameters from the prior, compute the
// likelihood, accumulate the posterior, repeat until the parameter space is sufficiently
// sampled; PAPER.md:170, 184-186 (section 3.2): the sampler is Nested Sampling (Skilling 2004,
// 2006), which also yields the evidence (eq. 13).  The paper hands this to the MultiNest
// library, one likelihood call per proposed vector.  Here the live points, their likelihoods,
// the proposal batch, the evidence accumulators and the dead points all stay on the device; a
// round proposes a whole batch inside the current likelihood contour, calls lensed_loglike ONCE
// on it (through the public ABI: this file is a client of include/lensed.h), and consumes the
// batch in order against the rising threshold; only a 64-byte state record comes back, every
// few rounds, to test convergence.  Bound for the constrained draw: MultiNest's ellipsoid
// around the live points, a single one (reading N1).
//
// Per round (K candidates, N live points, d free parameters), all sampler arithmetic in FP64:
//   ns_bound_kernel    mean, covariance, Cholesky factor G, scale s: {m + s G y, |y| <= 1}
//   ns_propose_kernel  x = m + s r^(1/d) G z/|z|, redrawn up to 16 times until inside the unit
//                      cube; theta = lo + x (hi - lo) rounded to float
//   lensed_image_plane_prior (optional), lensed_loglike                      <- the hot path
//   ns_update_kernel   for j = 0..K-1: if L_j > min_i L_i, the worst live point dies with weight
//                      X_(k-1) - X_k, X_k = e^(-k/N), Z and the information H (Skilling 2006
//                      eq. 2.11) are updated and candidate j takes its place
// then ns_final_kernel adds the live points (weight X_k / N each) and normalises the weights.
// Random numbers: Philox4x32-10 (Salmon et al. 2011) keyed by the seed, counters = (round,
// candidate, try, stream), restated here from the published algorithm; the CPU oracle states
// it again on its side, so both draw the same numbers.
#include "../../include/lensed.h"
#include "lensed_internal.h"

#include <math.h>
#include <stdint.h>

#include <algorithm>
#include <vector>

namespace lensed {
namespace {

constexpr int kMaxFree = 48;         // free parameters (the paper's largest model has 35)
constexpr int kMaxLive = 4096;       // live points (their logL sit in shared memory during the update)
constexpr int kTries = 16;
constexpr int kStreamInit = 0, kStreamDir = 1, kStreamRadius = 2;
constexpr double kTwoPi = 6.283185307179586476925286766559;

struct NsState {
    double ln_z, ln_x, info, max_logl;
    long long n_dead, n_written;
    int done, rounds;
};

struct NsProblem {
    const double *lo, *hi;           // [P] device
    const int *free_idx;             // [d] device: parameter index of each free dimension
    int P, d, N, K;
    double enlarge, ln_tol;
    unsigned long long seed;
};

// ---- Philox4x32-10 ----------------------------------------------------------------------------
struct U4 { uint32_t x, y, z, w; };

__host__ __device__ inline U4 philox4x32(U4 c, uint32_t k0, uint32_t k1)
{
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c.x, p1 = (uint64_t)0xCD9E8D57u * c.z;
        c = U4{(uint32_t)(p1 >> 32) ^ c.y ^ k0, (uint32_t)p1, (uint32_t)(p0 >> 32) ^ c.w ^ k1, (uint32_t)p0};
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return c;
}

__host__ __device__ inline double unit(uint32_t x) { return ((double)x + 0.5) * (1.0 / 4294967296.0); }

__device__ inline void uniforms4(unsigned long long seed, uint32_t stream, uint32_t a, uint32_t b, uint32_t c, double (&u)[4])
{
    const U4 w = philox4x32(U4{a, b, c, stream}, (uint32_t)seed, (uint32_t)(seed >> 32));
    u[0] = unit(w.x); u[1] = unit(w.y); u[2] = unit(w.z); u[3] = unit(w.w);
}

__device__ inline void normals4(unsigned long long seed, uint32_t stream, uint32_t a, uint32_t b, uint32_t c, double (&z)[4])
{
    double u[4];
    uniforms4(seed, stream, a, b, c, u);
    const double r0 = sqrt(-2.0 * log(u[0])), r1 = sqrt(-2.0 * log(u[2]));
    double s0, c0, s1, c1;
    sincos(kTwoPi * u[1], &s0, &c0);
    sincos(kTwoPi * u[3], &s1, &c1);
    z[0] = r0 * c0; z[1] = r0 * s0; z[2] = r1 * c1; z[3] = r1 * s1;
}

// theta = lo + u (hi - lo) on the free dimensions, lo on the fixed ones, rounded to float
__device__ inline void write_theta(const NsProblem &pb, const double *u, float *theta)
{
    for (int p = 0; p < pb.P; ++p) theta[p] = (float)pb.lo[p];
    for (int k = 0; k < pb.d; ++k) {
        const int p = pb.free_idx[k];
        theta[p] = (float)(pb.lo[p] + u[k] * (pb.hi[p] - pb.lo[p]));
    }
}

__global__ void ns_init_kernel(NsProblem pb, double *U, float *theta, NsState *st)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) *st = NsState{-INFINITY, 0.0, 0.0, -INFINITY, 0, 0, 0, 0};
    if (i >= pb.N) return;
    double u[kMaxFree];
    for (int blk = 0; 4 * blk < pb.d; ++blk) {
        double w[4];
        uniforms4(pb.seed, kStreamInit, (uint32_t)i, (uint32_t)blk, 0u, w);
        for (int e = 0; e < 4 && 4 * blk + e < pb.d; ++e) u[4 * blk + e] = w[e];
    }
    for (int k = 0; k < pb.d; ++k) U[(size_t)i * pb.d + k] = u[k];
    write_theta(pb, u, theta + (size_t)i * pb.P);
}

// ---- bound: one block ------------------------------------------------------------------------
// out: m[d], G[d][d] (lower triangle, row-major), s
__global__ void __launch_bounds__(256) ns_bound_kernel(NsProblem pb, const double *U, double *m, double *G, double *s,
                                                       const NsState *st)
{
    if (st->done) return;
    __shared__ double sm[kMaxFree];
    __shared__ double sC[kMaxFree * kMaxFree];
    __shared__ double sred[256];
    const int d = pb.d, N = pb.N, t = threadIdx.x;
    for (int k = t; k < d; k += 256) {
        double a = 0.0;
        for (int i = 0; i < N; ++i) a += U[(size_t)i * d + k];
        sm[k] = a / N;
    }
    __syncthreads();
    for (int e = t; e < d * d; e += 256) {
        const int a = e / d, b = e - a * d;
        if (b > a) continue;
        double acc = 0.0;
        for (int i = 0; i < N; ++i) acc += (U[(size_t)i * d + a] - sm[a]) * (U[(size_t)i * d + b] - sm[b]);
        sC[a * d + b] = acc / N + (a == b ? 1e-30 : 0.0);
    }
    __syncthreads();
    // Cholesky, column by column, in place in the lower triangle
    for (int j = 0; j < d; ++j) {
        if (t == 0) {
            double a = sC[j * d + j];
            for (int k = 0; k < j; ++k) a -= sC[j * d + k] * sC[j * d + k];
            sC[j * d + j] = sqrt(fmax(a, 1e-300));
        }
        __syncthreads();
        for (int i = j + 1 + t; i < d; i += 256) {
            double a = sC[i * d + j];
            for (int k = 0; k < j; ++k) a -= sC[i * d + k] * sC[j * d + k];
            sC[i * d + j] = a / sC[j * d + j];
        }
        __syncthreads();
    }
    // largest Mahalanobis radius of a live point: forward substitution y = G^-1 (u - m)
    double rmax = 0.0;
    for (int i = t; i < N; i += 256) {
        double y[kMaxFree], r2 = 0.0;
        for (int a = 0; a < d; ++a) {
            double v = U[(size_t)i * d + a] - sm[a];
            for (int b = 0; b < a; ++b) v -= sC[a * d + b] * y[b];
            y[a] = v / sC[a * d + a];
            r2 += y[a] * y[a];
        }
        rmax = fmax(rmax, r2);
    }
    sred[t] = rmax;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (t < o) sred[t] = fmax(sred[t], sred[t + o]);
        __syncthreads();
    }
    for (int k = t; k < d; k += 256) m[k] = sm[k];
    for (int e = t; e < d * d; e += 256) G[e] = (e % d) <= (e / d) ? sC[e] : 0.0;
    if (t == 0) *s = pb.enlarge * sqrt(sred[0]);
}

__global__ void ns_propose_kernel(NsProblem pb, const double *m, const double *G, const double *s, double *Uc,
                                  float *theta_c, const NsState *st)
{
    if (st->done) return;
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= pb.K) return;
    const int d = pb.d;
    const uint32_t rnd = (uint32_t)st->rounds;
    const double scale = *s;
    double x[kMaxFree];
    bool ok = false;
    for (int t = 0; t < kTries && !ok; ++t) {
        double z[kMaxFree + 3], n2 = 0.0;
        for (int blk = 0; 4 * blk < d; ++blk) {
            double w[4];
            normals4(pb.seed, kStreamDir, rnd, (uint32_t)j, (uint32_t)(t * 64 + blk), w);
            for (int e = 0; e < 4; ++e) z[4 * blk + e] = w[e];
        }
        for (int a = 0; a < d; ++a) n2 += z[a] * z[a];
        double u4[4];
        uniforms4(pb.seed, kStreamRadius, rnd, (uint32_t)j, (uint32_t)t, u4);
        const double f = pow(u4[0], 1.0 / d) / sqrt(n2);
        ok = true;
        for (int a = 0; a < d; ++a) {
            double v = 0.0;
            for (int b = 0; b <= a; ++b) v += G[a * d + b] * (z[b] * f);
            x[a] = m[a] + scale * v;
            ok = ok && x[a] > 0.0 && x[a] < 1.0;
        }
    }
    double *uo = Uc + (size_t)j * d;
    if (ok) {
        for (int a = 0; a < d; ++a) uo[a] = x[a];
    } else {                                   // void candidate: never accepted (ns_update_kernel)
        for (int a = 0; a < d; ++a) { uo[a] = nan(""); x[a] = 0.5; }
    }
    write_theta(pb, x, theta_c + (size_t)j * pb.P);
}

// block-wide argmin with the lower index winning ties (numpy's argmin); result in s_val[0], s_idx[0]
__device__ inline void block_argmin(const float *logl, int N, float *s_val, int *s_idx)
{
    const int t = threadIdx.x;
    float v = INFINITY;
    int at = 0x7fffffff;
    for (int i = t; i < N; i += 256) {
        const float l = logl[i];
        if (l < v || (l == v && i < at)) { v = l; at = i; }
    }
    s_val[t] = v; s_idx[t] = at;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (t < o) {
            const float l = s_val[t + o];
            const int i = s_idx[t + o];
            if (l < s_val[t] || (l == s_val[t] && i < s_idx[t])) { s_val[t] = l; s_idx[t] = i; }
        }
        __syncthreads();
    }
}

// ln Z and H after adding one point of likelihood ls and log-weight lw (Skilling 2006 eq. 2.11)
__device__ inline void accumulate(NsState &st, double ls, double lw)
{
    const double a = ls + lw;
    const double hi = fmax(st.ln_z, a), lo = fmin(st.ln_z, a);
    const double ln_z_new = isinf(lo) && lo < 0 ? hi : hi + log1p(exp(lo - hi));
    double info = exp(a - ln_z_new) * ls - ln_z_new;
    if (isfinite(st.ln_z)) info += exp(st.ln_z - ln_z_new) * (st.info + st.ln_z);
    st.info = info;
    st.ln_z = ln_z_new;
}

struct NsOut { float *samples, *logl, *logw; long long cap; };

__global__ void __launch_bounds__(256) ns_update_kernel(NsProblem pb, double *U, float *theta, float *logl_live,
                                                        const double *Uc, const float *theta_c, const float *logl_c,
                                                        NsOut out, NsState *st_g)
{
    if (st_g->done) return;
    __shared__ float s_logl[kMaxLive];
    __shared__ float s_val[256];
    __shared__ int s_idx[256];
    __shared__ NsState st;
    const int t = threadIdx.x, N = pb.N, d = pb.d, P = pb.P;
    for (int i = t; i < N; i += 256) s_logl[i] = logl_live[i];
    if (t == 0) st = *st_g;
    __syncthreads();
    block_argmin(s_logl, N, s_val, s_idx);
    const double ln_shell = log(-expm1(-1.0 / N));          // ln (X_(k-1) - X_k) - ln X_(k-1)
    for (int j = 0; j < pb.K; ++j) {
        const bool is_void = isnan(Uc[(size_t)j * d]);
        const float cl = is_void ? -INFINITY : logl_c[j];
        const float lmin = s_val[0];
        const int worst = s_idx[0];
        if (!(cl > lmin)) continue;                          // block-uniform
        __syncthreads();
        if (t == 0) {
            accumulate(st, (double)lmin, st.ln_x + ln_shell);
            st.ln_x -= 1.0 / N;
        }
        const long long slot = st.n_dead;                    // read before thread 0 bumps it (barrier below)
        if (slot < out.cap) {
            for (int p = t; p < P; p += 256) out.samples[(size_t)slot * P + p] = theta[(size_t)worst * P + p];
            if (t == 0) {
                out.logl[slot] = lmin;
                out.logw[slot] = (float)(st.ln_x + 1.0 / N + ln_shell);     // this point's ln w (ln_x already stepped)
            }
        }
        __syncthreads();
        for (int k = t; k < d; k += 256) U[(size_t)worst * d + k] = Uc[(size_t)j * d + k];
        for (int p = t; p < P; p += 256) theta[(size_t)worst * P + p] = theta_c[(size_t)j * P + p];
        if (t == 0) { s_logl[worst] = cl; st.n_dead += 1; }
        __syncthreads();
        block_argmin(s_logl, N, s_val, s_idx);
    }
    // convergence: max_i L_i X_k < tol Z
    float v = -INFINITY;
    for (int i = t; i < N; i += 256) v = fmaxf(v, s_logl[i]);
    __syncthreads();
    s_val[t] = v;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (t < o) s_val[t] = fmaxf(s_val[t], s_val[t + o]);
        __syncthreads();
    }
    for (int i = t; i < N; i += 256) logl_live[i] = s_logl[i];
    if (t == 0) {
        st.max_logl = (double)s_val[0];
        st.rounds += 1;
        st.done = (st.max_logl + st.ln_x < st.ln_z + pb.ln_tol) ? 1 : 0;
        st.n_written = st.n_dead < out.cap ? st.n_dead : out.cap;
        *st_g = st;
    }
}

// the live points join the dead, lowest likelihood first, weight X_k / N each; then the
// log-weights are normalised: logw <- ln(L w / Z)
__global__ void __launch_bounds__(256) ns_final_kernel(NsProblem pb, const float *theta, const float *logl_live,
                                                       NsOut out, NsState *st_g)
{
    __shared__ float s_logl[kMaxLive];
    __shared__ float s_val[256];
    __shared__ int s_idx[256];
    __shared__ NsState st;
    const int t = threadIdx.x, N = pb.N, P = pb.P;
    for (int i = t; i < N; i += 256) s_logl[i] = logl_live[i];
    if (t == 0) st = *st_g;
    __syncthreads();
    const double lw = st.ln_x - log((double)N);
    long long slot = st.n_dead;
    for (int n = 0; n < N; ++n, ++slot) {
        block_argmin(s_logl, N, s_val, s_idx);
        const int i = s_idx[0];
        const float li = s_val[0];
        if (t == 0) accumulate(st, (double)li, lw);
        if (slot < out.cap) {
            for (int p = t; p < P; p += 256) out.samples[(size_t)slot * P + p] = theta[(size_t)i * P + p];
            if (t == 0) { out.logl[slot] = li; out.logw[slot] = (float)lw; }
        }
        __syncthreads();
        if (t == 0) s_logl[i] = INFINITY;
        __syncthreads();
    }
    const long long n_out = slot < out.cap ? slot : out.cap;
    __syncthreads();
    for (long long k = t; k < n_out; k += 256) out.logw[k] = (float)((double)out.logl[k] + (double)out.logw[k] - st.ln_z);
    if (t == 0) { st.n_written = n_out; *st_g = st; }
}

struct Buffers {
    std::vector<void *> ptrs;
    ~Buffers() { for (void *p : ptrs) cudaFree(p); }
    template <class T> cudaError_t get(T **out, size_t n)
    {
        void *p = nullptr;
        cudaError_t e = cudaMalloc(&p, std::max<size_t>(n, 1) * sizeof(T));
        if (e == cudaSuccess) { ptrs.push_back(p); *out = (T *)p; }
        return e;
    }
};

}  // namespace
}  // namespace lensed

using namespace lensed;

extern "C" lensed_status lensed_ns_run(lensed_handle *h, const float *prior_lo, const float *prior_hi,
                                       const int *image_plane_sources, int n_image_plane,
                                       const lensed_ns_options *opt, lensed_ns_result *res,
                                       float *samples_dev, float *logl_dev, float *logw_dev, long long capacity,
                                       void *stream)
{
    if (!h || !prior_lo || !prior_hi || !opt || !res) return (lensed_status)handle_fail(h, LENSED_EINVAL, "lensed_ns_run: null argument");
    const int P = lensed_num_params(h);
    std::vector<double> lo(P), hi(P);
    std::vector<int> free_idx;
    for (int p = 0; p < P; ++p) {
        lo[p] = prior_lo[p]; hi[p] = prior_hi[p];
        if (!isfinite(lo[p]) || !isfinite(hi[p]) || hi[p] < lo[p])
            return (lensed_status)handle_fail(h, LENSED_EINVAL, "lensed_ns_run: prior of parameter %d is [%g, %g]", p, lo[p], hi[p]);
        if (hi[p] > lo[p]) free_idx.push_back(p);
    }
    const int d = (int)free_idx.size();
    if (d < 1) return (lensed_status)handle_fail(h, LENSED_EINVAL, "lensed_ns_run: no free parameter (every prior has lo == hi)");
    if (d > kMaxFree) return (lensed_status)handle_fail(h, LENSED_EUNSUPPORTED, "lensed_ns_run: %d free parameters > %d", d, kMaxFree);
    if (opt->n_live < d + 1 || opt->n_live > kMaxLive)
        return (lensed_status)handle_fail(h, LENSED_EINVAL, "lensed_ns_run: n_live = %d outside [%d, %d]", opt->n_live, d + 1, kMaxLive);
    if (opt->batch < 1 || opt->max_rounds < 1 || !(opt->tol > 0.0) || !(opt->enlarge >= 1.0))
        return (lensed_status)handle_fail(h, LENSED_EINVAL, "lensed_ns_run: batch >= 1, max_rounds >= 1, tol > 0, enlarge >= 1 required");
    if (capacity < 0 || (capacity > 0 && (!samples_dev || !logl_dev || !logw_dev)))
        return (lensed_status)handle_fail(h, LENSED_EINVAL, "lensed_ns_run: capacity %lld needs all three output arrays", capacity);
    if (n_image_plane < 0 || (n_image_plane > 0 && !image_plane_sources))
        return (lensed_status)handle_fail(h, LENSED_EINVAL, "lensed_ns_run: image_plane_sources missing");

    cudaStream_t st = (cudaStream_t)stream;
    const int N = opt->n_live, K = opt->batch;
#define NS_CU(call)                                                                                       \
    do {                                                                                                  \
        cudaError_t e_ = (call);                                                                          \
        if (e_ != cudaSuccess)                                                                            \
            return (lensed_status)handle_fail(h, e_ == cudaErrorMemoryAllocation ? LENSED_ENOMEM : LENSED_ECUDA, "%s: %s", #call, \
                               cudaGetErrorString(e_));                                                   \
    } while (0)
#define NS_OK(call) do { lensed_status s_ = (call); if (s_ != LENSED_OK) return s_; } while (0)
    NS_CU(cudaSetDevice(handle_device(h)));
    Buffers buf;
    double *d_lo, *d_hi, *d_U, *d_Uc, *d_m, *d_G, *d_s;
    int *d_free;
    float *d_theta, *d_theta_c, *d_logl, *d_logl_c;
    NsState *d_state;
    NS_CU(buf.get(&d_lo, P)); NS_CU(buf.get(&d_hi, P)); NS_CU(buf.get(&d_free, d));
    NS_CU(buf.get(&d_U, (size_t)N * d)); NS_CU(buf.get(&d_Uc, (size_t)K * d));
    NS_CU(buf.get(&d_m, d)); NS_CU(buf.get(&d_G, (size_t)d * d)); NS_CU(buf.get(&d_s, 1));
    NS_CU(buf.get(&d_theta, (size_t)N * P)); NS_CU(buf.get(&d_theta_c, (size_t)K * P));
    NS_CU(buf.get(&d_logl, N)); NS_CU(buf.get(&d_logl_c, K)); NS_CU(buf.get(&d_state, 1));
    NS_CU(cudaMemcpyAsync(d_lo, lo.data(), P * sizeof(double), cudaMemcpyHostToDevice, st));
    NS_CU(cudaMemcpyAsync(d_hi, hi.data(), P * sizeof(double), cudaMemcpyHostToDevice, st));
    NS_CU(cudaMemcpyAsync(d_free, free_idx.data(), d * sizeof(int), cudaMemcpyHostToDevice, st));
    NS_CU(cudaStreamSynchronize(st));                       // the host vectors above go out of scope otherwise

    const NsProblem pb{d_lo, d_hi, d_free, P, d, N, K, opt->enlarge, log(opt->tol), opt->seed};
    const NsOut out{samples_dev, logl_dev, logw_dev, capacity};

    // step 0: the live points from the prior
    ns_init_kernel<<<(N + 127) / 128, 128, 0, st>>>(pb, d_U, d_theta, d_state);
    NS_CU(cudaGetLastError());
    if (n_image_plane > 0) NS_OK(lensed_image_plane_prior(h, d_theta, N, image_plane_sources, n_image_plane, stream));
    NS_OK(lensed_loglike(h, d_theta, N, d_logl, stream));

    NsState host{};
    long long rounds_launched = 0;
    const int check_every = 4;
    for (;;) {
        for (int r = 0; r < check_every; ++r, ++rounds_launched) {
            ns_bound_kernel<<<1, 256, 0, st>>>(pb, d_U, d_m, d_G, d_s, d_state);
            ns_propose_kernel<<<(K + 127) / 128, 128, 0, st>>>(pb, d_m, d_G, d_s, d_Uc, d_theta_c, d_state);
            NS_CU(cudaGetLastError());
            if (n_image_plane > 0)
                NS_OK(lensed_image_plane_prior(h, d_theta_c, K, image_plane_sources, n_image_plane, stream));
            NS_OK(lensed_loglike(h, d_theta_c, K, d_logl_c, stream));
            ns_update_kernel<<<1, 256, 0, st>>>(pb, d_U, d_theta, d_logl, d_Uc, d_theta_c, d_logl_c, out, d_state);
            NS_CU(cudaGetLastError());
        }
        NS_CU(cudaMemcpyAsync(&host, d_state, sizeof host, cudaMemcpyDeviceToHost, st));
        NS_CU(cudaStreamSynchronize(st));
        if (host.done || host.rounds >= opt->max_rounds) break;
    }
    const int converged = host.done;
    const long long n_dead = host.n_dead, n_rounds = host.rounds;
    ns_final_kernel<<<1, 256, 0, st>>>(pb, d_theta, d_logl, out, d_state);
    NS_CU(cudaGetLastError());
    NS_CU(cudaMemcpyAsync(&host, d_state, sizeof host, cudaMemcpyDeviceToHost, st));
    NS_CU(cudaStreamSynchronize(st));
#undef NS_CU
#undef NS_OK
    res->ln_z = host.ln_z;
    res->information = host.info;
    res->ln_z_err = sqrt(fmax(host.info, 0.0) / N);
    res->n_rounds = n_rounds;
    res->n_likelihood = (long long)N + rounds_launched * K;
    res->n_dead = n_dead;
    res->n_samples = host.n_written;
    res->converged = converged;
    return LENSED_OK;
}

// test hook: the generator itself (tests pin it on the published known-answer vectors)
extern "C" void lensed_ns_philox(const unsigned *counter, const unsigned *key, unsigned *out)
{
    const U4 r = philox4x32(U4{counter[0], counter[1], counter[2], counter[3]}, key[0], key[1]);
    out[0] = r.x; out[1] = r.y; out[2] = r.z; out[3] = r.w;
}
