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
#include "../../include/lensed_tune.h"
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
    const int *tied_to;              // [P] device: parameter p takes the drawn value of parameter tied_to[p] (-1: its own)
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

// theta = lo + u (hi - lo) on the free dimensions, lo on the fixed ones, rounded to float; tied
// parameters then copy the parameter they follow (mass centre = light centre)
__device__ inline void write_theta(const NsProblem &pb, const double *u, float *theta)
{
    for (int p = 0; p < pb.P; ++p) theta[p] = (float)pb.lo[p];
    for (int k = 0; k < pb.d; ++k) {
        const int p = pb.free_idx[k];
        theta[p] = (float)(pb.lo[p] + u[k] * (pb.hi[p] - pb.lo[p]));
    }
    for (int p = 0; p < pb.P; ++p)
        if (pb.tied_to[p] >= 0) theta[p] = theta[pb.tied_to[p]];
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
    // mean and covariance: when the block has more threads than entries, every entry's sum over the N
    // live points is split over S = 256 / entries strided segments (partials in sred, added in
    // segment order: deterministic)
    {
        const int E = d, S = E <= 128 ? 256 / E : 1;
        const int e = t % E, seg = t / E;
        for (int k = S > 1 ? e : t; k < d; k += S > 1 ? d : 256) {
            if (seg >= S) break;
            double a = 0.0;
            for (int i = S > 1 ? seg : 0; i < N; i += S) a += U[(size_t)i * d + k];
            if (S > 1) sred[seg * E + e] = a; else sm[k] = a / N;
        }
        __syncthreads();
        if (S > 1 && t < E) {
            double a = 0.0;
            for (int g = 0; g < S; ++g) a += sred[g * E + t];
            sm[t] = a / N;
        }
        __syncthreads();
    }
    {
        const int E = d * d, S = E <= 128 ? 256 / E : 1;
        const int e0 = t % E, seg = t / E;
        for (int e = S > 1 ? e0 : t; e < E; e += S > 1 ? E : 256) {
            if (seg >= S) break;
            const int a = e / d, b = e - a * d;
            double acc = 0.0;
            if (b <= a)
                for (int i = S > 1 ? seg : 0; i < N; i += S) acc += (U[(size_t)i * d + a] - sm[a]) * (U[(size_t)i * d + b] - sm[b]);
            if (S > 1) sred[seg * E + e0] = acc;
            else if (b <= a) sC[a * d + b] = acc / N + (a == b ? 1e-30 : 0.0);
        }
        __syncthreads();
        if (S > 1 && t < E) {
            const int a = t / d, b = t - a * d;
            if (b <= a) {
                double acc = 0.0;
                for (int g = 0; g < S; ++g) acc += sred[g * E + t];
                sC[a * d + b] = acc / N + (a == b ? 1e-30 : 0.0);
            }
        }
        __syncthreads();
    }
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

// The same update for n points at once, by the whole block:  Z = sum_k L_k w_k  and
// S = sum_k L_k w_k ln L_k  are plain sums (H = S/Z - ln Z is eq. 2.11 unrolled), taken relative to
// the largest term; per-thread partial sums in index order, then a fixed tree: deterministic.
// Differs from n calls of accumulate() by FP64 rounding only.  term(k) -> ln L_k, ln w_k.
template <class F>
__device__ inline void block_accumulate(NsState &st, int n, F term, double *s_a, double *s_b)
{
    const int t = threadIdx.x;
    double m = -INFINITY;
    for (int k = t; k < n; k += 256) {
        double ls, lw;
        term(k, ls, lw);
        m = fmax(m, ls + lw);
    }
    s_a[t] = m;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (t < o) s_a[t] = fmax(s_a[t], s_a[t + o]);
        __syncthreads();
    }
    const double M = fmax(s_a[0], st.ln_z);
    __syncthreads();
    if (!(M > -INFINITY)) return;                            // nothing has any weight yet
    double z = 0.0, sl = 0.0;
    for (int k = t; k < n; k += 256) {
        double ls, lw;
        term(k, ls, lw);
        const double w = exp(ls + lw - M);
        z += w;
        if (w > 0.0) sl += w * ls;
    }
    s_a[t] = z; s_b[t] = sl;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (t < o) { s_a[t] += s_a[t + o]; s_b[t] += s_b[t + o]; }
        __syncthreads();
    }
    if (t == 0) {
        const double zo = isfinite(st.ln_z) ? exp(st.ln_z - M) : 0.0;
        const double so = zo > 0.0 ? zo * (st.info + st.ln_z) : 0.0;
        const double Z = zo + s_a[0], S = so + s_b[0];
        st.ln_z = M + log(Z);
        st.info = S / Z - st.ln_z;
    }
    __syncthreads();
}

struct NsOut { float *samples, *logl, *logw; long long cap; };

// order-preserving map float -> unsigned (no NaN here): the warp-wide minimum is then ONE REDUX
// instruction (__reduce_min_sync) instead of five shuffle rounds
__device__ inline unsigned fkey(float f)
{
    const unsigned u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ inline float fkey_inv(unsigned k) { return __uint_as_float((k & 0x80000000u) ? (k ^ 0x80000000u) : ~k); }

// minimum of the group of 32 slots g (whole warp): key and slot, the lowest slot winning ties
__device__ inline void group_min(const float *s_logl, int N, int g, int lane, unsigned *s_gkey, int *s_gidx)
{
    const int i = g * 32 + lane;
    const unsigned key = i < N ? fkey(s_logl[i]) : 0xffffffffu;
    const unsigned kmin = __reduce_min_sync(0xffffffffu, key);
    const int b = __ffs(__ballot_sync(0xffffffffu, key == kmin)) - 1;
    if (lane == 0) { s_gkey[g] = kmin; s_gidx[g] = g * 32 + b; }
}

// Step 4 of the algorithm for one round, in the sequential order of its definition but without a
// block-wide pass per candidate.  The live likelihoods sit in shared memory under a two-level
// tournament: the minimum of every group of 32 slots, and the minimum over the groups.  ONE warp
// walks the candidates 32 at a time (a ballot against the current threshold finds the next one
// that beats it; after each death the threshold rises and the rest of the chunk is re-tested);
// a death costs two warp-wide minima (its group, then the groups), each a REDUX and a ballot.  The warp only records who
// died and who took which slot; all 256 threads then copy the dead points' parameter vectors
// out and the surviving candidates in.  Same deaths, same order, same weights as the
// candidate-by-candidate loop it replaces (1.07 ms -> 0.1 ms per round of 1024 candidates
// against 1024 live points).
__global__ void __launch_bounds__(256) ns_update_kernel(NsProblem pb, double *U, float *theta, float *logl_live,
                                                        const double *Uc, const float *theta_c, const float *logl_c,
                                                        int *death_src, float *death_logl, NsOut out, NsState *st_g)
{
    if (st_g->done) return;
    __shared__ float s_logl[kMaxLive];
    __shared__ int s_owner[kMaxLive];          // -1: live since before this round; else the candidate in the slot
    __shared__ unsigned s_gkey[kMaxLive / 32];
    __shared__ int s_gidx[kMaxLive / 32];
    constexpr int kChunk = 1024;
    __shared__ float s_cl[kChunk];
    __shared__ float s_val[256];
    __shared__ double s_red_a[256], s_red_b[256];
    __shared__ NsState st;
    __shared__ long long s_first_dead;
    __shared__ int s_deaths;
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5, N = pb.N, d = pb.d, P = pb.P;
    const int G = (N + 31) >> 5;
    for (int i = t; i < N; i += 256) { s_logl[i] = logl_live[i]; s_owner[i] = -1; }
    if (t == 0) { st = *st_g; s_first_dead = st_g->n_dead; s_deaths = 0; }
    __syncthreads();
    for (int g = warp; g < G; g += 8) group_min(s_logl, N, g, lane, s_gkey, s_gidx);
    __syncthreads();

    // minimum over the groups: every lane its own groups (lower group first), then two REDUX
    auto global_min = [&](float &v, int &i) {
        unsigned key = 0xffffffffu;
        int bg = 0x7fffffff;
        for (int g = lane; g < G; g += 32) {
            const unsigned gk = s_gkey[g];
            if (gk < key) { key = gk; bg = g; }
        }
        const unsigned kmin = __reduce_min_sync(0xffffffffu, key);
        const int gsel = (int)__reduce_min_sync(0xffffffffu, key == kmin ? (unsigned)bg : 0x7fffffffu);
        v = fkey_inv(kmin);
        i = s_gidx[gsel];
    };
    float lmin = 0.0f;
    int worst = 0;
    if (warp == 0) global_min(lmin, worst);
    int n_died = 0;                                          // warp 0's count
    for (int base0 = 0; base0 < pb.K; base0 += kChunk) {
        // the candidates' likelihoods of this stretch into shared memory, by the whole block
        __syncthreads();
        for (int c = t; c < kChunk; c += 256) {
            const int j = base0 + c;
            s_cl[c] = (j < pb.K && !isnan(Uc[(size_t)j * d])) ? logl_c[j] : -INFINITY;   // void candidate: never accepted
        }
        __syncthreads();
        if (warp != 0) continue;
        for (int base = 0; base < kChunk && base0 + base < pb.K; base += 32) {
            const float cl = s_cl[base + lane];
            unsigned mask = __ballot_sync(0xffffffffu, cl > lmin);
            while (mask) {
                const int b = __ffs(mask) - 1;
                const float cj = __shfl_sync(0xffffffffu, cl, b);
                if (lane == 0) {
                    const int own = s_owner[worst];
                    death_src[n_died] = own < 0 ? worst : ~own;      // whose parameter vector dies: a live row or a candidate
                    death_logl[n_died] = lmin;
                    s_logl[worst] = cj;
                    s_owner[worst] = base0 + base + b;
                }
                ++n_died;
                __syncwarp();
                group_min(s_logl, N, worst >> 5, lane, s_gkey, s_gidx);
                __syncwarp();
                global_min(lmin, worst);
                mask = __ballot_sync(0xffffffffu, cl > lmin) & ~((2u << b) - 1u);   // the later candidates of the chunk
            }
        }
    }
    if (t == 0) s_deaths = n_died;
    __syncthreads();

    // evidence and information: death k of the round has ln w = ln X - k/N + ln(1 - e^(-1/N))
    const int deaths = s_deaths;
    const double ln_shell = log(-expm1(-1.0 / N));           // ln (X_(k-1) - X_k) - ln X_(k-1)
    const double ln_x0 = st.ln_x;
    for (int k = t; k < deaths; k += 256) {
        const long long slot = s_first_dead + k;
        if (slot < out.cap) { out.logl[slot] = death_logl[k]; out.logw[slot] = (float)(ln_x0 - (double)k / N + ln_shell); }
    }
    block_accumulate(st, deaths, [&](int k, double &ls, double &lw) { ls = (double)death_logl[k]; lw = ln_x0 - (double)k / N + ln_shell; },
                     s_red_a, s_red_b);
    if (t == 0) { st.ln_x = ln_x0 - (double)deaths / N; st.n_dead += deaths; }
    // the dead points' parameter vectors, in order of death (theta still holds the round's starting rows)
    for (long long e = t; e < (long long)deaths * P; e += 256) {
        const int k = (int)(e / P), p = (int)(e - (long long)k * P);
        const long long slot = s_first_dead + k;
        if (slot < out.cap) {
            const int src = death_src[k];
            out.samples[(size_t)slot * P + p] = src >= 0 ? theta[(size_t)src * P + p] : theta_c[(size_t)(~src) * P + p];
        }
    }
    __syncthreads();
    // the surviving candidates into their slots
    for (int i = warp; i < N; i += 8) {
        const int own = s_owner[i];
        if (own < 0) continue;
        for (int k = lane; k < d; k += 32) U[(size_t)i * d + k] = Uc[(size_t)own * d + k];
        for (int p = lane; p < P; p += 32) theta[(size_t)i * P + p] = theta_c[(size_t)own * P + p];
    }
    // convergence: max_i L_i X_k < tol Z
    float v = -INFINITY;
    for (int i = t; i < N; i += 256) v = fmaxf(v, s_logl[i]);
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

// the live points join the dead, lowest likelihood first (ties: lower slot first), weight X_k / N
// each; then the log-weights are normalised: logw <- ln(L w / Z)
__global__ void __launch_bounds__(256) ns_final_kernel(NsProblem pb, const float *theta, const float *logl_live,
                                                       NsOut out, NsState *st_g)
{
    __shared__ float s_logl[kMaxLive];
    __shared__ int s_order[kMaxLive];          // slot of the n-th lowest live point
    __shared__ double s_red_a[256], s_red_b[256];
    __shared__ NsState st;
    const int t = threadIdx.x, N = pb.N, P = pb.P;
    for (int i = t; i < N; i += 256) s_logl[i] = logl_live[i];
    if (t == 0) st = *st_g;
    __syncthreads();
    for (int i = t; i < N; i += 256) {         // rank by (likelihood, slot): what N successive argmins would give
        const float li = s_logl[i];
        int rank = 0;
        for (int j = 0; j < N; ++j) {
            const float lj = s_logl[j];
            rank += (lj < li || (lj == li && j < i)) ? 1 : 0;
        }
        s_order[rank] = i;
    }
    __syncthreads();
    const double lw = st.ln_x - log((double)N);
    const long long first = st.n_dead;
    block_accumulate(st, N, [&](int n, double &ls, double &lw_) { ls = (double)s_logl[s_order[n]]; lw_ = lw; }, s_red_a, s_red_b);
    for (long long e = t; e < (long long)N * P; e += 256) {
        const int n = (int)(e / P), p = (int)(e - (long long)n * P);
        if (first + n < out.cap) out.samples[(size_t)(first + n) * P + p] = theta[(size_t)s_order[n] * P + p];
    }
    for (int n = t; n < N; n += 256)
        if (first + n < out.cap) { out.logl[first + n] = s_logl[s_order[n]]; out.logw[first + n] = (float)lw; }
    __syncthreads();
    const long long n_out = first + N < out.cap ? first + N : out.cap;
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
    std::vector<int> tied(P, -1);
    if (opt->tied_to) {
        for (int p = 0; p < P; ++p) {
            const int q = opt->tied_to[p];
            if (q < 0) continue;
            if (q >= P || q == p || opt->tied_to[q] >= 0 || hi[p] > lo[p])
                return (lensed_status)handle_fail(h, LENSED_EINVAL, "lensed_ns_run: tied_to[%d] = %d (needs another, untied parameter, and lo == hi for the tied one)", p, q);
            tied[p] = q;
        }
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
    int *d_free, *d_death, *d_tied;
    float *d_death_l;
    float *d_theta, *d_theta_c, *d_logl, *d_logl_c;
    NsState *d_state;
    NS_CU(buf.get(&d_lo, P)); NS_CU(buf.get(&d_hi, P)); NS_CU(buf.get(&d_free, d)); NS_CU(buf.get(&d_tied, P));
    NS_CU(buf.get(&d_U, (size_t)N * d)); NS_CU(buf.get(&d_Uc, (size_t)K * d));
    NS_CU(buf.get(&d_m, d)); NS_CU(buf.get(&d_G, (size_t)d * d)); NS_CU(buf.get(&d_s, 1));
    NS_CU(buf.get(&d_theta, (size_t)N * P)); NS_CU(buf.get(&d_theta_c, (size_t)K * P));
    NS_CU(buf.get(&d_logl, N)); NS_CU(buf.get(&d_logl_c, K)); NS_CU(buf.get(&d_state, 1)); NS_CU(buf.get(&d_death, K)); NS_CU(buf.get(&d_death_l, K));
    NS_CU(cudaMemcpyAsync(d_lo, lo.data(), P * sizeof(double), cudaMemcpyHostToDevice, st));
    NS_CU(cudaMemcpyAsync(d_hi, hi.data(), P * sizeof(double), cudaMemcpyHostToDevice, st));
    NS_CU(cudaMemcpyAsync(d_free, free_idx.data(), d * sizeof(int), cudaMemcpyHostToDevice, st));
    NS_CU(cudaMemcpyAsync(d_tied, tied.data(), P * sizeof(int), cudaMemcpyHostToDevice, st));
    NS_CU(cudaStreamSynchronize(st));                       // the host vectors above go out of scope otherwise

    const NsProblem pb{d_lo, d_hi, d_free, d_tied, P, d, N, K, opt->enlarge, log(opt->tol), opt->seed};
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
        // never a round beyond max_rounds: the convergence check every few rounds must not overshoot it
        for (int r = 0; r < check_every && rounds_launched < opt->max_rounds; ++r, ++rounds_launched) {
            ns_bound_kernel<<<1, 256, 0, st>>>(pb, d_U, d_m, d_G, d_s, d_state);
            ns_propose_kernel<<<(K + 127) / 128, 128, 0, st>>>(pb, d_m, d_G, d_s, d_Uc, d_theta_c, d_state);
            NS_CU(cudaGetLastError());
            if (n_image_plane > 0)
                NS_OK(lensed_image_plane_prior(h, d_theta_c, K, image_plane_sources, n_image_plane, stream));
            NS_OK(lensed_loglike(h, d_theta_c, K, d_logl_c, stream));
            ns_update_kernel<<<1, 256, 0, st>>>(pb, d_U, d_theta, d_logl, d_Uc, d_theta_c, d_logl_c, d_death, d_death_l, out, d_state);
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
    // rounds the sampler used: batches launched after convergence within a group of check_every are
    // discarded by the ns_* kernels and not counted
    res->n_likelihood = (long long)N + n_rounds * K;
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
