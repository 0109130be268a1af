// api.cu -- the C ABI of include/lensed.h and include/lensed_tune.h: handle, argument checks, create-time tables
// (traced-pixel list, active tiles, flipped PSF, padded rule), batch chunking and launches.
// Host logic only; every step of the path runs in prep.cu / trace.cu / conv.cu.
#include "../../include/lensed.h"
#include "../../include/lensed_tune.h"
#include "lensed_internal.h"
#include "jit.h"

#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <atomic>
#include <mutex>
#include <utility>
#include <new>
#include <string>
#include <vector>

using namespace lensed;

namespace {

thread_local std::string g_last_error;

enum { PH_PREP = 0, PH_TRACE = 1, PH_REFINE = 2, PH_CONV = 3, PH_FINAL = 4, PH_COUNT = 5 };

struct EventPair { cudaEvent_t a, b; int phase; };

}  // namespace

// Reference count of what lensed_clone shares between handles: the large immutable device
// arrays of a problem (d_image, d_wmask, d_pix_ll, d_pix_all, the tap range / d_gtaps).
struct SharedArrays {
    std::atomic<int> refs{1};
};

struct lensed_handle {
    SharedArrays *shared = nullptr;
    int device = 0;
    int H = 0, W = 0;
    double scale = 0, zp = 0;
    Program prog{};
    int n_quad = 0, R = 1, nq_pad = 0;
    int np_pp = 2, nq_pp = 0;       // the rule in passes for the pixel-pair tracers (trace_static.cuh)
    std::vector<float4> h_quad_pp;
    std::vector<float4> h_quad;     // host copy of d_quad (lensed_set_error_rule rewrites .w)
    bool has_error_rule = false;
    int KH = 1, KW = 1, NC = 1;
    int tile_w = 0, tile_h = 0;
    int Hp = 0, Wp = 0;             // padded frame of the unconvolved images (conv.cu "Input")
    int ox_ll = 0, oy_ll = 0;       // origin of the loglike tile grid (render tiles start at 0, 0)
    int n_sm = 1;
    int tap_off = -1, tap_pairs = 0; // this handle's range of the constant tap pool
    unsigned long long *d_gtaps = nullptr;   // the taps in global memory instead, when the pool was full
    int shape = 1;                  // convolution shape: 0 narrow, 1 wide, 2 strip, 3 half-width strip (conv.cu)
    std::vector<uint8_t> counted;   // host copy of the counted-pixel map (lensed_set_conv_shape rebuilds the tiles)

    // device, immutable after create
    float *d_image = nullptr, *d_wmask = nullptr;
    float4 *d_quad = nullptr, *d_quad_pp = nullptr;
    uint32_t *d_pix_ll = nullptr, *d_pix_all = nullptr, *d_tiles_ll = nullptr, *d_tiles_all = nullptr;
    int npix_ll = 0, npix_all = 0, ntiles_ll = 0, ntiles_all = 0;

    // device scratch, grown on demand
    float *d_derived = nullptr; size_t cap_derived = 0;
    double *d_derived64 = nullptr; size_t cap_derived64 = 0;
    uint32_t *d_fixmask = nullptr; size_t cap_fixmask = 0;
    int *d_order = nullptr; size_t cap_order = 0;          // tracer block order (prep.cu order_kernel)
    uint2 *d_queue = nullptr; size_t cap_queue = 0;      // refine.cu: flagged pixels of one chunk
    unsigned *d_queue_count = nullptr;
    unsigned long long *d_refined = nullptr;   // pixels refined in FP64 since the last profile reset
    double refine_gain = 1.0;                  // lensed_set_refine
    double fgx_tau = 0.15;                     // lensed_set_fg_expansion (0 = off)
    bool rule_symmetric = true;                // odd moments of the rule vanish: the expansion may be used
    double rule_radius = 0.0;                  // farthest rule point from the pixel centre, pixels
    float *d_L = nullptr; size_t cap_L = 0;
    alignas(64) unsigned char tmap_L[128] = {};    // CUtensorMap of d_L for the convolution's tile loads (conv.cu)
    double *d_partial = nullptr; size_t cap_partial = 0;
    float *d_stage_in = nullptr; size_t cap_stage_in = 0;
    float *d_stage_out = nullptr; size_t cap_stage_out = 0;
    long long chunk_bytes = 1ll << 30;
    bool static_tracer = false;     // the model list has a specialised tracer (built in, or compiled at create: jit) and may use it
    const JitTracer *jit = nullptr; // the run-time compiled one (jit.cu), when the list has no built-in signature

    // instrumentation
    bool profiling = false;
    std::vector<EventPair> used;
    std::vector<EventPair> pool;
    double ms[PH_COUNT] = {0, 0, 0, 0, 0};
    long long launches[PH_COUNT] = {0, 0, 0, 0, 0};

    std::string err;
};

namespace {

// Constant tap pool (conv.cu c_taps): first-fit ranges per device, in tap pairs.
struct TapPool {
    std::mutex mu;
    std::vector<std::pair<int, int>> used[64];      // (offset, length), sorted by offset
    int take(int device, int n)
    {
        std::lock_guard<std::mutex> g(mu);
        auto &u = used[device & 63];
        int off = 0;
        size_t at = 0;
        for (; at < u.size(); ++at) {
            if (u[at].first - off >= n) break;
            off = u[at].first + u[at].second;
        }
        if (off + n > kTapPoolPairs) return -1;
        u.insert(u.begin() + at, std::make_pair(off, n));
        return off;
    }
    void give(int device, int off)
    {
        std::lock_guard<std::mutex> g(mu);
        auto &u = used[device & 63];
        for (size_t i = 0; i < u.size(); ++i)
            if (u[i].first == off) { u.erase(u.begin() + i); return; }
    }
} g_tap_pool;

lensed_status fail(lensed_handle *h, lensed_status st, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (h) h->err = buf;
    g_last_error = buf;
    return st;
}

#define CU(h, call)                                                                           \
    do {                                                                                      \
        cudaError_t e_ = (call);                                                              \
        if (e_ != cudaSuccess)                                                                \
            return fail(h, e_ == cudaErrorMemoryAllocation ? LENSED_ENOMEM : LENSED_ECUDA,    \
                        "%s: %s", #call, cudaGetErrorString(e_));                             \
    } while (0)

template <class T>
lensed_status upload(lensed_handle *h, T **dst, const T *src, size_t n)
{
    CU(h, cudaMalloc((void **)dst, std::max<size_t>(n, 1) * sizeof(T)));
    if (n) CU(h, cudaMemcpy(*dst, src, n * sizeof(T), cudaMemcpyHostToDevice));
    return LENSED_OK;
}

// Scratch grows to the high-water mark of the calls made so far, with stream-ordered
// allocation on the caller's stream: no device-wide synchronisation inside an asynchronous
// call (cudaFree / cudaMalloc would be one), and none at all once a batch size has been seen.
template <class T>
lensed_status grow(lensed_handle *h, T **buf, size_t *cap, size_t need, cudaStream_t st)
{
    if (need <= *cap) return LENSED_OK;
    if (*buf) { CU(h, cudaFreeAsync(*buf, st)); *buf = nullptr; *cap = 0; }
    CU(h, cudaMallocAsync((void **)buf, need * sizeof(T), st));
    *cap = need;
    return LENSED_OK;
}

// Pixels read by the PSF windows of the counted pixels, with border clamping (R8): a
// counted pixel (i, j) reads rows clamp(i+k), |k| <= p, and columns clamp(j+l), |l| <= q.
std::vector<uint8_t> dilate(const std::vector<uint8_t> &cnt, int H, int W, int p, int q)
{
    std::vector<uint8_t> rows((size_t)H * W, 0), out((size_t)H * W, 0);
    for (int i = 0; i < H; ++i)
        for (int k = -p; k <= p; ++k) {
            const int ii = std::min(std::max(i + k, 0), H - 1);
            for (int j = 0; j < W; ++j) rows[(size_t)ii * W + j] |= cnt[(size_t)i * W + j];
        }
    for (int i = 0; i < H; ++i)
        for (int j = 0; j < W; ++j) {
            if (!rows[(size_t)i * W + j]) continue;
            for (int l = -q; l <= q; ++l) out[(size_t)i * W + std::min(std::max(j + l, 0), W - 1)] = 1;
        }
    return out;
}

void pixel_list(const std::vector<uint8_t> &sel, int H, int W, std::vector<uint32_t> &out)
{
    out.clear();
    for (int i = 0; i < H; ++i)
        for (int j = 0; j < W; ++j)
            if (sel[(size_t)i * W + j]) out.push_back(((uint32_t)i << 16) | (uint32_t)j);
}

// Tiles of tw x th pixels with origin (ox, oy) that hold a selected pixel, packed
// (tile row << 16) | tile column; *ny, *nx = extent of the grid in tiles.
void tile_list(const std::vector<uint8_t> &cnt, int H, int W, int tw, int th, int ox, int oy,
               std::vector<uint32_t> &out, int *ny, int *nx)
{
    out.clear();
    *ny = *nx = 0;
    for (int ti = 0; oy + ti * th < H; ++ti)
        for (int tj = 0; ox + tj * tw < W; ++tj) {
            bool any = false;
            for (int i = oy + ti * th; i < std::min(H, oy + (ti + 1) * th) && !any; ++i)
                for (int j = ox + tj * tw; j < std::min(W, ox + (tj + 1) * tw); ++j)
                    if (cnt[(size_t)i * W + j]) { any = true; break; }
            if (any) {
                out.push_back(((uint32_t)ti << 16) | (uint32_t)tj);
                *ny = std::max(*ny, ti + 1); *nx = std::max(*nx, tj + 1);
            }
        }
}

// Strips of the strip shape (conv.cu): sw x sh pixels, packed (first row << 16) | first column in
// PIXEL coordinates.  Every band of sh rows (from the first selected row on) is covered on its own:
// strips start at the band's first selected column (rounded down to a multiple of 4) and skip
// stretches without a selected pixel, so a round mask is hugged band by band (SLACS annulus: 23
// strips against 25 on one grid).  *rows, *cols = extent the strips reach.
void strip_list(const std::vector<uint8_t> &sel, int H, int W, int sw, int sh, std::vector<uint32_t> &out, int *rows, int *cols)
{
    out.clear();
    *rows = *cols = 0;
    int y0 = H;
    for (int i = 0; i < H && y0 == H; ++i)
        for (int j = 0; j < W; ++j)
            if (sel[(size_t)i * W + j]) { y0 = i; break; }
    for (int y = y0; y < H; y += sh) {
        std::vector<uint8_t> col(W, 0);
        for (int i = y; i < std::min(H, y + sh); ++i)
            for (int j = 0; j < W; ++j) col[j] |= sel[(size_t)i * W + j];
        int x = 0;
        while (x < W) {
            while (x < W && !col[x]) ++x;
            if (x >= W) break;
            x = x / 4 * 4;
            out.push_back(((uint32_t)y << 16) | (uint32_t)x);
            *rows = std::max(*rows, y + sh); *cols = std::max(*cols, x + sw);
            x += sw;
        }
    }
}

lensed_status timed_begin(lensed_handle *h, int phase, cudaStream_t st)
{
    h->launches[phase] += 1;
    if (!h->profiling) return LENSED_OK;
    EventPair ep;
    if (!h->pool.empty()) { ep = h->pool.back(); h->pool.pop_back(); }
    else { CU(h, cudaEventCreate(&ep.a)); CU(h, cudaEventCreate(&ep.b)); }
    ep.phase = phase;
    CU(h, cudaEventRecord(ep.a, st));
    h->used.push_back(ep);
    return LENSED_OK;
}

lensed_status timed_end(lensed_handle *h, cudaStream_t st)
{
    if (!h->profiling) return LENSED_OK;
    CU(h, cudaEventRecord(h->used.back().b, st));
    return LENSED_OK;
}

lensed_status collect_profile(lensed_handle *h)
{
    for (EventPair &ep : h->used) {
        CU(h, cudaEventSynchronize(ep.b));
        float ms = 0.f;
        CU(h, cudaEventElapsedTime(&ms, ep.a, ep.b));
        h->ms[ep.phase] += ms;
        h->pool.push_back(ep);
    }
    h->used.clear();
    return LENSED_OK;
}

bool g_force_global_taps = false;     // lensed_debug_force_global_taps (tests)

// Tile lists and padded frame for one block shape of the convolution; frees the frame buffer
// (its layout changes).  Loglike tiles start at the corner of the counted pixels' bounding box
// (x rounded down to a 16-byte boundary for cp.async): a mask that is not tile-aligned costs
// fewer tiles.  The render grid starts at (0, 0).
lensed_status build_tiles(lensed_handle *h, int shape)
{
    const int H = h->H, W = h->W;
    h->shape = shape;
    conv_tile_shape(shape, &h->tile_w, &h->tile_h);
    std::vector<uint8_t> all((size_t)H * W, 1);
    std::vector<uint32_t> tiles_ll, tiles_all;
    int x0 = W, y0 = H;
    for (int i = 0; i < H; ++i)
        for (int j = 0; j < W; ++j)
            if (h->counted[(size_t)i * W + j]) { x0 = std::min(x0, j); y0 = std::min(y0, i); }
    h->ox_ll = x0 < W ? x0 / 4 * 4 : 0;
    h->oy_ll = y0 < H ? y0 : 0;
    int rows, cols;
    if (shape >= 2) {
        // strips carry their own pixel coordinates (strip_list): no grid origin
        int r1, c1, r2, c2;
        h->ox_ll = h->oy_ll = 0;
        strip_list(h->counted, H, W, h->tile_w, h->tile_h, tiles_ll, &r1, &c1);
        strip_list(all, H, W, h->tile_w, h->tile_h, tiles_all, &r2, &c2);
        rows = std::max(std::max(r1, r2), H);
        cols = std::max(std::max(c1, c2), W);
    } else {
        int ny_ll, nx_ll, ny_all, nx_all;
        tile_list(h->counted, H, W, h->tile_w, h->tile_h, h->ox_ll, h->oy_ll, tiles_ll, &ny_ll, &nx_ll);
        tile_list(all, H, W, h->tile_w, h->tile_h, 0, 0, tiles_all, &ny_all, &nx_all);
        // padded frame: the image, and every tile of either grid with its PSF halo
        rows = std::max(std::max(ny_all * h->tile_h, h->oy_ll + ny_ll * h->tile_h), H);
        cols = std::max(std::max(nx_all * h->tile_w, h->ox_ll + nx_ll * h->tile_w), W);
    }
    conv_padded_shape(rows, cols, h->KH, h->NC, &h->Hp, &h->Wp);
    h->ntiles_ll = (int)tiles_ll.size(); h->ntiles_all = (int)tiles_all.size();
    CU(h, cudaSetDevice(h->device));
    CU(h, cudaDeviceSynchronize());
    cudaFree(h->d_tiles_ll); cudaFree(h->d_tiles_all); cudaFree(h->d_L);
    h->d_tiles_ll = h->d_tiles_all = nullptr; h->d_L = nullptr; h->cap_L = 0;
    lensed_status s;
    if ((s = upload(h, &h->d_tiles_ll, tiles_ll.data(), tiles_ll.size())) != LENSED_OK) return s;
    return upload(h, &h->d_tiles_all, tiles_all.data(), tiles_all.size());
}

// Shape lensed_create picks, from the pixels each shape's tile list computes (tiles x tile area)
// and what was measured on the configs (profiles/r2b.md).  Large PSFs on full tiles: wide (31 x 31
// PSF, 4096 Euclid vectors: wide 32.4, narrow 34.7, strip 34.6 ms -- the strip shape has one stage
// per warp there and its unsynchronised warps miss the constant cache on the taps more often than
// a block's lock-step warps).  Masked images: the shape that computes at least 15 % fewer pixels
// (SLACS annulus: 23 strips = 23.6 k pixels against 8 narrow tiles = 32.8 k; 1.49 against 2.10 ms).
int default_shape(const lensed_handle *h)
{
#ifdef LENSED_CONV_FORCE_SHAPE
    return LENSED_CONV_FORCE_SHAPE;
#endif
    long long px[4];
    for (int shape = 0; shape < 4; ++shape) {
        int tw, th, ny, nx, x0 = h->W, y0 = h->H;
        conv_tile_shape(shape, &tw, &th);
        for (int i = 0; i < h->H; ++i)
            for (int j = 0; j < h->W; ++j)
                if (h->counted[(size_t)i * h->W + j]) { x0 = std::min(x0, j); y0 = std::min(y0, i); }
        std::vector<uint32_t> tiles;
        if (shape >= 2) strip_list(h->counted, h->H, h->W, tw, th, tiles, &ny, &nx);
        else tile_list(h->counted, h->H, h->W, tw, th, x0 < h->W ? x0 / 4 * 4 : 0, y0 < h->H ? y0 : 0, tiles, &ny, &nx);
        px[shape] = conv_shape_fits(h->KH, h->NC, shape) ? (long long)tiles.size() * tw * th : (1LL << 60);
    }
    const int block = px[0] * 100 <= px[1] * 85 ? 0 : 1;
    const int strip = conv_shape_fits(h->KH, h->NC, 3) ? 3 : 2;      // half-width strips wherever their two-vector stage fits
    if (!conv_shape_fits(h->KH, h->NC, strip)) return block;
    // strips: with PSFs up to 23 x 23 (where full strips are double buffered) they are as fast as the
    // wide tiles on full images and faster on small ones (HST 0.067 against 0.076 ms); with larger PSFs
    // only where they compute at least 15 % fewer pixels.  Half-width strips beat full ones on every
    // config (two vectors per tensor copy; SLACS annulus 39 x 512 = 20.0 k pixels against 23 x 1024 =
    // 23.6 k: 1.27 against 1.49 ms; Euclid 33.9 against 34.6; profiles/r2b.md).
    return conv_num_stages(h->KH, h->NC, false, 2) == 2 || px[strip] * 100 <= px[block] * 85 ? strip : block;
}

// Pixels of the traced list one tracer block walks: it amortises its prologue (constants, frame
// tables, rule moments, four barriers) over them, so few large blocks of EQUAL size -- the list is
// split into ceil(npix / kPpbMax) blocks and the block size rounded up to whole passes of 256
// threads.  Round 2, pixel-pair tracers, ms per step at fixed 1024 / 2048 / 4096 / 5120 / 8192:
// HST (10 000 pixels) 0.241 / 0.221 / 0.224 / 0.213 / 0.245 (5120 = two equal blocks), mock (14 400)
// 4.72 / 4.53 / 4.43 / 4.40 / 4.43, SLACS (21 160) 3.75 / - / 3.48 / 3.47 / 3.44.  At most 8192
// (32 flag bits per thread, TraceArgs::fixmask).
#ifndef LENSED_PPB_MAX
#define LENSED_PPB_MAX 8192
#endif
int pix_per_block(int npix)
{
#ifdef LENSED_PIX_PER_BLOCK             // tuning builds (build.py defines=...)
    return LENSED_PIX_PER_BLOCK;
#else
    if (npix <= 256) return 256;
    const int n_blocks = (npix + LENSED_PPB_MAX - 1) / LENSED_PPB_MAX;
    return ((npix + n_blocks - 1) / n_blocks + 255) / 256 * 256;
#endif
}

// The whole path for B vectors already on the device.
lensed_status run(lensed_handle *h, const float *params_dev, int B, float *out_dev, bool render,
                  cudaStream_t st)
{
    if (!h) return fail(nullptr, LENSED_EINVAL, "null handle");
    if (!params_dev || !out_dev) return fail(h, LENSED_EINVAL, "null device pointer");
    if (B < 1) return fail(h, LENSED_EINVAL, "B = %d < 1", B);
    CU(h, cudaSetDevice(h->device));
    const Program &prog = h->prog;
    const size_t HW = (size_t)h->H * h->W;
    const int n_tiles = render ? h->ntiles_all : h->ntiles_ll;
    const int npix = render ? h->npix_all : h->npix_ll;

    const size_t HWp = (size_t)h->Hp * h->Wp;
    long long per_chunk = std::max<long long>(1, h->chunk_bytes / (long long)(HWp * sizeof(float)));
    const int Bc = (int)std::min<long long>(std::min<long long>(per_chunk, 65535), B);

    lensed_status s;
    if ((s = grow(h, &h->d_derived, &h->cap_derived, (size_t)B * prog.D, st)) != LENSED_OK) return s;
    if ((s = grow(h, &h->d_derived64, &h->cap_derived64, (size_t)B * prog.n_models * kD64PerModel, st)) != LENSED_OK) return s;
    if ((size_t)Bc * HWp > h->cap_L) {
        // pad cells no pixel clamps to (tile overhang) are read, never written: keep them zero
        if ((s = grow(h, &h->d_L, &h->cap_L, (size_t)Bc * HWp, st)) != LENSED_OK) return s;
        CU(h, cudaMemsetAsync(h->d_L, 0, (size_t)Bc * HWp * sizeof(float), st));
        CU(h, conv_make_tensor_map(h->tmap_L, h->d_L, h->Wp, h->Hp, Bc, h->KH, h->NC, h->shape));
    }
    if (!render && (s = grow(h, &h->d_partial, &h->cap_partial, (size_t)B * std::max(n_tiles, 1), st)) != LENSED_OK)
        return s;
    const int ppb = pix_per_block(npix);
    const int n_tblocks = npix > 0 ? (npix + ppb - 1) / ppb : 0;
    const bool refine = h->refine_gain > 0.0 && n_tblocks > 0;
    if (refine && (s = grow(h, &h->d_fixmask, &h->cap_fixmask, (size_t)Bc * n_tblocks * 256, st)) != LENSED_OK) return s;
    const size_t queue_cap = (size_t)Bc * 64 + 4096;
    if (refine && (s = grow(h, &h->d_queue, &h->cap_queue, queue_cap, st)) != LENSED_OK) return s;

    PrepArgs pa{params_dev, h->d_derived, h->d_derived64, B,
                h->refine_gain > 0.0 ? h->refine_gain : (double)INFINITY,
                h->rule_symmetric && h->static_tracer ? h->fgx_tau : 0.0, h->rule_radius,
                h->scale, h->zp, 0.5 * (h->W - 1), 0.5 * (h->H - 1)};
    bool has_sie = false;                     // only the SIE has per-mode code paths worth sorting for
    for (int m = 0; m < prog.n_lens; ++m) has_sie = has_sie || prog.lens_kind[m] == K_SIE;
    const bool sorted = has_sie && npix > 0 && B > 1;
    if (sorted && (s = grow(h, &h->d_order, &h->cap_order, (size_t)B, st)) != LENSED_OK) return s;
    if ((s = timed_begin(h, PH_PREP, st)) != LENSED_OK) return s;
    CU(h, launch_prep(prog, pa, st));
    if (sorted) {
        CU(h, launch_order(h->d_derived, prog.D, B, Bc, h->d_order, st));
        h->launches[PH_PREP] += 1;                           // two kernels in this phase: prep, order
    }
    if ((s = timed_end(h, st)) != LENSED_OK) return s;

    for (int b0 = 0; b0 < B; b0 += Bc) {
        const int nb = std::min(Bc, B - b0);
        if (npix > 0) {
            TraceArgs ta{};
            ta.order = sorted ? h->d_order + b0 : nullptr;
            ta.derived = h->d_derived + (size_t)b0 * prog.D;
            ta.pix = render ? h->d_pix_all : h->d_pix_ll;
            ta.quad = h->d_quad;
            ta.quad_pp = h->d_quad_pp; ta.nq_pp = h->nq_pp; ta.np_pp = h->np_pp;
            ta.fixmask = refine ? h->d_fixmask : nullptr;
            ta.L = h->d_L;
            ta.l_stride = (long long)HWp;
            ta.npix = npix; ta.nq_pad = h->nq_pad;
            ta.H = h->H; ta.W = h->W; ta.Wp = h->Wp; ta.px = (h->KW - 1) / 2; ta.py = (h->KH - 1) / 2;
            ta.pix_per_block = ppb;
            ta.cxh = 0.5f * (h->W - 1); ta.cyh = 0.5f * (h->H - 1);
            if ((s = timed_begin(h, PH_TRACE, st)) != LENSED_OK) return s;
            CU(h, launch_trace(prog, ta, h->R, nb, h->static_tracer, h->jit, st));
            if ((s = timed_end(h, st)) != LENSED_OK) return s;
            if (refine) {
                // FP64 re-trace of the pixels the tracer flagged (refine.cu), before the convolution
                RefineArgs ra{ta, h->d_derived64 + (size_t)b0 * prog.n_models * kD64PerModel, ta.derived, h->d_refined,
                              h->d_queue, h->d_queue_count, (int)queue_cap, nb, n_tblocks, h->n_quad};
                if ((s = timed_begin(h, PH_REFINE, st)) != LENSED_OK) return s;
                CU(h, launch_refine(prog, ra, h->n_sm, st));
                h->launches[PH_REFINE] += 1;                       // two kernels: scan, queue
                if ((s = timed_end(h, st)) != LENSED_OK) return s;
            }
        }
        if (n_tiles > 0) {
            ConvArgs ca{};
            ca.Lp = h->d_L;
            ca.image = h->d_image;
            ca.wmask = h->d_wmask;
            ca.tiles = render ? h->d_tiles_all : h->d_tiles_ll;
            ca.partial = render ? nullptr : h->d_partial + (size_t)b0 * n_tiles;
            ca.model = render ? out_dev + (size_t)b0 * HW : nullptr;
            ca.derived = h->d_derived + (size_t)b0 * prog.D;
            ca.lp_stride = (long long)HWp;
            ca.D = prog.D;
            ca.H = h->H; ca.W = h->W; ca.Wp = h->Wp; ca.KH = h->KH; ca.KW = h->KW; ca.NC = h->NC;
            ca.n_tiles = n_tiles; ca.nb = nb;
            ca.tap_off = h->d_gtaps ? 0 : h->tap_off; ca.gtaps = h->d_gtaps; ca.shape = h->shape;
            ca.ox = render ? 0 : h->ox_ll; ca.oy = render ? 0 : h->oy_ll;
            if ((s = timed_begin(h, PH_CONV, st)) != LENSED_OK) return s;
            CU(h, launch_conv(ca, h->tmap_L, render, h->n_sm, st));
            if ((s = timed_end(h, st)) != LENSED_OK) return s;
        }
    }
    if (!render) {
        FinalArgs fa{h->d_partial, h->d_derived, out_dev, B, n_tiles, prog.D};
        if ((s = timed_begin(h, PH_FINAL, st)) != LENSED_OK) return s;
        CU(h, launch_final(fa, st));
        if ((s = timed_end(h, st)) != LENSED_OK) return s;
    }
    return LENSED_OK;
}

lensed_status run_host(lensed_handle *h, const float *params_host, int B, float *out_host, bool render,
                       cudaStream_t st)
{
    if (!h) return fail(nullptr, LENSED_EINVAL, "null handle");
    if (!params_host || !out_host) return fail(h, LENSED_EINVAL, "null host pointer");
    if (B < 1) return fail(h, LENSED_EINVAL, "B = %d < 1", B);
    CU(h, cudaSetDevice(h->device));
    const size_t n_in = (size_t)B * h->prog.P;
    const size_t n_out = render ? (size_t)B * h->H * h->W : (size_t)B;
    lensed_status s;
    if ((s = grow(h, &h->d_stage_in, &h->cap_stage_in, n_in, st)) != LENSED_OK) return s;
    if ((s = grow(h, &h->d_stage_out, &h->cap_stage_out, n_out, st)) != LENSED_OK) return s;
    CU(h, cudaMemcpyAsync(h->d_stage_in, params_host, n_in * sizeof(float), cudaMemcpyHostToDevice, st));
    if ((s = run(h, h->d_stage_in, B, h->d_stage_out, render, st)) != LENSED_OK) return s;
    CU(h, cudaMemcpyAsync(out_host, h->d_stage_out, n_out * sizeof(float), cudaMemcpyDeviceToHost, st));
    CU(h, cudaStreamSynchronize(st));
    return LENSED_OK;
}

}  // namespace

namespace lensed {
int handle_fail(::lensed_handle *h, int status, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    return fail(h, (lensed_status)status, "%s", buf);
}
int handle_device(const ::lensed_handle *h) { return h->device; }
}  // namespace lensed

extern "C" {

lensed_status lensed_create(int H, int W, double pixel_scale, const float *image, const float *weight,
                            const unsigned char *mask, const float *psf, int psf_h, int psf_w,
                            const float *quad, int n_quad, const int *models, int n_models,
                            double mag_zero_point, int device, lensed_handle **out)
{
    if (!out) return fail(nullptr, LENSED_EINVAL, "out is NULL");
    *out = nullptr;
    if (H < 1 || W < 1) return fail(nullptr, LENSED_EINVAL, "image size %d x %d", H, W);
    if (H > 32767 || W > 32767) return fail(nullptr, LENSED_EUNSUPPORTED, "image side > 32767");
    if (!(pixel_scale > 0.0) || !isfinite(pixel_scale)) return fail(nullptr, LENSED_EINVAL, "pixel_scale must be > 0");
    if (!isfinite(mag_zero_point)) return fail(nullptr, LENSED_EINVAL, "mag_zero_point not finite");
    if (!image || !weight) return fail(nullptr, LENSED_EINVAL, "image / weight is NULL");
    if (!quad || n_quad < 1) return fail(nullptr, LENSED_EINVAL, "quadrature rule missing (n_quad = %d)", n_quad);
    if (n_quad > LENSED_MAX_QUAD) return fail(nullptr, LENSED_EUNSUPPORTED, "n_quad %d > %d", n_quad, LENSED_MAX_QUAD);
    if (!models || n_models < 1) return fail(nullptr, LENSED_EINVAL, "model list missing");
    if (n_models > LENSED_MAX_MODELS) return fail(nullptr, LENSED_EUNSUPPORTED, "n_models %d > %d", n_models, LENSED_MAX_MODELS);
    const bool has_psf = psf && !(psf_h == 1 && psf_w == 1);
    if (psf) {
        if (psf_h < 1 || psf_w < 1 || psf_h % 2 == 0 || psf_w % 2 == 0)
            return fail(nullptr, LENSED_EINVAL, "PSF dims %d x %d must be odd (R11)", psf_h, psf_w);
        if (psf_h > LENSED_MAX_PSF || psf_w > LENSED_MAX_PSF)
            return fail(nullptr, LENSED_EUNSUPPORTED, "PSF side > %d", LENSED_MAX_PSF);
    }

    const size_t HW = (size_t)H * W;
    std::vector<uint8_t> counted(HW), all(HW, 1);
    std::vector<float> wmask(HW);
    for (size_t i = 0; i < HW; ++i) {
        const float w = weight[i];
        if (!(w >= 0.0f) || !isfinite(w)) return fail(nullptr, LENSED_EINVAL, "weight[%zu] negative or not finite", i);
        const bool on = (!mask || mask[i]) && w > 0.0f;
        if (on && !isfinite(image[i])) return fail(nullptr, LENSED_EINVAL, "image[%zu] not finite", i);
        wmask[i] = on ? w : 0.0f;
        counted[i] = on;
    }

    lensed_handle *h = new (std::nothrow) lensed_handle;
    if (!h) return fail(nullptr, LENSED_ENOMEM, "host allocation failed");
    h->shared = new (std::nothrow) SharedArrays;
    if (!h->shared) { delete h->shared; delete h; return fail(nullptr, LENSED_ENOMEM, "host allocation failed"); }
    lensed_status s = LENSED_OK;
#define CREATE_FAIL(expr)                                             \
    do { s = (expr); if (s != LENSED_OK) { g_last_error = h->err.empty() ? g_last_error : h->err; lensed_destroy(h); return s; } } while (0)

    h->device = device; h->H = H; h->W = W; h->scale = pixel_scale; h->zp = mag_zero_point;

    // model list -> program
    Program &pg = h->prog;
    pg.n_models = n_models;
    int P = 0;
    for (int m = 0; m < n_models; ++m) {
        const int k = models[m];
        if (k < 0 || k >= K_COUNT) { delete h->shared; delete h; return fail(nullptr, LENSED_EINVAL, "models[%d] = %d is not a lensed_kind", m, k); }
        pg.kind[m] = (uint8_t)k;
        pg.par_off[m] = (uint16_t)P;
        P += kind_num_params(k);
    }
    // canonical order (stable within a kind): lenses shear, SIE, SIS, point mass -- the first
    // shear initialises alpha in the tracer; lights source Sersic, source Gaussian, foreground
    // Sersic, foreground Gaussian, sky.  The sums over lenses and over lights do not depend on
    // the order beyond rounding.  The derived vector is laid out in that order too (header,
    // lenses, lights), so a static tracer signature fixes every block's offset at compile time
    // (trace_static.cuh TraceSig::lens_off4 / light_off4).
    int D = kHeaderFloats;
    {
        static const int lens_order[] = {K_SHEAR, K_SIE, K_SIS, K_POINT};
        static const int light_order[] = {K_SRC_SERSIC, K_SRC_GAUSS, K_FG_SERSIC, K_FG_GAUSS, K_SKY};
        for (int kind : lens_order)
            for (int m = 0; m < n_models; ++m)
                if (pg.kind[m] == kind) {
                    pg.der_off[m] = (uint16_t)D;
                    pg.lens_kind[pg.n_lens] = (uint8_t)kind; pg.lens_off[pg.n_lens++] = (uint16_t)D;
                    D += kind_num_derived(kind);
                }
        for (int kind : light_order)
            for (int m = 0; m < n_models; ++m)
                if (pg.kind[m] == kind) {
                    pg.der_off[m] = (uint16_t)D;
                    pg.light_kind[pg.n_light] = (uint8_t)kind; pg.light_off[pg.n_light++] = (uint16_t)D;
                    D += kind_num_derived(kind);
                }
    }
    pg.P = P; pg.D = D;
    h->static_tracer = trace_has_static(pg);

    // rule: weights to unit sum in double, padded with zero-weight points to a multiple of R
    double wsum = 0.0;
    for (int k = 0; k < n_quad; ++k) {
        for (int c = 0; c < 3; ++c)
            if (!isfinite(quad[3 * k + c])) { delete h->shared; delete h; return fail(nullptr, LENSED_EINVAL, "quad[%d] not finite", k); }
        wsum += (double)quad[3 * k + 2];
    }
    if (!(fabs(wsum) > 0.0)) { delete h->shared; delete h; return fail(nullptr, LENSED_EINVAL, "quadrature weights sum to zero"); }
    h->n_quad = n_quad;
    h->R = trace_pick_R(n_quad);
    h->nq_pad = (n_quad + h->R - 1) / h->R * h->R;
    std::vector<float4> hq(h->nq_pad, make_float4(0.f, 0.f, 0.f, 0.f));
    for (int k = 0; k < n_quad; ++k)
        hq[k] = make_float4(quad[3 * k], quad[3 * k + 1], (float)((double)quad[3 * k + 2] / wsum), 0.f);
    // the same rule in passes of np_pp points, every pass a 16-byte-aligned stretch of 4 or 8 table
    // entries (the rest zero-weight and never evaluated): layout of the pixel-pair tracers
    h->np_pp = trace_pick_np(n_quad);
    {
        const int npp = h->np_pp <= 4 ? 4 : 8, n_pass = (n_quad + h->np_pp - 1) / h->np_pp;
        h->nq_pp = n_pass * npp;
        h->h_quad_pp.assign(h->nq_pp, make_float4(0.f, 0.f, 0.f, 0.f));
        for (int k = 0; k < n_quad; ++k) h->h_quad_pp[(k / h->np_pp) * npp + k % h->np_pp] = hq[k];
    }
    {
        // first and third moments of the rule: the foreground expansion (trace_static.cuh) drops
        // them, so it is used only when they vanish (every Cartesian-product rule of the paper does)
        double m1[2] = {0, 0}, m3[4] = {0, 0, 0, 0}, rad = 0.0;
        for (int k = 0; k < n_quad; ++k) {
            const double x = quad[3 * k], y = quad[3 * k + 1], w = (double)quad[3 * k + 2] / wsum;
            m1[0] += w * x; m1[1] += w * y;
            m3[0] += w * x * x * x; m3[1] += w * x * x * y; m3[2] += w * x * y * y; m3[3] += w * y * y * y;
            rad = std::max(rad, sqrt(x * x + y * y));
        }
        h->rule_radius = rad;
        h->rule_symmetric = fabs(m1[0]) < 1e-7 && fabs(m1[1]) < 1e-7 && fabs(m3[0]) < 1e-8 && fabs(m3[1]) < 1e-8 &&
                            fabs(m3[2]) < 1e-8 && fabs(m3[3]) < 1e-8;
    }

    // PSF: normalise in double, flip (eq. 15 uses F_{-k,-l}) -> G[KH][KW]; the convolution
    // reads tap PAIRS  Q[j][c][k] = (G[j][4c+k], G[j-1][4c+k]),  j = 0..KH, G[-1] = G[KH] = 0,
    // columns zero padded to 4-tap chunks (conv.cu "Pairing")
    h->KH = has_psf ? psf_h : 1;
    h->KW = has_psf ? psf_w : 1;
    h->NC = (h->KW + 3) / 4;
    std::vector<float> G((size_t)h->KH * h->KW, 1.0f);
    if (has_psf) {
        double fsum = 0.0;
        for (int t = 0; t < psf_h * psf_w; ++t) {
            if (!isfinite(psf[t])) { delete h->shared; delete h; return fail(nullptr, LENSED_EINVAL, "psf[%d] not finite", t); }
            fsum += (double)psf[t];
        }
        if (!(fabs(fsum) > 0.0)) { delete h->shared; delete h; return fail(nullptr, LENSED_EINVAL, "PSF sums to zero"); }
        for (int ky = 0; ky < psf_h; ++ky)
            for (int kx = 0; kx < psf_w; ++kx)
                G[(size_t)ky * psf_w + kx] =
                    (float)((double)psf[(size_t)(psf_h - 1 - ky) * psf_w + (psf_w - 1 - kx)] / fsum);
    }
    std::vector<float> taps((size_t)(h->KH + 1) * h->NC * 8, 0.0f);
    for (int j = 0; j <= h->KH; ++j)
        for (int kx = 0; kx < h->KW; ++kx) {
            float *pair = &taps[((size_t)j * h->NC + kx / 4) * 8 + 2 * (kx % 4)];
            if (j < h->KH) pair[0] = G[(size_t)j * h->KW + kx];
            if (j > 0) pair[1] = G[(size_t)(j - 1) * h->KW + kx];
        }

    // pixel lists; the tile lists and the padded frame follow the convolution's block shape
    std::vector<uint32_t> pix_ll, pix_all;
    // traced set: the PSF windows of the counted pixels, one more row each way because a
    // counted row's pair partner multiplies its first / last window row by a zero tap
    pixel_list(dilate(counted, H, W, (h->KH - 1) / 2 + 1, (h->KW - 1) / 2), H, W, pix_ll);
    pixel_list(all, H, W, pix_all);
    h->counted = counted;
    h->npix_ll = (int)pix_ll.size(); h->npix_all = (int)pix_all.size();

    int ndev = 0;
    cudaError_t ce = cudaGetDeviceCount(&ndev);
    if (ce != cudaSuccess || ndev < 1) {
        delete h->shared; delete h;
        return fail(nullptr, LENSED_ECUDA, "no CUDA device (%s); there is no CPU fallback",
                    ce != cudaSuccess ? cudaGetErrorString(ce) : "device count 0");
    }
    if (device < 0 || device >= ndev) { delete h->shared; delete h; return fail(nullptr, LENSED_EINVAL, "device %d of %d", device, ndev); }
    {
        cudaError_t e1 = cudaSetDevice(device);
        if (e1 != cudaSuccess) { delete h->shared; delete h; return fail(nullptr, LENSED_ECUDA, "cudaSetDevice: %s", cudaGetErrorString(e1)); }
        cudaDeviceProp prop;
        e1 = cudaGetDeviceProperties(&prop, device);
        if (e1 != cudaSuccess) { delete h->shared; delete h; return fail(nullptr, LENSED_ECUDA, "cudaGetDeviceProperties: %s", cudaGetErrorString(e1)); }
        if (prop.major != 10) {
            delete h->shared; delete h;
            return fail(nullptr, LENSED_ECUDA, "device %d is sm_%d%d; this library holds sm_100a code only",
                        device, prop.major, prop.minor);
        }
        h->n_sm = prop.multiProcessorCount;
        e1 = conv_setup();
        if (e1 != cudaSuccess) { delete h->shared; delete h; return fail(nullptr, LENSED_ECUDA, "conv_setup: %s", cudaGetErrorString(e1)); }
    }
    CREATE_FAIL(upload(h, &h->d_image, image, HW));
    CREATE_FAIL(upload(h, &h->d_wmask, wmask.data(), HW));
    {
        // tap pairs into this handle's range of the constant pool (conv.cu "Taps")
        h->tap_pairs = (int)(taps.size() / 2);
        h->tap_off = g_force_global_taps ? -1 : g_tap_pool.take(device, h->tap_pairs);
        if (h->tap_off < 0) {
            // pool full: this handle's convolution reads its taps from global memory instead
            // (conv.cu GT: same values, LDG through L1 instead of the uniform datapath)
            CREATE_FAIL(upload(h, &h->d_gtaps, reinterpret_cast<const unsigned long long *>(taps.data()), (size_t)h->tap_pairs));
        } else {
            cudaError_t e2 = conv_upload_taps(taps.data(), h->tap_pairs, h->tap_off);
            if (e2 != cudaSuccess) { lensed_destroy(h); return fail(nullptr, LENSED_ECUDA, "tap upload: %s", cudaGetErrorString(e2)); }
        }
    }
    CREATE_FAIL(upload(h, &h->d_quad, hq.data(), hq.size()));
    CREATE_FAIL(upload(h, &h->d_quad_pp, h->h_quad_pp.data(), h->h_quad_pp.size()));
    {
        const unsigned long long zero = 0;
        CREATE_FAIL(upload(h, &h->d_refined, &zero, 1));
        const unsigned zero32 = 0;
        CREATE_FAIL(upload(h, &h->d_queue_count, &zero32, 1));
    }
    h->h_quad = hq;
    CREATE_FAIL(upload(h, &h->d_pix_ll, pix_ll.data(), pix_ll.size()));
    CREATE_FAIL(upload(h, &h->d_pix_all, pix_all.data(), pix_all.size()));
    CREATE_FAIL(build_tiles(h, default_shape(h)));
    if (!h->static_tracer) {
        // no built-in signature for this list: specialise the tracer for it now (jit.cu); on any
        // failure the interpreting tracer runs, as it does with LENSED_JIT=0
        int counts[K_COUNT] = {0};
        for (int m = 0; m < pg.n_models; ++m) counts[pg.kind[m]] += 1;
        if (jit_wanted(counts)) {
            std::string why;
            h->jit = jit_get(counts, h->np_pp, h->device, &why);
            h->static_tracer = h->jit != nullptr;
            if (!h->jit) h->err = "run-time specialisation of the tracer not available (" + why + "): interpreting tracer";
        }
    }
#undef CREATE_FAIL
    *out = h;
    return LENSED_OK;
}

lensed_status lensed_clone(const lensed_handle *src, lensed_handle **out)
{
    if (!out) return fail(nullptr, LENSED_EINVAL, "out is NULL");
    *out = nullptr;
    if (!src) return fail(nullptr, LENSED_EINVAL, "null handle");
    lensed_handle *h = new (std::nothrow) lensed_handle;
    if (!h) return fail(nullptr, LENSED_ENOMEM, "host allocation failed");
    // the problem: geometry, program, rule, PSF layout, options; the big arrays are shared
    h->shared = src->shared;
    h->shared->refs.fetch_add(1);
    h->device = src->device; h->H = src->H; h->W = src->W; h->scale = src->scale; h->zp = src->zp;
    h->prog = src->prog;
    h->n_quad = src->n_quad; h->R = src->R; h->nq_pad = src->nq_pad; h->h_quad = src->h_quad;
    h->np_pp = src->np_pp; h->nq_pp = src->nq_pp; h->h_quad_pp = src->h_quad_pp;
    h->has_error_rule = src->has_error_rule;
    h->KH = src->KH; h->KW = src->KW; h->NC = src->NC; h->n_sm = src->n_sm;
    h->tap_off = src->tap_off; h->tap_pairs = src->tap_pairs; h->d_gtaps = src->d_gtaps;
    h->counted = src->counted;
    h->d_image = src->d_image; h->d_wmask = src->d_wmask; h->d_pix_ll = src->d_pix_ll; h->d_pix_all = src->d_pix_all;
    h->npix_ll = src->npix_ll; h->npix_all = src->npix_all;
    h->chunk_bytes = src->chunk_bytes; h->static_tracer = src->static_tracer; h->jit = src->jit; h->refine_gain = src->refine_gain;
    h->fgx_tau = src->fgx_tau; h->rule_symmetric = src->rule_symmetric; h->rule_radius = src->rule_radius;
    lensed_status s = LENSED_OK;
#define CLONE_FAIL(expr) do { s = (expr); if (s != LENSED_OK) { g_last_error = h->err; lensed_destroy(h); return s; } } while (0)
    if (cudaSetDevice(h->device) != cudaSuccess) { lensed_destroy(h); return fail(nullptr, LENSED_ECUDA, "cudaSetDevice failed"); }
    CLONE_FAIL(upload(h, &h->d_quad, h->h_quad.data(), h->h_quad.size()));
    CLONE_FAIL(upload(h, &h->d_quad_pp, h->h_quad_pp.data(), h->h_quad_pp.size()));
    const unsigned long long zero = 0;
    const unsigned zero32 = 0;
    CLONE_FAIL(upload(h, &h->d_refined, &zero, 1));
    CLONE_FAIL(upload(h, &h->d_queue_count, &zero32, 1));
    CLONE_FAIL(build_tiles(h, src->shape));
#undef CLONE_FAIL
    *out = h;
    return LENSED_OK;
}

int lensed_num_params(const lensed_handle *h) { return h ? h->prog.P : -1; }
int lensed_num_traced(const lensed_handle *h) { return h ? h->npix_ll : -1; }
int lensed_num_pixels(const lensed_handle *h) { return h ? h->H * h->W : -1; }

lensed_status lensed_estimate_weights(long long n, const float *image, const float *gain, double gain0,
                                      const float *offset, double offset0, const float *extra, float *weight)
{
    if (!image || !weight) return fail(nullptr, LENSED_EINVAL, "image / weight is NULL");
    if (n < 1) return fail(nullptr, LENSED_EINVAL, "n = %lld < 1", n);
    for (long long i = 0; i < n; ++i) {
        const double d = image[i], g = gain ? (double)gain[i] : gain0, b = offset ? (double)offset[i] : offset0;
        const double x = extra ? (double)extra[i] : 1.0;
        if (!isfinite(d) || !isfinite(g) || !isfinite(b) || !isfinite(x))
            return fail(nullptr, LENSED_EINVAL, "non-finite input at pixel %lld", i);
        if (!(g > 0.0)) return fail(nullptr, LENSED_EINVAL, "gain %g at pixel %lld is not > 0", g, i);
        if (x < 0.0) return fail(nullptr, LENSED_EINVAL, "extra weight %g at pixel %lld is negative", x, i);
        const double counts_over_g2 = (d + b) / g;           // s_i^2, eq. 21
        weight[i] = counts_over_g2 > 0.0 ? (float)(x / counts_over_g2) : 0.0f;
    }
    return LENSED_OK;
}

lensed_status lensed_set_error_rule(lensed_handle *h, const float *w_embedded)
{
    if (!h) return fail(nullptr, LENSED_EINVAL, "null handle");
    if (!w_embedded) return fail(h, LENSED_EINVAL, "w_embedded is NULL");
    double sum = 0.0;
    for (int k = 0; k < h->n_quad; ++k) {
        if (!isfinite(w_embedded[k])) return fail(h, LENSED_EINVAL, "w_embedded[%d] not finite", k);
        sum += (double)w_embedded[k];
    }
    if (!(fabs(sum) > 0.0)) return fail(h, LENSED_EINVAL, "embedded weights sum to zero");
    CU(h, cudaSetDevice(h->device));
    CU(h, cudaDeviceSynchronize());                // no call of this handle may still read d_quad
    for (int k = 0; k < h->n_quad; ++k)
        h->h_quad[k].w = (float)((double)h->h_quad[k].z - (double)w_embedded[k] / sum);
    CU(h, cudaMemcpy(h->d_quad, h->h_quad.data(), h->h_quad.size() * sizeof(float4), cudaMemcpyHostToDevice));
    h->has_error_rule = true;
    return LENSED_OK;
}

lensed_status lensed_render_error(lensed_handle *h, const float *params_dev, int B, float *err_dev, void *stream)
{
    if (!h) return fail(nullptr, LENSED_EINVAL, "null handle");
    if (!params_dev || !err_dev) return fail(h, LENSED_EINVAL, "null device pointer");
    if (B < 1) return fail(h, LENSED_EINVAL, "B = %d < 1", B);
    if (!h->has_error_rule) return fail(h, LENSED_EINVAL, "no embedded rule: call lensed_set_error_rule first");
    cudaStream_t st = (cudaStream_t)stream;
    CU(h, cudaSetDevice(h->device));
    const Program &prog = h->prog;
    lensed_status s;
    if ((s = grow(h, &h->d_derived, &h->cap_derived, (size_t)B * prog.D, st)) != LENSED_OK) return s;
    if ((s = grow(h, &h->d_derived64, &h->cap_derived64, (size_t)B * prog.n_models * kD64PerModel, st)) != LENSED_OK) return s;
    PrepArgs pa{params_dev, h->d_derived, h->d_derived64, B, (double)INFINITY, 0.0, h->rule_radius, h->scale, h->zp,
                0.5 * (h->W - 1), 0.5 * (h->H - 1)};
    if ((s = timed_begin(h, PH_PREP, st)) != LENSED_OK) return s;
    CU(h, launch_prep(prog, pa, st));
    if ((s = timed_end(h, st)) != LENSED_OK) return s;
    const size_t HW = (size_t)h->H * h->W;
    for (int b0 = 0; b0 < B; b0 += 65535) {
        const int nb = std::min(65535, B - b0);
        TraceArgs ta{};
        ta.derived = h->d_derived + (size_t)b0 * prog.D;
        ta.pix = h->d_pix_all;
        ta.quad = h->d_quad;
        ta.err = err_dev + (size_t)b0 * HW;
        ta.npix = h->npix_all; ta.nq_pad = h->nq_pad;
        ta.H = h->H; ta.W = h->W;
        ta.pix_per_block = ta.npix >= (1 << 11) ? 2048 : 256;
        ta.cxh = 0.5f * (h->W - 1); ta.cyh = 0.5f * (h->H - 1);
        if ((s = timed_begin(h, PH_TRACE, st)) != LENSED_OK) return s;
        CU(h, launch_trace(prog, ta, h->R, nb, false, nullptr, st));
        if ((s = timed_end(h, st)) != LENSED_OK) return s;
    }
    return LENSED_OK;
}

lensed_status lensed_deflect(lensed_handle *h, const float *params_dev, int B, const float *xy_dev, int K,
                             float *out_dev, void *stream)
{
    if (!h) return fail(nullptr, LENSED_EINVAL, "null handle");
    if (!params_dev || !xy_dev || !out_dev) return fail(h, LENSED_EINVAL, "null device pointer");
    if (B < 1 || K < 1) return fail(h, LENSED_EINVAL, "B = %d, K = %d: both must be >= 1", B, K);
    CU(h, cudaSetDevice(h->device));
    CU(h, launch_deflect(h->prog, params_dev, B, xy_dev, K, out_dev, (cudaStream_t)stream));
    return LENSED_OK;
}

lensed_status lensed_image_plane_prior(lensed_handle *h, float *params_dev, int B, const int *source_models,
                                       int n_sources, void *stream)
{
    if (!h) return fail(nullptr, LENSED_EINVAL, "null handle");
    if (!params_dev || !source_models) return fail(h, LENSED_EINVAL, "null pointer");
    if (B < 1) return fail(h, LENSED_EINVAL, "B = %d < 1", B);
    if (n_sources < 1 || n_sources > kMaxModels) return fail(h, LENSED_EINVAL, "n_sources = %d", n_sources);
    int offs[kMaxModels];
    for (int i = 0; i < n_sources; ++i) {
        const int m = source_models[i];
        if (m < 0 || m >= h->prog.n_models)
            return fail(h, LENSED_EINVAL, "source_models[%d] = %d is not an index of the model list", i, m);
        const int k = h->prog.kind[m];
        if (k != K_SRC_SERSIC && k != K_SRC_GAUSS)
            return fail(h, LENSED_EINVAL, "model %d is not a source (LENSED_SRC_*): only sources live in the source plane", m);
        for (int j = 0; j < i; ++j)
            if (source_models[j] == m) return fail(h, LENSED_EINVAL, "model %d listed twice", m);
        offs[i] = h->prog.par_off[m];
    }
    CU(h, cudaSetDevice(h->device));
    CU(h, launch_image_plane_prior(h->prog, offs, n_sources, params_dev, B, (cudaStream_t)stream));
    return LENSED_OK;
}

lensed_status lensed_render(lensed_handle *h, const float *params_dev, int B, float *model_dev, void *stream)
{
    return run(h, params_dev, B, model_dev, true, (cudaStream_t)stream);
}

lensed_status lensed_loglike(lensed_handle *h, const float *params_dev, int B, float *logl_dev, void *stream)
{
    return run(h, params_dev, B, logl_dev, false, (cudaStream_t)stream);
}

lensed_status lensed_render_host(lensed_handle *h, const float *params_host, int B, float *model_host, void *stream)
{
    return run_host(h, params_host, B, model_host, true, (cudaStream_t)stream);
}

lensed_status lensed_loglike_host(lensed_handle *h, const float *params_host, int B, float *logl_host, void *stream)
{
    return run_host(h, params_host, B, logl_host, false, (cudaStream_t)stream);
}

lensed_status lensed_set_profiling(lensed_handle *h, int on)
{
    if (!h) return fail(nullptr, LENSED_EINVAL, "null handle");
    h->profiling = on != 0;
    return LENSED_OK;
}

lensed_status lensed_get_profile(lensed_handle *h, double *ms, long long *launches)
{
    if (!h) return fail(nullptr, LENSED_EINVAL, "null handle");
    lensed_status s = collect_profile(h);
    if (s != LENSED_OK) return s;
    for (int i = 0; i < PH_COUNT; ++i) {
        if (ms) ms[i] = h->ms[i];
        if (launches) launches[i] = h->launches[i];
    }
    return LENSED_OK;
}

lensed_status lensed_reset_profile(lensed_handle *h)
{
    if (!h) return fail(nullptr, LENSED_EINVAL, "null handle");
    lensed_status s = collect_profile(h);
    if (s != LENSED_OK) return s;
    for (int i = 0; i < PH_COUNT; ++i) { h->ms[i] = 0.0; h->launches[i] = 0; }
    CU(h, cudaSetDevice(h->device));
    CU(h, cudaDeviceSynchronize());
    CU(h, cudaMemset(h->d_refined, 0, sizeof(unsigned long long)));
    return LENSED_OK;
}

lensed_status lensed_set_refine(lensed_handle *h, double gain)
{
    if (!h) return fail(nullptr, LENSED_EINVAL, "null handle");
    if (gain != gain) return fail(h, LENSED_EINVAL, "gain is NaN");
    h->refine_gain = gain > 0.0 ? gain : 0.0;
    return LENSED_OK;
}

lensed_status lensed_set_fg_expansion(lensed_handle *h, double tau)
{
    if (!h) return fail(nullptr, LENSED_EINVAL, "null handle");
    if (tau != tau || tau > 0.5) return fail(h, LENSED_EINVAL, "tau = %g outside [0, 0.5]", tau);
    h->fgx_tau = tau > 0.0 ? tau : 0.0;
    return LENSED_OK;
}

namespace {
__global__ void fill_kernel(float *p, size_t n, float value)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) p[i] = value;
}
}  // namespace

lensed_status lensed_debug_fill_frames(lensed_handle *h, float value)
{
    if (!h) return fail(nullptr, LENSED_EINVAL, "null handle");
    if (!isfinite(value)) return fail(h, LENSED_EINVAL, "value must be finite (0 x NaN would leak through the zero taps)");
    CU(h, cudaSetDevice(h->device));
    CU(h, cudaDeviceSynchronize());
    if (h->d_L && h->cap_L) {
        fill_kernel<<<1024, 256>>>(h->d_L, h->cap_L, value);
        CU(h, cudaGetLastError());
        CU(h, cudaDeviceSynchronize());
    }
    return LENSED_OK;
}

lensed_status lensed_get_refined(lensed_handle *h, long long *pixels)
{
    if (!h) return fail(nullptr, LENSED_EINVAL, "null handle");
    if (!pixels) return fail(h, LENSED_EINVAL, "pixels is NULL");
    CU(h, cudaSetDevice(h->device));
    CU(h, cudaDeviceSynchronize());
    unsigned long long n = 0;
    CU(h, cudaMemcpy(&n, h->d_refined, sizeof n, cudaMemcpyDeviceToHost));
    *pixels = (long long)n;
    return LENSED_OK;
}

long long lensed_frame_bytes(const lensed_handle *h)
{
    return h ? (long long)((size_t)h->Hp * h->Wp * sizeof(float)) : -1;
}

lensed_status lensed_set_chunk_bytes(lensed_handle *h, long long bytes)
{
    if (!h) return fail(nullptr, LENSED_EINVAL, "null handle");
    if (bytes < lensed_frame_bytes(h))
        return fail(h, LENSED_EINVAL, "chunk of %lld bytes holds less than one padded frame (%lld bytes)", bytes,
                    lensed_frame_bytes(h));
    h->chunk_bytes = bytes;
    return LENSED_OK;
}

lensed_status lensed_set_conv_shape(lensed_handle *h, int shape)
{
    if (!h) return fail(nullptr, LENSED_EINVAL, "null handle");
    if (shape < 0 || shape > 3) return fail(h, LENSED_EINVAL, "shape = %d is not 0 (narrow), 1 (wide), 2 (strip) or 3 (half-width strip)", shape);
    if (!conv_shape_fits(h->KH, h->NC, shape))
        return fail(h, LENSED_EUNSUPPORTED, "a %d x %d PSF does not fit the %s shape's shared memory", h->KH, h->KW,
                    shape == 0 ? "narrow" : shape == 2 ? "strip" : "half-width strip");
    return build_tiles(h, shape);
}

int lensed_get_conv_shape(const lensed_handle *h) { return h ? h->shape : -1; }

void lensed_debug_force_global_taps(int on) { g_force_global_taps = on != 0; }

int lensed_uses_global_taps(const lensed_handle *h) { return h ? (h->d_gtaps ? 1 : 0) : -1; }

lensed_status lensed_set_static_tracer(lensed_handle *h, int on)
{
    if (!h) return fail(nullptr, LENSED_EINVAL, "null handle");
    if (on && !trace_has_static(h->prog) && !h->jit)
        return fail(h, LENSED_EUNSUPPORTED, "no specialised tracer for this model list");
    h->static_tracer = on != 0;
    return LENSED_OK;
}

int lensed_debug_jit_compile(const int *models, int n_models, int n_quad, char *log, int log_len)
{
    int counts[K_COUNT] = {0};
    if (!models || n_models < 1 || n_quad < 1) return -1;
    for (int m = 0; m < n_models; ++m) {
        if (models[m] < 0 || models[m] >= K_COUNT) return -1;
        counts[models[m]] += 1;
    }
    int n_pos = 0;
    for (int k = 0; k < K_SKY; ++k) n_pos += counts[k];
    std::vector<char> cubin;
    std::string name;
    const std::string msg = jit_compile(counts, trace_pick_np(n_quad), n_pos <= 5 ? 3 : 2, &cubin, &name);
    if (log && log_len > 0) snprintf(log, (size_t)log_len, "%s", msg.c_str());
    return msg.empty() ? (int)cubin.size() : -1;
}

int lensed_get_static_tracer(const lensed_handle *h)
{
    if (!h) return -1;
    return !h->static_tracer ? 0 : trace_has_static(h->prog) ? 1 : 2;
}

lensed_status lensed_issue_probe(int device, int kind, int n_extra, int warps, double *cycles_per_body)
{
    if (!cycles_per_body) return fail(nullptr, LENSED_EINVAL, "lensed_issue_probe: null argument");
    if (cudaSetDevice(device) != cudaSuccess)
        return fail(nullptr, LENSED_ECUDA, "lensed_issue_probe: no CUDA device %d", device);
    const cudaError_t e = run_issue_probe(kind, n_extra, warps, cycles_per_body);
    if (e == cudaErrorInvalidValue) return fail(nullptr, LENSED_EINVAL, "lensed_issue_probe: kind 0..4, n_extra in {0, 8, 16, 32, 64}, warps in {1, 2, 4}");
    if (e != cudaSuccess) return fail(nullptr, LENSED_ECUDA, "lensed_issue_probe: %s", cudaGetErrorString(e));
    return LENSED_OK;
}

lensed_status lensed_fma_peak(int device, int iters, double *tflops)
{
    if (!tflops || iters < 1) return fail(nullptr, LENSED_EINVAL, "lensed_fma_peak: bad argument");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev)
        return fail(nullptr, LENSED_ECUDA, "lensed_fma_peak: no CUDA device %d", device);
    CU(nullptr, cudaSetDevice(device));
    CU(nullptr, run_fma_peak(iters, tflops));
    return LENSED_OK;
}

const char *lensed_last_error(const lensed_handle *h)
{
    return h ? h->err.c_str() : g_last_error.c_str();
}

void lensed_destroy(lensed_handle *h)
{
    if (!h) return;
    cudaSetDevice(h->device);
    cudaDeviceSynchronize();
    for (EventPair &ep : h->used) { cudaEventDestroy(ep.a); cudaEventDestroy(ep.b); }
    for (EventPair &ep : h->pool) { cudaEventDestroy(ep.a); cudaEventDestroy(ep.b); }
    cudaFree(h->d_quad); cudaFree(h->d_quad_pp); cudaFree(h->d_tiles_ll); cudaFree(h->d_tiles_all);
    if (h->shared && h->shared->refs.fetch_sub(1) == 1) {       // the last handle of this problem
        // the pointers of the handle are the shared ones unless create failed half-way
        cudaFree(h->d_image); cudaFree(h->d_wmask); cudaFree(h->d_pix_ll); cudaFree(h->d_pix_all); cudaFree(h->d_gtaps);
        if (h->tap_off >= 0) g_tap_pool.give(h->device, h->tap_off);
        delete h->shared;
    }
    cudaFree(h->d_derived); cudaFree(h->d_L); cudaFree(h->d_partial);
    cudaFree(h->d_derived64); cudaFree(h->d_fixmask); cudaFree(h->d_order); cudaFree(h->d_refined);
    cudaFree(h->d_queue); cudaFree(h->d_queue_count);
    cudaFree(h->d_stage_in); cudaFree(h->d_stage_out);
    delete h;
}

}  // extern "C"
