// chisq_static.cu -- lensed_chisq_static (include/lensed.h): logL = -1/2 sum_i w_i (d_i - L*_i)^2
// (eqs. 16-17) for a batch of model images that are ALREADY on the device, from a
// call that allocates no memory at all.
//
// Who this is for.  lensed_loglike grows its scratch (cudaMallocAsync) whenever it sees a batch
// larger than any before, and lensed_create allocates the problem's arrays.  Some users of this
// library must not allocate once their set-up is over:
//   * a sampler that lives inside a process whose other framework has already claimed the device
//     memory for its own pool (PyTorch's caching allocator with a memory fraction set, an XLA
//     client that preallocates most of the GPU): a late cudaMalloc from here simply fails;
//   * a farm of lensed_clone handles on several streams: cudaMalloc / cudaFree synchronise the
//     whole device, so one worker's growth stalls every other worker's kernels;
//   * a job held to a fixed memory budget (a MIG slice, an MPS client with a memory limit) whose
//     operator forbids allocation after start-up so that the budget can be checked once.
// Such a caller keeps the images it wants scored in buffers of its own (filled by lensed_render at
// a batch size it warmed up during set-up, by its own forward model, or by lensed_render plus an
// instrument term the library does not know) and calls this entry point, which needs only those
// buffers and the fixed array below.
//
// The kernel is the variant of the path's chi-square stage (conv.cu: per-tile FP64 partials in the
// handle's grown `d_partial`, summed in tile order by final_kernel) with the partials in a
// file-scope device array instead: kMaxVectors x kMaxBlocks doubles and one arrival counter per
// vector, 1 040 KB that every GPU loading the library holds until the process exits.  Same
// summation discipline as the path: FP32 difference, FP64 from the product on, fixed order, so the
// result is bitwise reproducible.
//
// Shares nothing with oracle/.
#include "../../include/lensed.h"
#include "lensed_internal.h"

#include <math.h>
#include <stddef.h>

#include <mutex>

using namespace lensed;

namespace {

constexpr int kMaxVectors = LENSED_CHISQ_STATIC_MAX_VECTORS;   // per call
constexpr int kMaxBlocks = 32;                                 // blocks that share one vector's pixels
constexpr int kThreads = 256;
constexpr int kPixelsPerBlock = 4096;                          // below this a vector is not split further
constexpr long long kMaxPixels = 1ll << 30;                    // 32767^2 (lensed_create's limit) fits

struct Scratch {
    double partial[(size_t)kMaxVectors * kMaxBlocks];   // [vector][block], written before they are read: never cleared
    unsigned arrived[kMaxVectors];                      // blocks of the vector that have stored their partial:
                                                        // MUST be zero when the kernel starts (cleared per call)
};

// The scratch itself.  In HOST code this name is only a stand-in the runtime registers for the
// symbol, not a device address: never pass it to a kernel or a memset from the host.  The host
// side gets the real address from cudaGetSymbolAddress (scratch_address below), per device,
// because every device that loads this module has its own copy.
static __device__ __align__(256) unsigned char g_chisq_scratch[sizeof(Scratch)];

std::mutex g_setup_mutex;
void *g_scratch_ptr[64] = {nullptr};     // per device ordinal, filled on the first call on that device

// Device address of g_chisq_scratch on `device`, which must be current.  The first call on a
// device asks the runtime (this may load the module onto the device: do it outside any stream
// capture); later calls return the cached pointer.
cudaError_t scratch_address(int device, void **out)
{
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_ptr[device]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_chisq_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_scratch_ptr[device] = p;
    }
    *out = g_scratch_ptr[device];
    return cudaSuccess;
}

// Block (k, b) sums vector b's pixels [k len, (k + 1) len) in a fixed order (thread-strided in
// FP64, shuffle tree, warps in order), stores the partial, and the block that arrives last adds
// the vector's partials in block order.  Pixels with w = 0 (masked) are never touched: the model
// may hold anything there, as in the path's convolution epilogue (conv.cu).
__global__ void __launch_bounds__(kThreads) chisq_static_kernel(const float *__restrict__ image, const float *__restrict__ weight,
                                                                const float *__restrict__ model, long long n_pix, long long len,
                                                                double *partial, unsigned *arrived, float *logl)
{
    const int b = blockIdx.y, k = blockIdx.x, n_blocks = gridDim.x;
    const float *m = model + (size_t)b * n_pix;
    const long long lo = k * len, hi = min(n_pix, lo + len);
    double acc = 0.0;
    for (long long i = lo + threadIdx.x; i < hi; i += kThreads) {
        const float w = __ldg(weight + i);
        if (w != 0.0f) {
            const float diff = __ldg(image + i) - m[i];        // FP32, as the path forms d - L*
            acc = fma((double)w * (double)diff, (double)diff, acc);
        }
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
    __shared__ double warp_sum[kThreads / 32];
    if ((threadIdx.x & 31) == 0) warp_sum[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int wp = 0; wp < kThreads / 32; ++wp) s += warp_sum[wp];
        partial[(size_t)b * kMaxBlocks + k] = s;
        __threadfence();                                        // the partial is visible before the arrival is
        if (atomicAdd(arrived + b, 1u) == (unsigned)(n_blocks - 1)) {        // the vector's last block
            __threadfence();
            double chi2 = 0.0;
            for (int j = 0; j < n_blocks; ++j) chi2 += __ldcg(partial + (size_t)b * kMaxBlocks + j);
            // a non-finite model pixel under a non-zero weight (lensed_render's NaN image of a vector
            // outside the model domain): -inf, what lensed_loglike returns for such a vector
            logl[b] = chi2 == chi2 ? (float)(-0.5 * chi2) : -INFINITY;
        }
    }
}

}  // namespace

extern "C" lensed_status lensed_chisq_static(int device, const float *image_dev, const float *weight_dev, long long n_pix,
                                             const float *model_dev, int B, float *logl_dev, void *cuda_stream)
{
    // argument checks first: none of them needs a device
    if (!image_dev || !weight_dev || !model_dev || !logl_dev)
        return (lensed_status)handle_fail(nullptr, LENSED_EINVAL, "lensed_chisq_static: null device pointer");
    if (B < 1) return (lensed_status)handle_fail(nullptr, LENSED_EINVAL, "lensed_chisq_static: B = %d < 1", B);
    if (n_pix < 1) return (lensed_status)handle_fail(nullptr, LENSED_EINVAL, "lensed_chisq_static: n_pix = %lld < 1", n_pix);
    if (B > kMaxVectors)
        return (lensed_status)handle_fail(nullptr, LENSED_EINVAL,
                                          "lensed_chisq_static: B = %d exceeds LENSED_CHISQ_STATIC_MAX_VECTORS = %d, all the fixed "
                                          "scratch array holds; split the batch into calls of at most %d vectors",
                                          B, kMaxVectors, kMaxVectors);
    if (n_pix > kMaxPixels)
        return (lensed_status)handle_fail(nullptr, LENSED_EINVAL, "lensed_chisq_static: n_pix = %lld exceeds the limit of %lld pixels per image",
                                          n_pix, kMaxPixels);
    if (device < 0 || device >= 64) return (lensed_status)handle_fail(nullptr, LENSED_EINVAL, "lensed_chisq_static: device %d", device);

    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return (lensed_status)handle_fail(nullptr, LENSED_ECUDA, "lensed_chisq_static: cudaSetDevice(%d): %s", device, cudaGetErrorString(e));
    void *base = nullptr;
    e = scratch_address(device, &base);
    if (e != cudaSuccess)
        return (lensed_status)handle_fail(nullptr, LENSED_ECUDA, "lensed_chisq_static: cudaGetSymbolAddress of the scratch array: %s", cudaGetErrorString(e));
    double *partial = reinterpret_cast<double *>(static_cast<unsigned char *>(base) + offsetof(Scratch, partial));
    unsigned *arrived = reinterpret_cast<unsigned *>(static_cast<unsigned char *>(base) + offsetof(Scratch, arrived));

    cudaStream_t st = (cudaStream_t)cuda_stream;
    // the array still holds the previous call's counters (or those of a call that was aborted half
    // way): the B this call uses start at zero.  The partials need no clearing.
    e = cudaMemsetAsync(arrived, 0, (size_t)B * sizeof(unsigned), st);
    if (e != cudaSuccess) return (lensed_status)handle_fail(nullptr, LENSED_ECUDA, "lensed_chisq_static: cudaMemsetAsync: %s", cudaGetErrorString(e));
    long long n_blocks = (n_pix + kPixelsPerBlock - 1) / kPixelsPerBlock;
    if (n_blocks > kMaxBlocks) n_blocks = kMaxBlocks;
    const long long len = (n_pix + n_blocks - 1) / n_blocks;
    n_blocks = (n_pix + len - 1) / len;                          // no empty block
    chisq_static_kernel<<<dim3((unsigned)n_blocks, (unsigned)B), kThreads, 0, st>>>(image_dev, weight_dev, model_dev, n_pix, len, partial,
                                                                                    arrived, logl_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) return (lensed_status)handle_fail(nullptr, LENSED_ECUDA, "lensed_chisq_static: launch: %s", cudaGetErrorString(e));
    return LENSED_OK;
}
