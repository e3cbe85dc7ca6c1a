// hq_noalloc.cu — include/hq_noalloc.h: the split-K tensor-core GEMM as an entry point that allocates
// nothing.  The split-K partial buffers, which the model carves from the caller's workspace, live in a file-scope
// static __device__ array here; see the header for the sharing rules (one array per GPU, overlapping calls race).
#include <mutex>

#include "hq_common.cuh"
#include "hq_internal.h"

namespace hq {

// ---- the scratch --------------------------------------------------------------------------------------------------
// [split][n_tokens][n_rows] fp32 partial products.  Resident on every GPU that loads this module, until process exit.
constexpr size_t kNoAllocFloats = HQ_NOALLOC_SCRATCH_BYTES / sizeof(float);
static __device__ __align__(256) float g_noalloc_scratch[kNoAllocFloats];

// In HOST code the name g_noalloc_scratch is a host-side stand-in, not a device address.  The address a kernel can use
// is taken once per device with cudaGetSymbolAddress (below, with that device current) and kept here.
constexpr int kNoAllocMaxDevices = 64;
static float *g_scratch_addr[kNoAllocMaxDevices] = {};
static std::mutex g_setup_mutex;

// out[i] = part[0][i] + part[1][i] + ... in that order (bit-reproducible), i < n.  part[z] = part + z * stride.
__global__ void __launch_bounds__(256) sum_partials_kernel(const float *__restrict__ part, int n_parts, size_t stride, float *__restrict__ out,
                                                           size_t n, int vec4) {
    const size_t step = (size_t)gridDim.x * blockDim.x;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (vec4) {
        const size_t n4 = n >> 2;
        for (; i < n4; i += step) {
            float4 acc = ld_act4(part + 4 * i);
            for (int z = 1; z < n_parts; ++z) {
                const float4 v = ld_act4(part + (size_t)z * stride + 4 * i);
                acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
            }
            *reinterpret_cast<float4 *>(out + 4 * i) = acc;
        }
    } else {
        for (; i < n; i += step) {
            float acc = ld_act(part + i);
            for (int z = 1; z < n_parts; ++z) acc += ld_act(part + (size_t)z * stride + i);
            out[i] = acc;
        }
    }
}

// Set-up of the current device; *addr = device address of the scratch on it.  No allocation: cudaGetSymbolAddress
// resolves a symbol of an already defined array, gemm_prepare sets kernel attributes.
static int32_t noalloc_setup_current(float **addr) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return set_error(HQ_ERR_CUDA, "hq_noalloc: cudaGetDevice failed: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= kNoAllocMaxDevices) return set_error(HQ_ERR_UNSUPPORTED, "hq_noalloc: device ordinal %d outside [0, %d)", dev, kNoAllocMaxDevices);
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_addr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p)
            return set_error(HQ_ERR_CUDA, "hq_noalloc: cudaGetSymbolAddress(scratch) failed on device %d: %s", dev, cudaGetErrorString(e));
        e = gemm_prepare();   // shared-memory opt-in of the GEMM kernels on this device
        if (e != cudaSuccess) return set_error(HQ_ERR_CUDA, "hq_noalloc: gemm_prepare failed on device %d: %s", dev, cudaGetErrorString(e));
        g_scratch_addr[dev] = static_cast<float *>(p);
    }
    if (addr) *addr = g_scratch_addr[dev];
    return HQ_OK;
}

}  // namespace hq

using namespace hq;

extern "C" size_t hq_noalloc_scratch_bytes(void) { return HQ_NOALLOC_SCRATCH_BYTES; }

extern "C" int32_t hq_noalloc_setup(void) { return noalloc_setup_current(nullptr); }

extern "C" int32_t hq_gemm_noalloc(void *cuda_stream, const void *w_dev, const void *x_dev, float *out_dev, int32_t n_rows, int32_t k,
                                   int32_t n_tokens, int32_t token_tile, int32_t splits) {
    if (!w_dev || !x_dev || !out_dev || n_rows <= 0 || k <= 0 || n_tokens <= 0 || splits < 1)
        return set_error(HQ_ERR_INVALID_ARG, "hq_gemm_noalloc: bad argument (NULL pointer, non-positive size or splits < 1)");
    if (token_tile != 32 && token_tile != 64 && token_tile != 128 && token_tile != 256)
        return set_error(HQ_ERR_INVALID_ARG, "hq_gemm_noalloc: token_tile must be 32, 64, 128 or 256");
    if (k % 8 != 0) return set_error(HQ_ERR_UNSUPPORTED, "hq_gemm_noalloc: k must be a multiple of 8");
    // the split count launch_gemm will run with (a fixed point of its own clamping: see launch_gemm)
    const int kblocks = (k + 63) / 64;
    int sp = splits > kblocks ? kblocks : splits;
    const int per = (kblocks + sp - 1) / sp;
    sp = (kblocks + per - 1) / per;
    const size_t n = (size_t)n_tokens * (size_t)n_rows, need = (size_t)sp * n * sizeof(float);
    if (need > HQ_NOALLOC_SCRATCH_BYTES)
        return set_error(HQ_ERR_CAPACITY, "hq_gemm_noalloc: %d splits x %d tokens x %d rows need %zu bytes of scratch, the static array holds %zu",
                         sp, n_tokens, n_rows, need, (size_t)HQ_NOALLOC_SCRATCH_BYTES);
    float *scratch = nullptr;
    const int32_t rc = noalloc_setup_current(&scratch);
    if (rc != HQ_OK) return rc;

    TensorMap mw, mx;   // host-side descriptors, passed to the kernel by value
    if (!make_tensor_map_16b(&mw, w_dev, (uint64_t)n_rows, (uint64_t)k, 128) ||
        !make_tensor_map_16b(&mx, x_dev, 2 * (uint64_t)n_tokens, (uint64_t)k, (uint32_t)token_tile))
        return set_error(HQ_ERR_CUDA, "hq_gemm_noalloc: cuTensorMapEncodeTiled failed");
    const cudaStream_t stream = (cudaStream_t)cuda_stream;
    const LaunchCtx lc{stream, false, 148};
    // every split z stores its partial [n_tokens][n_rows] at scratch + z * n: each element the sum below reads is written
    // by this call, so the array needs no clearing between calls
    cudaError_t e = launch_gemm(lc, EPI_STORE, mw, nullptr, mx, n_tokens, n_rows, k, n_tokens, token_tile, sp, scratch, nullptr, 0, n_rows, n);
    if (e != cudaSuccess) return set_error(HQ_ERR_CUDA, "hq_gemm_noalloc: GEMM launch failed: %s", cudaGetErrorString(e));
    const int vec4 = (n % 4 == 0 && (reinterpret_cast<uintptr_t>(out_dev) & 15) == 0) ? 1 : 0;
    const size_t work = vec4 ? n / 4 : n;
    size_t blocks = (work + 255) / 256;
    if (blocks > 4 * 148) blocks = 4 * 148;
    sum_partials_kernel<<<(unsigned)blocks, 256, 0, stream>>>(scratch, sp, n, out_dev, n, vec4);
    e = cudaGetLastError();
    if (e != cudaSuccess) return set_error(HQ_ERR_CUDA, "hq_gemm_noalloc: sum launch failed: %s", cudaGetErrorString(e));
    return HQ_OK;
}
