// hq_probe.cu — read-only streaming probe ("a read-only streaming probe the bench runs itself (a
// sum-reduction) as the practical ceiling").  A third roofline denominator beside the 8 TB/s spec and the measured copy
// bandwidth: what a kernel that only READS HBM, like the decode GEMVs, can reach on this box.
#include "hq_common.cuh"
#include "hq_internal.h"

namespace hq {

// grid-stride sum of 32-bit words; 8 independent 16-byte loads per thread in flight, non-coherent path, no L1 allocation
__global__ void __launch_bounds__(512) read_probe_kernel(const uint4 *__restrict__ src, size_t n16, unsigned int *out) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned int acc = 0u;
    for (; i + 7 * stride < n16; i += 8 * stride) {
        uint4 v[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) v[j] = ld_weight16(src + i + (size_t)j * stride);
#pragma unroll
        for (int j = 0; j < 8; ++j) acc += v[j].x + v[j].y + v[j].z + v[j].w;
    }
    for (; i < n16; i += stride) {
        const uint4 v = ld_weight16(src + i);
        acc += v.x + v.y + v.z + v.w;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) atomicAdd(out, acc);
}

cudaError_t launch_read_probe(cudaStream_t stream, const void *src, size_t bytes, unsigned int *out, int n_sms) {
    read_probe_kernel<<<n_sms * 4, 512, 0, stream>>>(static_cast<const uint4 *>(src), bytes / 16, out);
    return cudaGetLastError();
}

// ---- bulk-copy size probe ---------------------------------------------------------------------------------------------
// What one SM pulls from HBM through cp.async.bulk as a function of the size of the individual copy: n_ctas CTAs (one per
// SM) each stream their share of the buffer through a ring of 3 x 64 KB stages, a stage being 64 KB / copy_bytes copies
// issued by 16 lanes; nothing is computed (a consumer thread releases every stage as soon as it has landed).  This is the
// measurement behind "one copy per stage" in hq_stream.cu / hq_attn.cu (profiles/r02_copy_size.md).
constexpr int kCpStages = 3, kCpStageBytes = 65536;
__global__ void __launch_bounds__(64, 1) copy_probe_kernel(const uint8_t *__restrict__ src, size_t bytes, int copy_bytes) {
    extern __shared__ __align__(128) uint8_t cp_smem[];
    __shared__ uint64_t full[kCpStages], empty[kCpStages];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < kCpStages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
        mbar_fence_init();
    }
    __syncthreads();
    const size_t n_stages = bytes / kCpStageBytes / gridDim.x;
    const uint8_t *base = src + (size_t)blockIdx.x * n_stages * kCpStageBytes;
    const int per_stage = kCpStageBytes / copy_bytes;
    if (warp == 0) {
        const uint64_t pol = l2_policy_evict_first();
        for (size_t n = 0; n < n_stages; ++n) {
            const int slot = (int)(n % kCpStages);
            while (!mbar_try_wait(&empty[slot], (uint32_t)(((n / kCpStages) & 1) ^ 1))) {}
            if (lane == 0) mbar_expect_tx(&full[slot], kCpStageBytes);
            __syncwarp();
            for (int c = lane; c < per_stage; c += 32)
                bulk_g2s_hint(cp_smem + (size_t)slot * kCpStageBytes + (size_t)c * copy_bytes,
                              base + n * kCpStageBytes + (size_t)c * copy_bytes, (uint32_t)copy_bytes, &full[slot], pol);
        }
    } else if (lane == 0) {
        for (size_t n = 0; n < n_stages; ++n) {
            const int slot = (int)(n % kCpStages);
            while (!mbar_try_wait(&full[slot], (uint32_t)((n / kCpStages) & 1))) {}
            mbar_arrive(&empty[slot]);
        }
    }
}

cudaError_t launch_copy_probe(cudaStream_t stream, const void *src, size_t bytes, int copy_bytes, int n_ctas) {
    cudaError_t e = cudaFuncSetAttribute(copy_probe_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kCpStages * kCpStageBytes);
    if (e != cudaSuccess) return e;
    copy_probe_kernel<<<n_ctas, 64, kCpStages * kCpStageBytes, stream>>>(static_cast<const uint8_t *>(src), bytes, copy_bytes);
    return cudaGetLastError();
}

}  // namespace hq
