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

}  // namespace hq
