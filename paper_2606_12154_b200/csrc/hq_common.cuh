// hq_common.cuh — device helpers shared by the libhq translation units (sm_100a only).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace hq {

// ---- programmatic dependent launch (PDL) ----------------------------------------------------------
// launch_dependents: lets the next kernel in the stream/graph start its prologue (weight prefetch).
// grid_dep_wait: blocks until every prerequisite grid has completed and its writes are visible.
__device__ __forceinline__ void pdl_launch_dependents() {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// ---- loads ------------------------------------------------------------------------------------------
// Weights: immutable, streamed once per token -> non-coherent path, do not allocate in L1.
__device__ __forceinline__ uint4 ld_weight16(const void *p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}
// Activations written by an earlier kernel that may still have been running when this CTA
// started (PDL): read through L2 only (never a stale L1 line).
__device__ __forceinline__ float4 ld_act4(const float *p) { return __ldcg(reinterpret_cast<const float4 *>(p)); }
__device__ __forceinline__ float ld_act(const float *p) { return __ldcg(p); }
__device__ __forceinline__ int ld_act(const int *p) { return __ldcg(p); }

// bf16 pair (packed in a u32, element 0 in the low half) -> two fp32, exact
__device__ __forceinline__ float bf16lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf16hi(uint32_t u) { return __uint_as_float(u & 0xFFFF0000u); }

// 8 bf16 (one 16-byte chunk) dotted with 8 fp32
__device__ __forceinline__ float dot8(const uint4 &w, const float (&x)[8], float acc) {
    acc = fmaf(bf16lo(w.x), x[0], acc);
    acc = fmaf(bf16hi(w.x), x[1], acc);
    acc = fmaf(bf16lo(w.y), x[2], acc);
    acc = fmaf(bf16hi(w.y), x[3], acc);
    acc = fmaf(bf16lo(w.z), x[4], acc);
    acc = fmaf(bf16hi(w.z), x[5], acc);
    acc = fmaf(bf16lo(w.w), x[6], acc);
    acc = fmaf(bf16hi(w.w), x[7], acc);
    return acc;
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// Transposed butterfly: every lane holds N partial sums v[0..N) (N a power of two <= 32).  After
// the call v[0] on every lane holds the warp total of row warp_row_of_lane<N>(lane); N-1 + log2(32/N)
// shuffles instead of 5N.
template <int N>
__device__ __forceinline__ void warp_reduce_rows(float (&v)[N], int lane) {
    static_assert(N >= 1 && N <= 32 && (N & (N - 1)) == 0, "N must be a power of two");
    int bit = 16;
#pragma unroll
    for (int n = N; n > 1; n >>= 1, bit >>= 1) {
        const bool up = (lane & bit) != 0;
#pragma unroll
        for (int i = 0; i < n / 2; ++i) {
            float keep = up ? v[i + n / 2] : v[i];
            float send = up ? v[i] : v[i + n / 2];
            v[i] = keep + __shfl_xor_sync(0xffffffffu, send, bit);
        }
    }
    for (; bit > 0; bit >>= 1) v[0] += __shfl_xor_sync(0xffffffffu, v[0], bit);
}
// Row index (0..N-1) whose total lane `lane` holds in v[0] after warp_reduce_rows<N>.
template <int N>
__device__ __forceinline__ int warp_row_of_lane(int lane) {
    int row = 0, bit = 16;
#pragma unroll
    for (int n = N; n > 1; n >>= 1, bit >>= 1) row += (lane & bit) ? n / 2 : 0;
    return row;
}
// Lowest lane holding each row is the one whose bits below the consumed ones are zero.
template <int N>
__device__ __forceinline__ bool warp_row_leader(int lane) {
    int used = 0, bit = 16;
#pragma unroll
    for (int n = N; n > 1; n >>= 1, bit >>= 1) used |= bit;
    return (lane & ~used & 31) == 0;
}

// float -> u32 whose unsigned order equals the float order (for packed atomicMax argmax)
__device__ __forceinline__ uint32_t float_order_key(float f) {
    uint32_t u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ unsigned long long pack_argmax(float v, int idx) {
    return (static_cast<unsigned long long>(float_order_key(v)) << 32) |
           static_cast<unsigned long long>(0xFFFFFFFFu - static_cast<uint32_t>(idx));
}
__device__ __forceinline__ int unpack_argmax_idx(unsigned long long p) {
    return static_cast<int>(0xFFFFFFFFu - static_cast<uint32_t>(p & 0xFFFFFFFFull));
}

// x = hi + lo with hi = bf16(x), lo = bf16(x - hi): 16 mantissa bits in two tensor-core operands
__device__ __forceinline__ void split_bf16(float x, __nv_bfloat16 &hi, __nv_bfloat16 &lo) {
    hi = __float2bfloat16_rn(x);
    lo = __float2bfloat16_rn(x - __bfloat162float(hi));
}
__device__ __forceinline__ void split_bf16x2(float a, float b, uint32_t &hi, uint32_t &lo) {
    __nv_bfloat162 h = __floats2bfloat162_rn(a, b);
    const float2 hf = __bfloat1622float2(h);
    __nv_bfloat162 l = __floats2bfloat162_rn(a - hf.x, b - hf.y);
    hi = *reinterpret_cast<uint32_t *>(&h);
    lo = *reinterpret_cast<uint32_t *>(&l);
}

__device__ __forceinline__ float silu_f(float z) { return z / (1.0f + expf(-z)); }

}  // namespace hq
