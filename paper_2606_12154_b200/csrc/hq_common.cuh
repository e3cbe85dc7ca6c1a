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

// ---- mbarrier / bulk async copy (TMA) / thread-block cluster wrappers -------------------------------------
__device__ __forceinline__ uint32_t smem_addr_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_addr_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_addr_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
// acquire at cluster scope: pairs with remote arrives (mbar_arrive_remote) of other CTAs of the cluster
__device__ __forceinline__ bool mbar_try_wait_cluster(uint64_t *bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_addr_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {}
}
__device__ __forceinline__ void bulk_g2s(void *smem_dst, const void *gmem_src, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_addr_u32(smem_dst)),
                 "l"(gmem_src), "r"(bytes), "r"(smem_addr_u32(bar))
                 : "memory");
}
// weights are read once per token: evict-first keeps the KV cache and the activations resident in the 126 MB L2
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void bulk_g2s_hint(void *smem_dst, const void *gmem_src, uint32_t bytes, uint64_t *bar, uint64_t pol) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
                     smem_addr_u32(smem_dst)),
                 "l"(gmem_src), "r"(bytes), "r"(smem_addr_u32(bar)), "l"(pol)
                 : "memory");
}
__device__ __forceinline__ uint32_t cluster_ctarank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ uint32_t cluster_id_x() { uint32_t r; asm volatile("mov.u32 %0, %%clusterid.x;" : "=r"(r)); return r; }
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// address of the same shared-memory location in CTA `rank` of the cluster (distributed shared memory)
__device__ __forceinline__ uint32_t cluster_map(uint32_t smem_addr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_cluster_f32x2(uint32_t addr, float a, float b) {
    asm volatile("st.shared::cluster.v2.f32 [%0], {%1, %2};" ::"r"(addr), "f"(a), "f"(b) : "memory");
}
__device__ __forceinline__ float ld_cluster_f32(uint32_t addr) {
    float v;
    asm volatile("ld.shared::cluster.f32 %0, [%1];" : "=f"(v) : "r"(addr) : "memory");
    return v;
}
// Asynchronous store of two floats into the shared memory of a CTA of the cluster; the bytes are credited (complete_tx)
// to an mbarrier of the SAME destination CTA, whose waiters then see the data: a push with no fence and no release (a
// release at cluster scope also waits for the SM's bulk copies in flight: measured ~1.5 us under a weight prefetch).
__device__ __forceinline__ void st_async_f32x2(uint32_t cluster_addr, float a, float b, uint32_t cluster_mbar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f32 [%0], {%1, %2}, [%3];" ::"r"(cluster_addr),
                 "f"(a), "f"(b), "r"(cluster_mbar)
                 : "memory");
}
// L2 prefetch of a contiguous global range (bytes a multiple of 16)
__device__ __forceinline__ void bulk_prefetch_l2(const void *gmem_src, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(gmem_src), "r"(bytes) : "memory");
}

// ---- step timeline (hq_debug_step_trace): per launch [0] earliest CTA start, [1] earliest end of the dependency wait,
// [2] latest CTA end, [3] latest CTA start (global timer, ns).  One thread per CTA stamps; NULL = off.
__device__ __forceinline__ void step_stamp(unsigned long long *trace, int slot, int which) {
    if (trace) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        if (which < 2) atomicMin(trace + 4 * slot + which, t);
        else atomicMax(trace + 4 * slot + which, t);
    }
}

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

// ---- packed fp32 pairs: Blackwell issues two fp32 FMAs per instruction (fma.rn.f32x2 -> FFMA2) ----------------------
typedef unsigned long long f32x2_t;
__device__ __forceinline__ f32x2_t pack_f32x2(float lo, float hi) {
    f32x2_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ float sum_f32x2(f32x2_t v) {
    float lo, hi;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
    return lo + hi;
}
__device__ __forceinline__ void ffma2(f32x2_t &acc, f32x2_t a, f32x2_t b) {
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(a), "l"(b));
}
// two bf16 packed in a u32 (element 0 in the low half) -> fp32 pair, exact
__device__ __forceinline__ f32x2_t bf16x2_to_f32x2(uint32_t u) { return pack_f32x2(__uint_as_float(u << 16), __uint_as_float(u & 0xFFFF0000u)); }
// 8 bf16 (one 16-byte chunk) times 8 fp32 held as 4 pairs, accumulated pairwise into acc[0..3]: 4 FFMA2 + 8 ALU ops
__device__ __forceinline__ void dot8_x2(const uint4 &w, const f32x2_t (&x)[4], f32x2_t (&acc)[4]) {
    ffma2(acc[0], bf16x2_to_f32x2(w.x), x[0]);
    ffma2(acc[1], bf16x2_to_f32x2(w.y), x[1]);
    ffma2(acc[2], bf16x2_to_f32x2(w.z), x[2]);
    ffma2(acc[3], bf16x2_to_f32x2(w.w), x[3]);
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
