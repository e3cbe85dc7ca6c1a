// hq_gemm.cu — tcgen05 / TMEM / TMA GEMM for envelope prefill and batched decode.
//
//   D[n, t] = sum_k W[n, k] * X[t, k]        W: bf16 weights [N, K] (nn.Linear layout, K-major)
//                                            X: activations [T, K] (K-major) as two bf16 planes hi + lo (act_t)
// "Swap-AB": the weight tile is the UMMA A operand (M = 128 weight rows), the token tile is the
// B operand (UMMA N = NT tokens, 32..256), so the accumulator D lives in TMEM with one weight row
// per lane and one token per column, and every weight byte is streamed from HBM exactly once per
// token tile.  Both operands are staged by TMA (cp.async.bulk.tensor, SWIZZLE_128B, 64-element
// K blocks) into an mbarrier ring; one elected thread issues tcgen05.mma; four epilogue warps
// read TMEM with tcgen05.ld and apply the fused epilogue:
//   EPI_STORE   out_f32[t][n]  = D            (split-K: atomic add into a zeroed buffer)
//   EPI_RESID   x[t][n]       += D            (residual add; split-K partials add atomically)
//   EPI_SWIGLU  act[t][f]      = hi/lo bf16 of silu(D_gate) * D_up   two accumulators, two weight maps
//   EPI_SWIGLU64  the same result from 64-row weight tiles: one CTA takes 64 gate rows AND the 64 up rows of the same
//               features as the two halves of ONE 128-row A tile (one accumulator; the epilogue warps of the up half
//               hand their values to the gate half through shared memory).  Twice the CTAs of EPI_SWIGLU: the form
//               batched decode uses, where ffn / 128 tiles leave more than half of the SMs idle.
// Warp roles (192 threads): warp 0 TMA producer, warp 1 TMEM owner + MMA issuer, warps 2-5 epilogue.
#include <cuda.h>

#include "hq_common.cuh"
#include "hq_internal.h"

namespace hq {

constexpr int kGemmThreads = 192;
constexpr int kBlockM = 128;  // weight rows per CTA (UMMA M)
constexpr int kBlockK = 64;   // bf16 elements per K block = 128 bytes = one swizzle row

// ---- PTX wrappers --------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbarrier_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbarrier_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbarrier_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred P1;\n\tLAB_WAIT:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
        "@P1 bra DONE;\n\tbra LAB_WAIT;\n\tDONE:\n\t}" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_2d(const CUtensorMap *map, uint64_t *bar, void *smem_dst, int c0, int c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(
            smem_u32(smem_dst)),
        "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
        : "memory");
}
__device__ __forceinline__ void tcgen05_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tcgen05_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tcgen05_commit(uint64_t *bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// D[tmem] (+)= A[smem desc] * B[smem desc]
__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem_d),
        "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate)
        : "memory");
}
// ---- CTA pair (cta_group::2): two CTAs of a cluster run ONE MMA of M = 256: each holds 128 rows of A (weights) and half of
// the rows of B (here: one of the two activation planes); both TMA-load into their own shared memory and credit the bytes to
// the LEADER's (even rank's) mbarrier; the leader issues the MMA and its commit arrives on the barriers of both CTAs.
constexpr uint32_t kPeerBitMask = 0xFEFFFFFFu;   // clears the peer bit of a shared-window address: the even CTA of the pair
__device__ __forceinline__ void tma_load_2d_pair(const CUtensorMap *map, uint64_t *leader_bar, void *smem_dst, int c0, int c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(
            smem_u32(smem_dst)),
        "l"(map), "r"(smem_u32(leader_bar) & kPeerBitMask), "r"(c0), "r"(c1)
        : "memory");
}
__device__ __forceinline__ void umma_bf16_pair(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, {%5, %5, %5, %5, %5, %5, %5, %5}, p;\n\t}" ::"r"(tmem_d),
        "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate), "r"(0u)
        : "memory");
}
// arrives (once the MMAs issued so far have retired) on the barrier at the same shared-memory offset in BOTH CTAs of the pair
__device__ __forceinline__ void tcgen05_commit_pair(uint64_t *bar) {
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(smem_u32(bar)),
                 "h"((unsigned short)3)
                 : "memory");
}

// 32 lanes x 32 columns of fp32: thread (lane) gets 32 consecutive columns of its own TMEM lane
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
          "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
          "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// K-major, SWIZZLE_128B shared-memory matrix descriptor: rows of 128 bytes, 8-row groups 1024 bytes
// apart (stride byte offset); leading byte offset unused for swizzled K-major; descriptor version 1.
__device__ __forceinline__ uint64_t make_smem_desc(uint32_t smem_addr) {
    uint64_t d = 0;
    d |= (uint64_t)((smem_addr & 0x3FFFF) >> 4);        // start address, bits [0,14)
    d |= (uint64_t)(1024 >> 4) << 32;                   // stride byte offset, bits [32,46)
    d |= (uint64_t)1 << 46;                             // version = 1 (sm_100)
    d |= (uint64_t)2 << 61;                             // layout type SWIZZLE_128B
    return d;
}
// kind::f16 instruction descriptor: D fp32 (bits 4-5 = 1), A and B bf16 (bits 7-9 and 10-12 = 1; the two
// formats must match: a bf16 x fp16 descriptor raises an illegal-instruction fault on sm_100a), both K-major
// (bits 15, 16 = 0), N >> 3 at bits 17-22, M >> 4 at bits 24-28
__host__ __device__ inline uint32_t make_idesc(int n, int m = kBlockM) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(m >> 4) << 24);
}

__device__ __forceinline__ unsigned long long gemm_time() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// ---- epilogue helpers.  The epilogue runs after the last MMA with nothing left to overlap it (one tile per CTA), and all
// CTAs reach it together: its length is pure instruction count (measured with globaltimer stamps: 0.85 us per 32-token
// chunk of plain stores with a bounds branch and a mode branch per element, 2.9 us per chunk of the SwiGLU form; after
// the rewrite below ~0.3 / ~1 us).  So: no per-element branches (a chunk is either complete or takes the predicated
// copy of the loop), reciprocal and exponential from the SFU, and bf16 outputs leave as 32-bit pairs.
// a[j] = silu(g[j]) * u[j] for the 32 tokens of a chunk, as four passes over the registers: 32 independent ex2, then 32
// independent rcp (SFU approximations, <= 2 ulp each) -- written element by element the compiler chained exp -> add ->
// rcp -> mul per element and the 32 chains ran back to back (2.1 us per chunk, measured).
__device__ __forceinline__ void swiglu32(const uint32_t (&g)[32], const float (&u)[32], float (&a)[32]) {
    float e[32];
#pragma unroll
    for (int j = 0; j < 32; ++j) asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e[j]) : "f"(__uint_as_float(g[j]) * -1.4426950408889634f));
#pragma unroll
    for (int j = 0; j < 32; ++j) e[j] += 1.0f;
#pragma unroll
    for (int j = 0; j < 32; ++j) asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(e[j]) : "f"(e[j]));
#pragma unroll
    for (int j = 0; j < 32; ++j) a[j] = (__uint_as_float(g[j]) * e[j]) * u[j];
}

// a[j]: this lane's feature n, token j of the chunk (32 tokens).  Writes the hi / lo bf16 planes out[t][n]: lanes exchange
// with their neighbour so that an even lane stores features (n, n + 1) of an even token and an odd lane those of the
// next token, as one 32-bit word per plane (half the store instructions; 64 B per token row and instruction).
// Needs even n0, ld and n_rows (pairs never straddle the end of a row or of the matrix).
__device__ __forceinline__ void store_act_pairs(const float (&a)[32], act_t *out, size_t lo_offset, size_t ld, int n, bool row_ok, int nvalid, int lane) {
    const bool odd = lane & 1;
    act_t *dst = out + (size_t)(odd ? 1 : 0) * ld + (n - (odd ? 1 : 0));
#pragma unroll
    for (int j = 0; j < 32; j += 2) {
        const float other = __shfl_xor_sync(0xffffffffu, odd ? a[j] : a[j + 1], 1);
        const float x0 = odd ? other : a[j], x1 = odd ? a[j + 1] : other;   // features (n even, n even + 1) of token j + odd
        uint32_t hi, lo;
        split_bf16x2(x0, x1, hi, lo);
        if (row_ok && j + (odd ? 1 : 0) < nvalid) {
            *reinterpret_cast<uint32_t *>(dst + (size_t)j * ld) = hi;
            *reinterpret_cast<uint32_t *>(dst + lo_offset + (size_t)j * ld) = lo;
        }
    }
}
__device__ __forceinline__ void store_act_scalar(const float (&a)[32], act_t *out, size_t lo_offset, size_t ld, bool row_ok, int nvalid) {
#pragma unroll
    for (int j = 0; j < 32; ++j) {
        act_t hi, lo;
        split_bf16(a[j], hi, lo);
        if (row_ok && j < nvalid) {
            out[(size_t)j * ld] = hi;
            out[lo_offset + (size_t)j * ld] = lo;
        }
    }
}

// TRACE: the timeline instantiations (hq_debug_gemm_timeline) are separate kernels: the stamps cost the batched-decode
// step 3 % when they were run-time branches in the product kernels.
template <int MODE, int CTAS, bool TRACE = false>
__global__ void __launch_bounds__(kGemmThreads, 1)
gemm_tc_kernel(const __grid_constant__ CUtensorMap map_w, const __grid_constant__ CUtensorMap map_w2,
               const __grid_constant__ CUtensorMap map_w3, const __grid_constant__ CUtensorMap map_x, const GemmParams p) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    constexpr int NACC = (MODE == EPI_SWIGLU) ? 2 : 1;
    constexpr bool HALF = MODE == EPI_SWIGLU64;
    const int NT = p.NT;
    const uint32_t a_bytes = kBlockM * kBlockK * 2;          // 16 KB per weight tile
    const uint32_t b_bytes = (uint32_t)NT * kBlockK * 2;      // one plane (hi or lo) of the token tile
    // CTA pair: this CTA holds ONE plane (rank 0 hi, rank 1 lo): together the B operand of 2 NT rows of the pair's MMA
    const uint32_t stage_bytes = NACC * a_bytes + (CTAS == 2 ? 1 : 2) * b_bytes;
    const uint32_t pair_rank = CTAS == 2 ? cluster_ctarank() : 0;
    const int stages = p.stages;

    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    uint64_t *full_bar = reinterpret_cast<uint64_t *>(smem + (size_t)stages * stage_bytes);
    uint64_t *empty_bar = full_bar + stages;
    uint64_t *acc_bar = empty_bar + stages;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(acc_bar + 1);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n0 = blockIdx.x * (HALF ? kBlockM / 2 : kBlockM);   // first weight row of this CTA
    const int t0 = blockIdx.y * NT;                // first token of this CTA
    const int kb0 = blockIdx.z * p.k_blocks_per_split;
    const int kb1 = min(kb0 + p.k_blocks_per_split, p.k_blocks);
    const int nkb = kb1 - kb0;
    // NT <= 128: the hi and lo activation planes of a stage lie back to back and are ONE B operand of 2 NT rows: one MMA per
    // K step fills D columns [0, NT) with W x_hi and [NT, 2 NT) with W x_lo (half the MMA instructions, a quarter less
    // operand traffic from shared memory than two MMAs into the same columns); the epilogue adds the two halves
    const bool stacked = NT <= 128;   // always true for CTA pairs (launch_mode)
    const int acc_cols = stacked ? 2 * NT : NT;          // TMEM columns of one accumulator
    // Token tiles of <= 32 rows, one accumulator, single CTA (batched decode): the four K = 16 MMAs of a K block go to FOUR
    // accumulators (summed by the epilogue) instead of one.  Consecutive MMAs into the same tensor-memory columns are a
    // dependent chain, and at N <= 64 an MMA is far shorter than its latency: one chain cost 0.43 us per K block, four
    // independent ones 0.35 (bench.py --gemm-timeline; profiles/r02_batched_decode.md).
    const bool quad = CTAS == 1 && NACC == 1 && NT <= 32;
    const uint32_t need_cols = (uint32_t)(NACC * acc_cols) * (quad ? 4u : 1u);
    const uint32_t tmem_cols = need_cols <= 32 ? 32 : need_cols <= 64 ? 64 : need_cols <= 128 ? 128 : need_cols <= 256 ? 256 : 512;

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&map_w) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&map_x) : "memory");
        if (NACC == 2 || HALF) asm volatile("prefetch.tensormap [%0];" ::"l"(&map_w2) : "memory");
        for (int s = 0; s < stages; ++s) {
            mbarrier_init(&full_bar[s], 1);
            mbarrier_init(&empty_bar[s], 1);
        }
        mbarrier_init(acc_bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (CTAS == 2) cluster_sync_all();   // the barriers of both CTAs exist before either allocates, loads or commits
    if (warp == 1) {
        if (CTAS == 2) {
            asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(tmem_cols) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
        } else {
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(tmem_cols) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
        }
    }
    tcgen05_fence_before();
    __syncthreads();
    tcgen05_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    // optional timeline (hq_debug_gemm_timeline): five globaltimer stamps per CTA of the first token tile / K split
    unsigned long long *tr = (TRACE && p.trace && blockIdx.y == 0 && blockIdx.z == 0) ? p.trace + (size_t)blockIdx.x * kGemmTraceLen : nullptr;
    if (TRACE && tr && threadIdx.x == 0) tr[0] = gemm_time();   // barriers and tensor memory are up
    pdl_launch_dependents();

    if (warp == 0) {
        // ===== TMA producer =====
        if (lane == 0) {
            // EPI_STORE with p.tiles_w1 > 0: three weight matrices stacked along n in one launch (Q | K | V)
            const CUtensorMap *mw = &map_w;
            int nw = n0;
            if (MODE == EPI_STORE && p.tiles_w1 > 0 && (int)blockIdx.x >= p.tiles_w1) {
                if ((int)blockIdx.x < p.tiles_w1 + p.tiles_w2) { mw = &map_w2; nw = n0 - p.tiles_w1 * kBlockM; }
                else { mw = &map_w3; nw = n0 - (p.tiles_w1 + p.tiles_w2) * kBlockM; }
            }
            // Weights do not depend on the previous kernel: the first ring of weight tiles is requested BEFORE the
            // programmatic-dependency wait, so the launch and the first HBM round trip overlap the previous kernel's tail.
            const int pre = nkb < stages ? nkb : stages;
            // CTA pair: every load of both CTAs is credited to the leader's barrier, which expects both CTAs' stage bytes
            auto load_w = [&](int s, int kc) {
                uint8_t *st = smem + (size_t)s * stage_bytes;
                if (CTAS == 2) {
                    if (pair_rank == 0) mbarrier_expect_tx(&full_bar[s], 2 * stage_bytes);
                    tma_load_2d_pair(mw, &full_bar[s], st, kc, nw);
                    if (NACC == 2) tma_load_2d_pair(&map_w2, &full_bar[s], st + a_bytes, kc, n0);
                } else {
                    mbarrier_expect_tx(&full_bar[s], stage_bytes);
                    tma_load_2d(mw, &full_bar[s], st, kc, nw);   // HALF: a 64-row box (rows 0..63 of the A tile: gate)
                    if (NACC == 2) tma_load_2d(&map_w2, &full_bar[s], st + a_bytes, kc, n0);
                    if (HALF) tma_load_2d(&map_w2, &full_bar[s], st + a_bytes / 2, kc, n0);   // rows 64..127: up
                }
            };
            for (int i = 0; i < pre; ++i) load_w(i, (kb0 + i) * kBlockK);
            pdl_wait();   // activations come from earlier kernels
            for (int i = 0; i < nkb; ++i) {
                const int s = i % stages;
                const uint32_t ph = (i / stages) & 1;
                uint8_t *st = smem + (size_t)s * stage_bytes;
                const int kc = (kb0 + i) * kBlockK;
                if (i >= pre) {
                    mbarrier_wait(&empty_bar[s], ph ^ 1);
                    load_w(s, kc);
                }
                if (CTAS == 2) {
                    tma_load_2d_pair(&map_x, &full_bar[s], st + NACC * a_bytes, kc, (pair_rank ? p.x_lo_row : 0) + t0);
                } else {
                    tma_load_2d(&map_x, &full_bar[s], st + NACC * a_bytes, kc, t0);
                    tma_load_2d(&map_x, &full_bar[s], st + NACC * a_bytes + b_bytes, kc, p.x_lo_row + t0);
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer (one elected thread) =====
        if (lane == 0 && CTAS == 2) {
            // leader of the pair only: M = 256 (128 rows of A from each CTA), N = 2 NT (the hi plane from rank 0, the lo plane from rank 1)
            if (pair_rank == 0) {
                const uint32_t idesc = make_idesc(2 * NT, 2 * kBlockM);
                for (int i = 0; i < nkb; ++i) {
                    const int s = i % stages;
                    const uint32_t ph = (i / stages) & 1;
                    mbarrier_wait(&full_bar[s], ph);
                    tcgen05_fence_after();
                    if (TRACE && tr && (i == 0 || i == nkb - 1)) tr[i == 0 ? 1 : 2] = gemm_time();   // first / last stage landed
                    const uint32_t a_addr = smem_u32(smem + (size_t)s * stage_bytes);
                    const uint64_t da = make_smem_desc(a_addr), da2 = make_smem_desc(a_addr + a_bytes), db = make_smem_desc(a_addr + NACC * a_bytes);
#pragma unroll
                    for (int k = 0; k < kBlockK / 16; ++k) {
                        const uint32_t acc = (i > 0 || k > 0) ? 1u : 0u;
                        umma_bf16_pair(tmem_base, da + 2 * k, db + 2 * k, idesc, acc);
                        if (NACC == 2) umma_bf16_pair(tmem_base + acc_cols, da2 + 2 * k, db + 2 * k, idesc, acc);
                    }
                    tcgen05_commit_pair(&empty_bar[s]);   // frees the stage in BOTH CTAs when these MMAs retire
                }
                tcgen05_commit_pair(acc_bar);             // accumulators of both CTAs complete
            }
        } else if (lane == 0) {
            const uint32_t idesc = make_idesc(stacked ? 2 * NT : NT);
            unsigned long long t_first = 0, t_last = 0;
            for (int i = 0; i < nkb; ++i) {
                const int s = i % stages;
                const uint32_t ph = (i / stages) & 1;
                mbarrier_wait(&full_bar[s], ph);
                tcgen05_fence_after();
                if (TRACE && tr && i == 0) t_first = gemm_time();        // first stage landed
                if (TRACE && tr && i == nkb - 1) t_last = gemm_time();   // last stage landed
                const uint32_t a_addr = smem_u32(smem + (size_t)s * stage_bytes);
                const uint32_t b_addr = a_addr + NACC * a_bytes;
                const uint64_t da = make_smem_desc(a_addr), db = make_smem_desc(b_addr);
                const uint64_t da2 = make_smem_desc(a_addr + a_bytes), dbl = make_smem_desc(b_addr + b_bytes);
#pragma unroll
                for (int k = 0; k < kBlockK / 16; ++k) {
                    const uint32_t acc = (i > 0 || k > 0) ? 1u : 0u;
                    // advance 16 elements = 32 bytes inside the 128-byte swizzle row: +2 in the >>4 address field
                    if (quad) {
                        umma_bf16(tmem_base + k * acc_cols, da + 2 * k, db + 2 * k, idesc, i > 0 ? 1u : 0u);   // chain k of four
                    } else if (stacked) {
                        umma_bf16(tmem_base, da + 2 * k, db + 2 * k, idesc, acc);       // W * [x_hi ; x_lo]
                        if (NACC == 2) umma_bf16(tmem_base + acc_cols, da2 + 2 * k, db + 2 * k, idesc, acc);
                    } else {
                        umma_bf16(tmem_base, da + 2 * k, db + 2 * k, idesc, acc);       // W * x_hi
                        umma_bf16(tmem_base, da + 2 * k, dbl + 2 * k, idesc, 1u);       // W * x_lo
                        if (NACC == 2) {
                            umma_bf16(tmem_base + acc_cols, da2 + 2 * k, db + 2 * k, idesc, acc);
                            umma_bf16(tmem_base + acc_cols, da2 + 2 * k, dbl + 2 * k, idesc, 1u);
                        }
                    }
                }
                tcgen05_commit(&empty_bar[s]);   // frees the smem stage when these MMAs retire
            }
            tcgen05_commit(acc_bar);             // accumulator complete
            if (TRACE && tr) { tr[1] = t_first; tr[2] = t_last; }
        }
    } else {
        // ===== epilogue: warp w owns TMEM lanes 32*(w%4) .. +31 =====
        const int q = warp & 3;
        const int n = n0 + 32 * (HALF ? (q & 1) : q) + lane;
        pdl_wait();   // the output buffer (residual, zeroed split-K target) belongs to earlier kernels until now
        mbarrier_wait(acc_bar, 0);
        tcgen05_fence_after();
        if (TRACE && tr && warp == 2 && lane == 0) tr[3] = gemm_time();   // accumulator complete
        if (TRACE) __syncwarp();   // the tensor-memory loads below are warp-aligned instructions
        const uint32_t lane_addr = tmem_base + ((uint32_t)(32 * q) << 16);
        const bool row_ok = n < p.n_rows;
        const bool pairable = (p.n_rows & 1) == 0 && (p.ld_out & 1) == 0;   // bf16 outputs as 32-bit pairs
        for (int c = 0; c < NT; c += 32) {
            const int nvalid = min(p.T - (t0 + c), NT - c);   // tokens of this chunk that exist and belong to this tile (>= 32: all)
            uint32_t v[32];
            tmem_ld32(lane_addr + c, v);
            if (quad) {
                // four accumulators of 2 NT columns ([hi | lo] each) = NT / 4 loads of 32 columns, added column-wise; then the
                // 32 columns fold to NT tokens (8: four groups of 8; 16: two groups of 16; 32: the loads already alternate
                // hi and lo of the same tokens)
                const int n_loads = NT >> 2;
#pragma unroll
                for (int ql = 1; ql < 8; ++ql) {
                    if (ql < n_loads) {   // warp-uniform
                        uint32_t w[32];
                        tmem_ld32(lane_addr + 32 * ql, w);
#pragma unroll
                        for (int j = 0; j < 32; ++j) v[j] = __float_as_uint(__uint_as_float(v[j]) + __uint_as_float(w[j]));
                    }
                }
                if (NT == 8) {
#pragma unroll
                    for (int j = 0; j < 8; ++j)
                        v[j] = __float_as_uint((__uint_as_float(v[j]) + __uint_as_float(v[8 + j])) + (__uint_as_float(v[16 + j]) + __uint_as_float(v[24 + j])));
                } else if (NT == 16) {
#pragma unroll
                    for (int j = 0; j < 16; ++j) v[j] = __float_as_uint(__uint_as_float(v[j]) + __uint_as_float(v[16 + j]));
                }
            } else if (stacked) {
                uint32_t w[32];
                tmem_ld32(lane_addr + NT + c, w);
#pragma unroll
                for (int j = 0; j < 32; ++j) v[j] = __float_as_uint(__uint_as_float(v[j]) + __uint_as_float(w[j]));
            }
            if (HALF || MODE == EPI_SWIGLU) {
                float a[32];
                if (HALF) {
                    // lanes 64..127 of the accumulator (warps q = 2, 3) hold the up projection of the features whose gate
                    // projection is in lanes 0..63 (q = 0, 1): hand it over through stage 0 of the ring (every load has been
                    // consumed and every MMA has retired once acc_bar completes), [token][feature] so that lanes do not conflict
                    float *xch = reinterpret_cast<float *>(smem);
                    if (q >= 2) {
#pragma unroll
                        for (int j = 0; j < 32; ++j) xch[j * 64 + 32 * (q - 2) + lane] = __uint_as_float(v[j]);
                    }
                    asm volatile("bar.sync 1, 128;" ::: "memory");
                    if (q < 2) {
                        float u[32];
#pragma unroll
                        for (int j = 0; j < 32; ++j) u[j] = xch[j * 64 + 32 * q + lane];
                        swiglu32(v, u, a);
                    }
                } else {
                    uint32_t u[32];
                    tmem_ld32(lane_addr + acc_cols + c, u);
                    if (stacked) {
                        uint32_t w[32];
                        tmem_ld32(lane_addr + acc_cols + NT + c, w);
#pragma unroll
                        for (int j = 0; j < 32; ++j) u[j] = __float_as_uint(__uint_as_float(u[j]) + __uint_as_float(w[j]));
                    }
                    float uf[32];
#pragma unroll
                    for (int j = 0; j < 32; ++j) uf[j] = __uint_as_float(u[j]);
                    swiglu32(v, uf, a);
                }
                if ((!HALF || q < 2) && nvalid > 0) {   // warp-uniform
                    act_t *out = p.out_act + (size_t)(t0 + c) * p.ld_out;
                    if (pairable) store_act_pairs(a, out, p.out_lo_offset, (size_t)p.ld_out, n, row_ok, nvalid, lane);
                    else store_act_scalar(a, out + n, p.out_lo_offset, (size_t)p.ld_out, row_ok, nvalid);
                }
                if (HALF && c + 32 < NT) asm volatile("bar.sync 1, 128;" ::: "memory");
            } else if (row_ok && nvalid > 0) {
                float *dst = p.out_f32 + (size_t)blockIdx.z * p.split_stride + (size_t)(t0 + c) * p.ld_out + n;
                const size_t ld = (size_t)p.ld_out;
                if (p.atomic) {
#pragma unroll
                    for (int j = 0; j < 32; ++j)
                        if (j < nvalid) atomicAdd(dst + j * ld, __uint_as_float(v[j]));
                } else if (MODE == EPI_RESID) {
#pragma unroll
                    for (int j = 0; j < 32; ++j)
                        if (j < nvalid) dst[j * ld] = __ldcg(dst + j * ld) + __uint_as_float(v[j]);
                } else if (nvalid >= 32) {
#pragma unroll
                    for (int j = 0; j < 32; ++j) dst[j * ld] = __uint_as_float(v[j]);
                } else {
#pragma unroll
                    for (int j = 0; j < 32; ++j)
                        if (j < nvalid) dst[j * ld] = __uint_as_float(v[j]);
                }
            }
        }
        tcgen05_fence_before();
        if (TRACE && tr && warp == 2 && lane == 0) tr[4] = gemm_time();   // this warp's share of the epilogue issued
    }
    __syncthreads();
    if (CTAS == 2) cluster_sync_all();   // neither CTA frees tensor memory or exits while the pair's MMAs / loads may still touch it
    if (warp == 1) {
        tcgen05_fence_after();
        if (CTAS == 2) asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(tmem_cols) : "memory");
        else asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(tmem_cols) : "memory");
    }
}

// ---- host side -----------------------------------------------------------------------------------------
typedef CUresult (*PFN_encodeTiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static PFN_encodeTiled get_encode() {
    static PFN_encodeTiled fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (PFN_encodeTiled)p;
    }
    return fn;
}

// 2-D tensor of 16-bit elements [rows][cols] row-major, box = box_rows x 64 columns, 128-byte swizzle
// (weights, and the stacked hi/lo planes of an activation buffer).
bool make_tensor_map_16b(TensorMap *out, const void *base, uint64_t rows, uint64_t cols, uint32_t box_rows) {
    PFN_encodeTiled enc = get_encode();
    if (!enc) return false;
    static_assert(sizeof(TensorMap) == sizeof(CUtensorMap), "TensorMap must mirror CUtensorMap");
    cuuint64_t dims[2] = {cols, rows};
    cuuint64_t strides[1] = {cols * 2};
    cuuint32_t box[2] = {(cuuint32_t)kBlockK, box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(reinterpret_cast<CUtensorMap *>(out), CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void *>(base),
                     dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                     CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

static const int kSmemBudget = 200 * 1024;

template <int MODE>
static cudaError_t launch_mode(const LaunchCtx &c, const TensorMap &w, const TensorMap &w2, const TensorMap &w3,
                               const TensorMap &x, GemmParams p, int n_tiles, int t_tiles, int splits) {
    const int nacc = (MODE == EPI_SWIGLU) ? 2 : 1;
    // CTA pairs (cta_group::2, M = 256) for prefill-sized passes: the activation tile is shared by two weight tiles, each CTA
    // loads one of its two planes (a third less operand traffic from L2, the bound of these GEMMs).  Needs the stacked-plane
    // form (token tile <= 128); batched-decode steps (<= 32 rows) keep single CTAs.
    const bool pair = MODE != EPI_SWIGLU64 && p.NT >= 32 && p.NT <= 128 && p.T > 32;
    const int stage_bytes = nacc * kBlockM * kBlockK * 2 + (pair ? 1 : 2) * p.NT * kBlockK * 2;
    // Decode GEMMs that run as many waves of CTAs (the LM head: 1002 tiles over 148 SMs) take half-size rings: two CTAs then
    // share an SM and one's set-up and first loads run under the other's main loop (B = 8 step 960 -> 946 us, B = 32 x 512
    // 1,345 -> 1,307).  The one-wave GEMMs of a layer do NOT: there the co-resident CTAs belong to the NEXT kernel and their
    // prefetch only competes (profiles/r02_batched_decode.md, item 13).
    const bool two_per_sm = !pair && p.T <= 32 && n_tiles * t_tiles * splits > 2 * c.n_sms;
    int stages = (two_per_sm ? 108 * 1024 : kSmemBudget) / stage_bytes;
    if (stages > 8) stages = 8;
    if (stages > p.k_blocks_per_split) stages = p.k_blocks_per_split < 2 ? 2 : p.k_blocks_per_split;
    p.stages = stages;
    const size_t smem = (size_t)stages * stage_bytes + 1024 + (2 * stages + 1) * 8 + 16;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(pair ? (n_tiles + 1) / 2 * 2 : n_tiles, t_tiles, splits);   // a pair's odd tile past the end loads zeros (TMA) and stores nothing
    cfg.blockDim = dim3(kGemmThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = c.stream;
    cudaLaunchAttribute attr[2];
    int na = 0;
    if (c.pdl) {
        attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    if (pair) {
        attr[na].id = cudaLaunchAttributeClusterDimension;
        attr[na].val.clusterDim.x = 2;
        attr[na].val.clusterDim.y = 1;
        attr[na].val.clusterDim.z = 1;
        ++na;
    }
    cfg.attrs = attr;
    cfg.numAttrs = na;
    typedef void (*kernel_t)(const CUtensorMap, const CUtensorMap, const CUtensorMap, const CUtensorMap, const GemmParams);
    kernel_t k = p.trace ? gemm_tc_kernel<MODE, 1, true> : gemm_tc_kernel<MODE, 1, false>;
    if constexpr (MODE != EPI_SWIGLU64)
        if (pair) k = p.trace ? gemm_tc_kernel<MODE, 2, true> : gemm_tc_kernel<MODE, 2, false>;
    if (p.trace) {   // diagnostics only: opt in here instead of in gemm_prepare
        cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
        if (e != cudaSuccess) return e;
    }
    return cudaLaunchKernelEx(&cfg, k, *reinterpret_cast<const CUtensorMap *>(&w), *reinterpret_cast<const CUtensorMap *>(&w2),
                              *reinterpret_cast<const CUtensorMap *>(&w3), *reinterpret_cast<const CUtensorMap *>(&x), p);
}

// token tiles: 32, 64, 128, 256, and 8 / 16 for passes of <= 16 rows (not for the two-accumulator SwiGLU form, whose second
// accumulator the epilogue reads with a 32-column load of its own)
static bool gemm_token_tile_ok(int NT, int mode) {
    if (NT == 8 || NT == 16) return mode != EPI_SWIGLU;
    return NT % 32 == 0 && NT >= 32 && NT <= 256;
}

// n_rows: weight rows (output features; for EPI_SWIGLU the ffn size), K: reduction size (multiple of 64),
// T: valid tokens, NT: token tile (32/64/128/256).  splits > 1 requires atomic accumulation (EPI_STORE into a
// zeroed buffer, EPI_RESID always legal).
cudaError_t launch_gemm(const LaunchCtx &c, GemmEpilogue mode, const TensorMap &w, const TensorMap *w2,
                        const TensorMap &x, int x_lo_row, int n_rows, int K, int T, int NT, int splits, float *out_f32,
                        act_t *out_act, size_t out_lo_offset, int ld_out, size_t split_stride, unsigned long long *trace) {
    // K need not be a multiple of 64: TMA zero-fills the out-of-range tail of the last K block
    if (K % 8 != 0 || !gemm_token_tile_ok(NT, mode) || T <= 0) return cudaErrorInvalidValue;
    const int kblocks = (K + kBlockK - 1) / kBlockK;
    if (splits < 1) splits = 1;
    if (splits > kblocks) splits = kblocks;
    GemmParams p = {};
    p.K = K; p.n_rows = n_rows; p.T = T; p.NT = NT; p.k_blocks = kblocks;
    p.k_blocks_per_split = (kblocks + splits - 1) / splits;
    splits = (kblocks + p.k_blocks_per_split - 1) / p.k_blocks_per_split;
    p.out_f32 = out_f32; p.out_act = out_act; p.out_lo_offset = out_lo_offset; p.x_lo_row = x_lo_row; p.ld_out = ld_out;
    p.split_stride = mode == EPI_STORE ? split_stride : 0;
    p.trace = trace;
    p.atomic = (splits > 1 && p.split_stride == 0) ? 1 : 0;
    const int n_tiles = (n_rows + kBlockM - 1) / kBlockM, t_tiles = (T + NT - 1) / NT;
    switch (mode) {
        case EPI_STORE: return launch_mode<EPI_STORE>(c, w, w, w, x, p, n_tiles, t_tiles, splits);
        case EPI_RESID: return launch_mode<EPI_RESID>(c, w, w, w, x, p, n_tiles, t_tiles, splits);
        case EPI_SWIGLU:
            if (splits != 1 || !w2) return cudaErrorInvalidValue;
            return launch_mode<EPI_SWIGLU>(c, w, *w2, w, x, p, n_tiles, t_tiles, 1);
        case EPI_SWIGLU64:   // w, w2: tensor maps with 64-ROW boxes
            if (splits != 1 || !w2 || n_rows % (kBlockM / 2) != 0) return cudaErrorInvalidValue;
            return launch_mode<EPI_SWIGLU64>(c, w, *w2, w, x, p, n_rows / (kBlockM / 2), t_tiles, 1);
    }
    return cudaErrorInvalidValue;
}

// Q, K and V projections in ONE launch: three weight matrices with n1, n2, n3 rows (multiples of 128) stacked along
// the output dimension of out_f32 [T][n1 + n2 + n3].
cudaError_t launch_gemm_qkv(const LaunchCtx &c, const TensorMap &wq, const TensorMap &wk, const TensorMap &wv, const TensorMap &x,
                            int x_lo_row, int n1, int n2, int n3, int K, int T, int NT, int splits, float *out_f32, int ld_out,
                            size_t split_stride) {
    if (K % 8 != 0 || !gemm_token_tile_ok(NT, EPI_STORE) || T <= 0 || n1 % kBlockM || n2 % kBlockM || n3 % kBlockM)
        return cudaErrorInvalidValue;
    const int kblocks = (K + kBlockK - 1) / kBlockK;
    if (splits < 1) splits = 1;
    if (splits > kblocks) splits = kblocks;
    GemmParams p = {};
    p.K = K; p.n_rows = n1 + n2 + n3; p.T = T; p.NT = NT; p.k_blocks = kblocks;
    p.k_blocks_per_split = (kblocks + splits - 1) / splits;
    splits = (kblocks + p.k_blocks_per_split - 1) / p.k_blocks_per_split;
    p.out_f32 = out_f32; p.x_lo_row = x_lo_row; p.ld_out = ld_out; p.split_stride = split_stride;
    p.atomic = (splits > 1 && split_stride == 0) ? 1 : 0;
    p.tiles_w1 = n1 / kBlockM; p.tiles_w2 = n2 / kBlockM;
    return launch_mode<EPI_STORE>(c, wq, wk, wv, x, p, p.n_rows / kBlockM, (T + NT - 1) / NT, splits);
}

// Shared-memory opt-in of every instantiation on the CURRENT device (the attribute is per device: hq_model_create and
// hq_debug_gemm call this, not a process-wide once-flag).
cudaError_t gemm_prepare() {
    cudaError_t e = cudaFuncSetAttribute(gemm_tc_kernel<EPI_STORE, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(gemm_tc_kernel<EPI_RESID, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(gemm_tc_kernel<EPI_SWIGLU, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(gemm_tc_kernel<EPI_SWIGLU64, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(gemm_tc_kernel<EPI_STORE, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(gemm_tc_kernel<EPI_RESID, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(gemm_tc_kernel<EPI_SWIGLU, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    return e;
}

}  // namespace hq
