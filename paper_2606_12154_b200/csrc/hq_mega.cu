// hq_mega.cu — persistent batch-1 decode: SURVEY.md §8(a) rows A1-A9 for n_steps tokens in ONE launch.
//
// Why: one token is a chain of 81 HBM-bound matrix-vector products over 2.47 GB of bf16 weights.  With one
// kernel per product the three small products of every layer (QKV, attention, O) cost more in kernel-boundary
// latency than in DRAM time (profiles/r01_decode_launches_v1.md: 53 % of the copy peak).  Here the weight
// stream never stops:
//   * grid = one CTA per SM, 9 warps.  Warp 8 is the PRODUCER: one elected thread walks the static schedule
//     (layer, phase, this CTA's rows) and streams every weight row with cp.async.bulk (TMA bulk copy,
//     mbarrier complete_tx) into a ring of kMkStages x 64 KB shared-memory stages.  Weights are immutable, so
//     the producer runs ahead of the phase barriers: while the consumers wait for the other SMs, do the
//     attention, or reduce, the next phases' rows are already landing.
//   * warps 0-7 are CONSUMERS and never synchronise with one another inside a weight phase.  A stage holds
//     8/S "units" (a unit = two rows: RoPE pair (i, i+32) / gate+up pair / two adjacent rows); a row is cut
//     into S slices of <= 2048 elements and warp w owns slice w % S of unit w / S, so the slice of the
//     (normalised) input vector it needs stays in 64 registers for the whole phase.  Per stage and warp: two
//     conflict-free 16-byte shared loads per chunk, fp32 FMA, one 6-shuffle reduction for both rows, one
//     mbarrier arrive, and the fused epilogue (RoPE + KV append, SwiGLU, logits + packed argmax) from lane 0.
//     Only the residual projections (O, down) park their per-slice partials in shared memory and finish after
//     one CTA barrier at the end of the phase.
//   * phases are separated by a grid barrier (red.release + ld.acquire poll on a global counter): per layer
//     QKV | attention | O | gate/up | down, then the LM head.  The token and the position stay on the device;
//     the kernel loops over n_steps tokens (hq_decode_run) so there is no launch gap between tokens either.
//   * attention: work item = (KV head, context split); warp = (query head of the group, sub-split); LANE =
//     POSITION: every lane runs its own online softmax over its positions (K/V rows are one 128-byte line each,
//     read with 256-bit loads), then the 32 lane states are merged with a transposed butterfly, the sub-splits
//     through shared memory, and the splits by the last CTA of the KV head (ticket), so the O phase reads a
//     plain vector.
#include "hq_common.cuh"
#include "hq_internal.h"

namespace hq {

constexpr int kMkConsumerWarps = 8;
constexpr int kMkConsumers = 32 * kMkConsumerWarps;
constexpr int kMkThreads = kMkConsumers + 32;
constexpr int kMkPartRows = 64;
constexpr int kMkStagedK = 8 * kMkConsumers;      // 2048: one 8-element chunk per consumer thread                   // residual rows of one CTA in one phase (2 * units)
constexpr long long kSpinCycles = 6000000000ll;   // ~3 s of SM clocks: a lost arrival traps instead of hanging the GPU

enum { PH_QKV = 0, PH_O = 1, PH_GATEUP = 2, PH_DOWN = 3, PH_HEAD = 4 };

// ---- small PTX wrappers -------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t mk_smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mk_mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mk_smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mk_mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mk_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mk_mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mk_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mk_mbar_try_wait(uint64_t *bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(mk_smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mk_fail(int *err, int code) {
    atomicExch(err, code);
    __threadfence_system();
    __trap();
}
__device__ __forceinline__ void mk_mbar_wait(uint64_t *bar, uint32_t parity, int *err) {
    if (mk_mbar_try_wait(bar, parity)) return;
    const long long t0 = clock64();
    unsigned spins = 0;
    while (!mk_mbar_try_wait(bar, parity))
        if ((++spins & 1023u) == 0 && clock64() - t0 > kSpinCycles) mk_fail(err, 1);
}
__device__ __forceinline__ void mk_bulk_g2s(void *smem_dst, const void *gmem_src, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     mk_smem_u32(smem_dst)),
                 "l"(gmem_src), "r"(bytes), "r"(mk_smem_u32(bar))
                 : "memory");
}
// weights are read once per token: mark their L2 lines evict-first so that the activations, the attention partials and
// the KV cache (re-read every token) stay resident in the 126 MB L2
__device__ __forceinline__ uint64_t mk_policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void mk_bulk_g2s_hint(void *smem_dst, const void *gmem_src, uint32_t bytes, uint64_t *bar, uint64_t pol) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
                     mk_smem_u32(smem_dst)),
                 "l"(gmem_src), "r"(bytes), "r"(mk_smem_u32(bar)), "l"(pol)
                 : "memory");
}
// fire-and-forget HBM -> L2 prefetch of a weight row (no completion tracking: the later bulk copy just hits L2)
__device__ __forceinline__ void mk_bulk_prefetch_l2(const void *gmem_src, uint32_t bytes, uint64_t pol) {
    asm volatile("cp.async.bulk.prefetch.L2.global.L2::cache_hint [%0], %1, %2;" ::"l"(gmem_src), "r"(bytes), "l"(pol) : "memory");
}
__device__ __forceinline__ void consumer_sync() { asm volatile("bar.sync 1, %0;" ::"n"(kMkConsumers) : "memory"); }
__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned *p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_add(unsigned *p, unsigned v) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned long long mk_globaltimer() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
// one 128-byte K or V row (64 fp16) of a cache position.  Plain (coherent-after-acquire) loads: the row of the
// current position was written in this launch, before the grid barrier that precedes the attention phase.
struct KvRow { uint4 v[8]; };
__device__ __forceinline__ void ld_kv_row(KvRow &r, const kv_t *p) {
#pragma unroll
    for (int j = 0; j < 4; ++j)
        asm volatile("ld.global.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                     : "=r"(r.v[2 * j].x), "=r"(r.v[2 * j].y), "=r"(r.v[2 * j].z), "=r"(r.v[2 * j].w),
                       "=r"(r.v[2 * j + 1].x), "=r"(r.v[2 * j + 1].y), "=r"(r.v[2 * j + 1].z), "=r"(r.v[2 * j + 1].w)
                     : "l"(p + 16 * j)
                     : "memory");
}
__device__ __forceinline__ float2 h2f(uint32_t u) { return __half22float2(*reinterpret_cast<const __half2 *>(&u)); }

// ---- static schedule shared by producer and consumers -----------------------------------------------------
struct PhaseGeom {
    int K, row_bytes;
    int S, log2S;      // K-slices per row (1, 2, 4 or 8): S warps share a unit
    int cps;           // 16-byte chunks per slice (<= 256)
    int ups;           // units per stage = 8 / S; a stage holds 2*ups rows
    int u0, u1;        // this CTA's units [u0, u1)
    int n_stages;
};

__device__ __forceinline__ int phase_units(const MegaParams &p, int ph) {
    switch (ph) {
        case PH_QKV: return (p.n_heads + 2 * p.n_kv_heads) * 32;
        case PH_O: return p.hidden / 2;
        case PH_GATEUP: return p.ffn;
        case PH_DOWN: return p.hidden / 2;
        default: return p.vocab / 2;
    }
}
__device__ __forceinline__ int phase_k(const MegaParams &p, int ph) {
    switch (ph) {
        case PH_O: return p.n_heads * kHeadDim;
        case PH_DOWN: return p.ffn;
        default: return p.hidden;
    }
}
__device__ __forceinline__ PhaseGeom phase_geom(const MegaParams &p, int ph) {
    PhaseGeom g;
    g.K = phase_k(p, ph);
    g.row_bytes = g.K * 2;
    const int chunks = g.K >> 3;
    g.S = 1;
    g.log2S = 0;
    while ((chunks + g.S - 1) / g.S > kMkSliceChunks) { g.S <<= 1; ++g.log2S; }
    g.cps = (chunks + g.S - 1) / g.S;
    g.ups = kMkConsumerWarps >> g.log2S;
    const int n = phase_units(p, ph), per = n / gridDim.x, rem = n % gridDim.x, b = blockIdx.x;
    g.u0 = b * per + min(b, rem);
    g.u1 = g.u0 + per + (b < rem ? 1 : 0);
    g.n_stages = (g.u1 - g.u0 + g.ups - 1) / g.ups;
    return g;
}
// the two weight rows of unit u
__device__ __forceinline__ void unit_row_ptrs(const MegaParams &p, const LayerW &w, int ph, int K, int u, const bf16 *&ra,
                                              const bf16 *&rb) {
    if (ph == PH_QKV) {
        const int hh = u >> 5, i = u & 31;
        const bf16 *base;
        int h;
        if (hh < p.n_heads) { base = w.wq; h = hh; }
        else if (hh < p.n_heads + p.n_kv_heads) { base = w.wk; h = hh - p.n_heads; }
        else { base = w.wv; h = hh - p.n_heads - p.n_kv_heads; }
        ra = base + (size_t)(h * kHeadDim + i) * K;
        rb = ra + (size_t)32 * K;
    } else if (ph == PH_GATEUP) {
        ra = w.w_gate + (size_t)u * K;
        rb = w.w_up + (size_t)u * K;
    } else {
        const bf16 *base = ph == PH_O ? w.wo : (ph == PH_DOWN ? w.w_down : p.lm_head);
        ra = base + (size_t)(2 * u) * K;
        rb = ra + K;
    }
}

struct MkShared {
    uint64_t full[kMkStages], empty[kMkStages];
    alignas(16) float xs[kMkStagedK];            // phase input staged once per CTA (phases with K <= kMkStagedK)
    float part[kMkPartRows][kMkConsumerWarps];   // residual phases: [row of this CTA][slice] partial sums
    float2 rope[32];
    alignas(16) float q[kMkConsumerWarps][kHeadDim];   // per warp: pre-scaled query of its head
    float mrg[kMkConsumerWarps][kHeadDim + 2];   // attention: sub-split states (o[64], m, l)
    float red[kMkConsumerWarps];                 // RMSNorm: per-warp sum of squares
    unsigned long long wbest[kMkConsumerWarps];  // LM head: per-warp packed argmax
};

// ---- producer ----------------------------------------------------------------------------------------------
// Position in this CTA's static stage schedule: (step, phase index, stage of the phase).
struct MkCursor {
    int step, pi, s, ph, layer;
    PhaseGeom geo;
    bool done;
};
__device__ __forceinline__ void cursor_load_phase(const MegaParams &p, MkCursor &c) {
    const int n_ph = p.n_layers * 4 + (p.with_head ? 1 : 0);
    for (;;) {   // skip phases in which this CTA owns no unit
        if (c.pi == n_ph) { c.pi = 0; ++c.step; }
        if (c.step >= p.n_steps) { c.done = true; return; }
        c.layer = c.pi >> 2;
        c.ph = c.layer < p.n_layers ? (c.pi & 3) : PH_HEAD;
        c.geo = phase_geom(p, c.ph);
        if (c.geo.n_stages > 0) return;
        ++c.pi;
    }
}
__device__ __forceinline__ void cursor_init(const MegaParams &p, MkCursor &c) {
    c.step = 0; c.pi = 0; c.s = 0; c.done = false;
    cursor_load_phase(p, c);
}
__device__ __forceinline__ void cursor_next(const MegaParams &p, MkCursor &c) {
    if (++c.s == c.geo.n_stages) { c.s = 0; ++c.pi; cursor_load_phase(p, c); }
}

// One elected thread.  Two cursors walk the same schedule: `ld` fills the shared-memory ring (TMA bulk copies, mbarrier
// complete_tx), `pf` runs p.prefetch_stages stages ahead of it and only pulls the rows HBM -> L2.  The ring alone holds
// ~4 us of streaming; the dependent chain down -> QKV -> attention -> O of a layer is longer than that, so without the
// L2 look-ahead the HBM pipe would idle while the consumers sit in grid barriers.
__device__ void mk_producer(const MegaParams &p, uint8_t *ring, MkShared &sh) {
    const uint64_t pol = mk_policy_evict_first();
    MkCursor ld, pf;
    cursor_init(p, ld);
    pf = ld;
    int ahead = 0;   // stages pf is ahead of ld
    unsigned g = 0;  // stages produced so far
    while (!ld.done) {
        while (!pf.done && ahead < p.prefetch_stages) {
            if (ahead > 0) {   // distance 0 would duplicate the bulk copy issued right below
                const LayerW &w = p.layers[pf.layer < p.n_layers ? pf.layer : 0];
                const int ub = pf.geo.u0 + pf.s * pf.geo.ups;
                const int nu = min(pf.geo.ups, pf.geo.u1 - ub);
                for (int j = 0; j < nu; ++j) {
                    const bf16 *ra, *rb;
                    unit_row_ptrs(p, w, pf.ph, pf.geo.K, ub + j, ra, rb);
                    mk_bulk_prefetch_l2(ra, pf.geo.row_bytes, pol);
                    mk_bulk_prefetch_l2(rb, pf.geo.row_bytes, pol);
                }
            }
            cursor_next(p, pf);
            ++ahead;
        }
        const int slot = g % kMkStages;
        const uint32_t par = (g / kMkStages) & 1;
        mk_mbar_wait(&sh.empty[slot], par ^ 1, p.err);
        const LayerW &w = p.layers[ld.layer < p.n_layers ? ld.layer : 0];
        const int ub = ld.geo.u0 + ld.s * ld.geo.ups;
        const int nu = min(ld.geo.ups, ld.geo.u1 - ub);
        mk_mbar_expect_tx(&sh.full[slot], (uint32_t)(2 * nu * ld.geo.row_bytes));
        uint8_t *dst = ring + (size_t)slot * kMkStageBytes;
        for (int j = 0; j < nu; ++j) {
            const bf16 *ra, *rb;
            unit_row_ptrs(p, w, ld.ph, ld.geo.K, ub + j, ra, rb);
            mk_bulk_g2s_hint(dst + (size_t)(2 * j) * ld.geo.row_bytes, ra, ld.geo.row_bytes, &sh.full[slot], pol);
            mk_bulk_g2s_hint(dst + (size_t)(2 * j + 1) * ld.geo.row_bytes, rb, ld.geo.row_bytes, &sh.full[slot], pol);
        }
        cursor_next(p, ld);
        ++g;
        if (ahead > 0) --ahead;
    }
}

// ---- consumer state ------------------------------------------------------------------------------------------
struct MkCtx {
    unsigned g;          // stages consumed so far
    unsigned bar_target; // thread 0: arrivals expected at the next grid barrier
    int pos, tok;
    int layer;
    int ti;              // trace cursor (thread 0)
    unsigned long long best;
};

// optional timeline (hq_debug_trace): every CTA's thread 0 stamps the global timer at each phase boundary
__device__ __forceinline__ void mk_trace(const MegaParams &p, MkCtx &c) {
    if (p.trace && threadIdx.x == 0) {
        if (c.ti < p.trace_cap) p.trace[(size_t)blockIdx.x * p.trace_cap + c.ti] = mk_globaltimer();
        ++c.ti;
    }
}

// Grid barrier.  bar.sync orders every consumer's global stores of the phase before thread 0's gpu-scope
// release (cumulativity); the acquire poll + bar.sync orders the other CTAs' stores before every consumer's
// later loads.
__device__ __forceinline__ void grid_barrier(const MegaParams &p, MkCtx &c) {
    consumer_sync();
    if (threadIdx.x == 0) {
        c.bar_target += gridDim.x;
        red_release_add(p.bar, 1u);
        mk_trace(p, c);
        const long long t0 = clock64();
        unsigned spins = 0;
        while ((int)(ld_acquire_u32(p.bar) - c.bar_target) < 0)
            if ((++spins & 1023u) == 0 && clock64() - t0 > kSpinCycles) mk_fail(p.err, 2);
    }
    consumer_sync();
    mk_trace(p, c);
}

// attention split policy (device only; a function of the context length and the grid): one 32-position
// iteration per warp while the grid has CTAs to spare, then longer splits.  n_kv_heads * splits <= gridDim.x, so
// every CTA owns at most one (KV head, split) item.
__device__ __forceinline__ int mk_num_splits(const MegaParams &p, int n_ctx, int nsub) {
    int ns_max = (int)gridDim.x / p.n_kv_heads;
    ns_max = ns_max < 1 ? 1 : (ns_max > kMkMaxSplits ? kMkMaxSplits : ns_max);
    const int per = 32 * nsub;
    const int want = (n_ctx + per - 1) / per;
    return want < ns_max ? want : ns_max;
}

// Phase input, K <= kMkStagedK: the CTA reads the vector from L2 ONCE (thread t owns elements [8t, 8t+8)), applies the
// fused prologue, and leaves it in shared memory for its 8 warps.  (Every warp fetching its own copy made all 1184
// warps of the chip hit the same 64 L2 lines at once: 4-5 us per phase, profiles/r01_mega_timeline.md.)
//   QKV, gate/up, LM head: A2 RMSNorm (sum of squares reduced across the CTA, deterministic), gain multiply
//   O:                     A5 merge of the split-KV partials (m, l, o) written by the attention phase
//   down (small models):   plain copy
__device__ __forceinline__ void stage_input(const MegaParams &p, const MkCtx &c, int ph, int K, MkShared &sh) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const bool has = tid * 8 < K;
    float v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = 0.f;
    if (ph == PH_O) {
        if (has) {
            const int G = p.n_heads / p.n_kv_heads;
            const int ns = mk_num_splits(p, c.pos + 1, kMkConsumerWarps / G);
            const int h = tid >> 3, d0 = (tid & 7) * 8;
            const float2 *ml = p.part_ml + (size_t)h * kMkMaxSplits;
            const float *po = p.part_o + (size_t)h * kMkMaxSplits * kHeadDim + d0;
            float Mx = -INFINITY;
            for (int s = 0; s < ns; ++s) Mx = fmaxf(Mx, __ldcg(&ml[s]).x);
            float den = 0.f;
            for (int s = 0; s < ns; ++s) {
                const float2 m = __ldcg(&ml[s]);
                const float wgt = (m.x == -INFINITY) ? 0.f : __expf(m.x - Mx);
                const float4 a = ld_act4(po + (size_t)s * kHeadDim), b = ld_act4(po + (size_t)s * kHeadDim + 4);
                den = fmaf(wgt, m.y, den);
                v[0] = fmaf(wgt, a.x, v[0]); v[1] = fmaf(wgt, a.y, v[1]); v[2] = fmaf(wgt, a.z, v[2]); v[3] = fmaf(wgt, a.w, v[3]);
                v[4] = fmaf(wgt, b.x, v[4]); v[5] = fmaf(wgt, b.y, v[5]); v[6] = fmaf(wgt, b.z, v[6]); v[7] = fmaf(wgt, b.w, v[7]);
            }
            const float inv = 1.0f / den;
#pragma unroll
            for (int i = 0; i < 8; ++i) v[i] *= inv;
        }
    } else if (ph == PH_DOWN) {
        if (has) {
            const float4 a = ld_act4(p.act + (size_t)tid * 8), b = ld_act4(p.act + (size_t)tid * 8 + 4);
            v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
        }
    } else {
        const bf16 *gain = ph == PH_QKV ? p.layers[c.layer].attn_norm : (ph == PH_GATEUP ? p.layers[c.layer].ffn_norm : p.final_norm);
        uint4 gq = make_uint4(0, 0, 0, 0);
        if (has) {
            gq = __ldg(reinterpret_cast<const uint4 *>(gain) + tid);
            if (ph == PH_QKV && c.layer == 0) {   // A1: the residual stream starts as the embedding row
                const uint4 e = __ldg(reinterpret_cast<const uint4 *>(p.emb + (size_t)c.tok * p.hidden) + tid);
                v[0] = bf16lo(e.x); v[1] = bf16hi(e.x); v[2] = bf16lo(e.y); v[3] = bf16hi(e.y);
                v[4] = bf16lo(e.z); v[5] = bf16hi(e.z); v[6] = bf16lo(e.w); v[7] = bf16hi(e.w);
            } else {
                const float4 a = ld_act4(p.x + (size_t)tid * 8), b = ld_act4(p.x + (size_t)tid * 8 + 4);
                v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
            }
        }
        float ss = 0.f;
#pragma unroll
        for (int i = 0; i < 8; ++i) ss = fmaf(v[i], v[i], ss);
        ss = warp_sum(ss);
        if (lane == 0) sh.red[warp] = ss;
        consumer_sync();
        float tot = 0.f;
#pragma unroll
        for (int k = 0; k < kMkConsumerWarps; ++k) tot += sh.red[k];
        const float inv = 1.0f / sqrtf(tot / (float)K + p.eps);
        const uint32_t gg[4] = {gq.x, gq.y, gq.z, gq.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            v[2 * i] *= inv * bf16lo(gg[i]);
            v[2 * i + 1] *= inv * bf16hi(gg[i]);
        }
    }
    if (has) {
        float4 *dst = reinterpret_cast<float4 *>(sh.xs + tid * 8);
        dst[0] = make_float4(v[0], v[1], v[2], v[3]);
        dst[1] = make_float4(v[4], v[5], v[6], v[7]);
    }
    consumer_sync();
}

// Phase input slice -> registers.  Lane owns chunks (8 elements) c0 + j*32 + lane, j < NCH, of the row.
template <int NCH>
__device__ __forceinline__ void load_x_staged(const MkShared &sh, int my_chunks, float (&xr)[NCH][8]) {
    const int lane = threadIdx.x & 31;
    const float4 *xs4 = reinterpret_cast<const float4 *>(sh.xs);
#pragma unroll
    for (int j = 0; j < NCH; ++j) {
        const int ch = j * 32 + lane;
        if (ch < my_chunks) {
            const float4 a = xs4[2 * ch], b = xs4[2 * ch + 1];
            xr[j][0] = a.x; xr[j][1] = a.y; xr[j][2] = a.z; xr[j][3] = a.w;
            xr[j][4] = b.x; xr[j][5] = b.y; xr[j][6] = b.z; xr[j][7] = b.w;
        } else {
#pragma unroll
            for (int i = 0; i < 8; ++i) xr[j][i] = 0.f;
        }
    }
}
// K > kMkStagedK (the down projection of the 1B model, K = 8192): every warp reads its own slice from L2
template <int NCH>
__device__ __forceinline__ void load_x_direct(const float *src, int c0, int my_chunks, float (&xr)[NCH][8]) {
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int j = 0; j < NCH; ++j) {
        const int ch = j * 32 + lane;
        if (ch < my_chunks) {
            const float4 a = ld_act4(src + (size_t)(c0 + ch) * 8), b = ld_act4(src + (size_t)(c0 + ch) * 8 + 4);
            xr[j][0] = a.x; xr[j][1] = a.y; xr[j][2] = a.z; xr[j][3] = a.w;
            xr[j][4] = b.x; xr[j][5] = b.y; xr[j][6] = b.z; xr[j][7] = b.w;
        } else {
#pragma unroll
            for (int i = 0; i < 8; ++i) xr[j][i] = 0.f;
        }
    }
}

// fused epilogue of one finished unit (two row totals a, b) of a phase whose rows are whole in one warp
__device__ __forceinline__ void finish_unit(const MegaParams &p, MkCtx &c, int ph, int u, float a, float b, const MkShared &sh) {
    if (ph == PH_QKV) {
        // A4: RoPE on q and k heads (pair (i, i+32)), q -> scratch, k/v -> cache row of this position (fp16)
        const int hh = u >> 5, i = u & 31;
        if (hh < p.n_heads) {
            const float2 cs = sh.rope[i];
            p.qkv[hh * kHeadDim + i] = a * cs.x - b * cs.y;
            p.qkv[hh * kHeadDim + i + 32] = b * cs.x + a * cs.y;
        } else {
            const bool is_k = hh < p.n_heads + p.n_kv_heads;
            const int kvh = hh - p.n_heads - (is_k ? 0 : p.n_kv_heads);
            float o0 = a, o1 = b;
            if (is_k) {
                const float2 cs = sh.rope[i];
                o0 = a * cs.x - b * cs.y;
                o1 = b * cs.x + a * cs.y;
            }
            kv_t *row = (is_k ? p.kc : p.vc) + (size_t)c.layer * p.layer_kv + ((size_t)kvh * p.max_seq + c.pos) * kHeadDim;
            row[i] = __float2half_rn(o0);
            row[i + 32] = __float2half_rn(o1);
        }
    } else if (ph == PH_GATEUP) {
        p.act[u] = silu_f(a) * b;   // A7: fused SwiGLU
    } else {
        // A9: logits + running packed argmax (lowest index wins ties)
        *reinterpret_cast<float2 *>(p.logits + 2 * u) = make_float2(a, b);
        unsigned long long ka = pack_argmax(a, 2 * u), kb = pack_argmax(b, 2 * u + 1);
        ka = ka > kb ? ka : kb;
        c.best = c.best > ka ? c.best : ka;
    }
}

// One weight phase on the consumer side: input slice -> registers, then stage by stage, no CTA-wide sync.
template <int NCH>
__device__ __forceinline__ void consume_phase(const MegaParams &p, MkCtx &c, int ph, const PhaseGeom &geo, const uint8_t *ring,
                                              MkShared &sh) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int slice = warp & (geo.S - 1), pair = warp >> geo.log2S;
    const int chunks = geo.K >> 3, c0 = slice * geo.cps;
    const int my_chunks = min(chunks, c0 + geo.cps) - c0;   // may be <= 0 for a ragged tail slice
    const bool resid = (ph == PH_O || ph == PH_DOWN);

    // A6/A8: the threads that will finish the residual rows fetch the old values now
    float rold = 0.f;
    const int n_rows_cta = 2 * (geo.u1 - geo.u0);
    if (resid && tid < n_rows_cta) {
        const int r = 2 * geo.u0 + tid;
        rold = (ph == PH_O && c.layer == 0) ? __bfloat162float(p.emb[(size_t)c.tok * p.hidden + r]) : ld_act(p.x + r);
    }

    float xr[NCH][8];
    if (geo.K <= kMkStagedK) {   // S == 1: the warp holds the whole vector
        stage_input(p, c, ph, geo.K, sh);
        load_x_staged<NCH>(sh, my_chunks, xr);
    } else {
        load_x_direct<NCH>(p.act, c0, my_chunks, xr);   // only the down projection has K > kMkStagedK
    }
    mk_trace(p, c);

    for (int s = 0; s < geo.n_stages; ++s, ++c.g) {
        const int slot = c.g % kMkStages;
        const uint32_t par = (c.g / kMkStages) & 1;
        const int ub = geo.u0 + s * geo.ups;
        const int nu = min(geo.ups, geo.u1 - ub);
        mk_mbar_wait(&sh.full[slot], par, p.err);
        if (s == 0) mk_trace(p, c);
        float a0 = 0.f, a1 = 0.f, b0 = 0.f, b1 = 0.f;
        if (pair < nu) {
            const uint4 *r0 = reinterpret_cast<const uint4 *>(ring + (size_t)slot * kMkStageBytes + (size_t)(2 * pair) * geo.row_bytes) + c0;
            const uint4 *r1 = r0 + (geo.row_bytes >> 4);
#pragma unroll
            for (int j = 0; j < NCH; ++j) {
                const int ch = j * 32 + lane;
                if (ch < my_chunks) {
                    if (j & 1) { a1 = dot8(r0[ch], xr[j], a1); b1 = dot8(r1[ch], xr[j], b1); }
                    else { a0 = dot8(r0[ch], xr[j], a0); b0 = dot8(r1[ch], xr[j], b0); }
                }
            }
        }
        float a = a0 + a1, b = b0 + b1;
        // both row totals with 6 shuffles: halves swap rows, 4 butterfly steps, one exchange
        const bool up = (lane & 16) != 0;
        float v = (up ? b : a) + __shfl_xor_sync(0xffffffffu, up ? a : b, 16);
#pragma unroll
        for (int o = 8; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        const float w = __shfl_xor_sync(0xffffffffu, v, 16);   // lane 0: v = row a total, w = row b total
        if (lane == 0) {
            mk_mbar_arrive(&sh.empty[slot]);   // the shuffles ordered every lane's shared loads before this
            if (pair < nu) {
                if (resid) {
                    const int rl = 2 * (s * geo.ups + pair);
                    sh.part[rl][slice] = v;
                    sh.part[rl + 1][slice] = w;
                } else {
                    finish_unit(p, c, ph, ub + pair, v, w, sh);
                }
            }
        }
    }
    if (resid) {
        consumer_sync();
        if (tid < n_rows_cta) {
            float t = rold;
            for (int k = 0; k < geo.S; ++k) t += sh.part[tid][k];
            p.x[2 * geo.u0 + tid] = t;
        }
        // sh.part is next written after the grid barrier that follows every residual phase
    }
}

__device__ __forceinline__ void run_phase(const MegaParams &p, MkCtx &c, int ph, const uint8_t *ring, MkShared &sh) {
    const PhaseGeom geo = phase_geom(p, ph);
    const int nch = (geo.cps + 31) / 32;
    if (nch <= 1) consume_phase<1>(p, c, ph, geo, ring, sh);
    else if (nch <= 2) consume_phase<2>(p, c, ph, geo, ring, sh);
    else if (nch <= 4) consume_phase<4>(p, c, ph, geo, ring, sh);
    else consume_phase<8>(p, c, ph, geo, ring, sh);
    mk_trace(p, c);
}

// ---- A5: attention phase ---------------------------------------------------------------------------------------
// Work item of a CTA = (KV head, context split); warp = (query head of the group, sub-split); LANE = POSITION.
// attn_prefetch runs BEFORE the grid barrier that ends the QKV phase: the K/V rows of earlier positions do not depend
// on this step's projections, so their HBM/L2 latency overlaps the barrier.  Only the row of the current position
// (written by the QKV phase of this step) has to wait.
struct AttnItem {
    int kvh, split, g, sub, w1, t0;
    bool has_item, active, pre;
};
__device__ __forceinline__ void attn_prefetch(const MegaParams &p, const MkCtx &c, AttnItem &it, KvRow &kr, KvRow &vr) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int G = p.n_heads / p.n_kv_heads, nsub = kMkConsumerWarps / G;
    const int n_ctx = c.pos + 1;
    const int ns = mk_num_splits(p, n_ctx, nsub);
    const int len = (n_ctx + ns - 1) / ns;
    it.has_item = (int)blockIdx.x < p.n_kv_heads * ns;
    it.kvh = (int)blockIdx.x / ns;
    it.split = (int)blockIdx.x % ns;
    it.g = warp % G;
    it.sub = warp / G;
    it.active = it.has_item && warp < G * nsub;
    const int s0 = it.split * len, s1 = min(n_ctx, s0 + len);
    const int sub_len = (max(s1 - s0, 0) + nsub - 1) / nsub;
    const int w0 = s0 + it.sub * sub_len;
    it.w1 = min(s1, w0 + sub_len);
    it.t0 = w0 + lane;
    it.pre = it.active && it.t0 < it.w1 && it.t0 < c.pos;
    if (it.pre) {
        const size_t off = (size_t)c.layer * p.layer_kv + ((size_t)it.kvh * p.max_seq + it.t0) * kHeadDim;
        ld_kv_row(kr, p.kc + off);
        ld_kv_row(vr, p.vc + off);
    }
}

__device__ void attention_phase(const MegaParams &p, MkCtx &c, MkShared &sh, const AttnItem &it, KvRow &kr, KvRow &vr) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (!it.has_item) { mk_trace(p, c); mk_trace(p, c); mk_trace(p, c); return; }
    const int G = p.n_heads / p.n_kv_heads, nsub = kMkConsumerWarps / G;
    const int head = it.kvh * G + it.g;
    const int r = warp_row_of_lane<32>(lane);   // the output dims (r, 32 + r) this lane holds after the merge
    float M = -INFINITY, l_tot = 0.f, o_lo = 0.f, o_hi = 0.f;
    if (it.active) {
        // the warp's query, pre-scaled by 1/sqrt(64) = 0.125 (exact), broadcast-read from shared memory below
        if (lane < 16) {
            float4 qv = ld_act4(p.qkv + (size_t)head * kHeadDim + lane * 4);
            qv.x *= 0.125f; qv.y *= 0.125f; qv.z *= 0.125f; qv.w *= 0.125f;
            reinterpret_cast<float4 *>(sh.q[warp])[lane] = qv;
        }
        __syncwarp();
    }
    mk_trace(p, c);
    if (it.active) {
        const kv_t *kg = p.kc + (size_t)c.layer * p.layer_kv + (size_t)it.kvh * p.max_seq * kHeadDim;
        const kv_t *vg = p.vc + (size_t)c.layer * p.layer_kv + (size_t)it.kvh * p.max_seq * kHeadDim;
        const float4 *q4 = reinterpret_cast<const float4 *>(sh.q[warp]);
        float m = -INFINITY, l = 0.f, o[kHeadDim];
#pragma unroll
        for (int d = 0; d < kHeadDim; ++d) o[d] = 0.f;
        bool loaded = it.pre;
        for (int t = it.t0; t < it.w1; t += 32) {
            if (!loaded) {
                ld_kv_row(kr, kg + (size_t)t * kHeadDim);
                ld_kv_row(vr, vg + (size_t)t * kHeadDim);
            }
            loaded = false;
            float s = 0.f, s2 = 0.f;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const float4 qa = q4[2 * j], qb = q4[2 * j + 1];
                const float2 k0 = h2f(kr.v[j].x), k1 = h2f(kr.v[j].y), k2 = h2f(kr.v[j].z), k3 = h2f(kr.v[j].w);
                s = fmaf(qa.x, k0.x, s); s2 = fmaf(qa.y, k0.y, s2);
                s = fmaf(qa.z, k1.x, s); s2 = fmaf(qa.w, k1.y, s2);
                s = fmaf(qb.x, k2.x, s); s2 = fmaf(qb.y, k2.y, s2);
                s = fmaf(qb.z, k3.x, s); s2 = fmaf(qb.w, k3.y, s2);
            }
            s += s2;
            const float m_new = fmaxf(m, s);
            const float corr = __expf(m - m_new);   // m = -inf the first time -> 0
            const float pr = __expf(s - m_new);
            l = l * corr + pr;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const float2 v0 = h2f(vr.v[j].x), v1 = h2f(vr.v[j].y), v2 = h2f(vr.v[j].z), v3 = h2f(vr.v[j].w);
                o[8 * j + 0] = fmaf(pr, v0.x, o[8 * j + 0] * corr);
                o[8 * j + 1] = fmaf(pr, v0.y, o[8 * j + 1] * corr);
                o[8 * j + 2] = fmaf(pr, v1.x, o[8 * j + 2] * corr);
                o[8 * j + 3] = fmaf(pr, v1.y, o[8 * j + 3] * corr);
                o[8 * j + 4] = fmaf(pr, v2.x, o[8 * j + 4] * corr);
                o[8 * j + 5] = fmaf(pr, v2.y, o[8 * j + 5] * corr);
                o[8 * j + 6] = fmaf(pr, v3.x, o[8 * j + 6] * corr);
                o[8 * j + 7] = fmaf(pr, v3.y, o[8 * j + 7] * corr);
            }
            m = m_new;
        }
        // merge the 32 lane states: common max, rescale, transposed butterfly over the 64 dims
        M = warp_max(m);
        const float sc = (m == -INFINITY) ? 0.f : __expf(m - M);
        l_tot = warp_sum(l * sc);
#pragma unroll
        for (int d = 0; d < kHeadDim; ++d) o[d] *= sc;
        float(&h0)[32] = *reinterpret_cast<float(*)[32]>(&o[0]);
        float(&h1)[32] = *reinterpret_cast<float(*)[32]>(&o[32]);
        warp_reduce_rows<32>(h0, lane);
        warp_reduce_rows<32>(h1, lane);
        o_lo = h0[0];
        o_hi = h1[0];
        if (it.sub > 0) {   // park the state for the sub-split 0 warp of this head
            sh.mrg[warp][r] = o_lo;
            sh.mrg[warp][32 + r] = o_hi;
            if (lane == 0) { sh.mrg[warp][kHeadDim] = M; sh.mrg[warp][kHeadDim + 1] = l_tot; }
        }
    }
    if (nsub > 1) consumer_sync();
    if (it.active && it.sub == 0) {
        for (int k = 1; k < nsub; ++k) {
            const float *o2 = sh.mrg[k * G + it.g];
            const float M2 = o2[kHeadDim], l2 = o2[kHeadDim + 1];
            const float Mn = fmaxf(M, M2);
            const float wa = (M == -INFINITY) ? 0.f : __expf(M - Mn), wb = (M2 == -INFINITY) ? 0.f : __expf(M2 - Mn);
            l_tot = l_tot * wa + l2 * wb;
            o_lo = o_lo * wa + o2[r] * wb;
            o_hi = o_hi * wa + o2[32 + r] * wb;
            M = Mn;
        }
        // unnormalised split state; the O phase of every CTA merges the splits while it stages its input (stage_input)
        const size_t pidx = (size_t)head * kMkMaxSplits + it.split;
        p.part_o[pidx * kHeadDim + r] = o_lo;
        p.part_o[pidx * kHeadDim + 32 + r] = o_hi;
        if (lane == 0) p.part_ml[pidx] = make_float2(M, l_tot);
    }
    mk_trace(p, c);
    mk_trace(p, c);
    // sh.q / sh.mrg are next written after two more grid barriers
}

// ---- the kernel -----------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kMkThreads, 1) mega_decode_kernel(const __grid_constant__ MegaParams p) {
    extern __shared__ __align__(128) uint8_t mk_smem[];
    uint8_t *ring = mk_smem;
    MkShared &sh = *reinterpret_cast<MkShared *>(mk_smem + (size_t)kMkStages * kMkStageBytes);
    const int tid = threadIdx.x, warp = tid >> 5;

    if (tid == 0) {
        for (int s = 0; s < kMkStages; ++s) {
            mk_mbar_init(&sh.full[s], 1);
            mk_mbar_init(&sh.empty[s], kMkConsumerWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == kMkConsumerWarps) {
        if ((tid & 31) == 0) mk_producer(p, ring, sh);
        return;
    }

    MkCtx c;
    c.g = 0;
    c.bar_target = 0;
    c.best = 0ull;
    c.ti = 0;
    c.pos = ld_act(p.pos);
    c.tok = ld_act(p.tok_src);
    mk_trace(p, c);
    for (int step = 0; step < p.n_steps; ++step) {
        if (tid < 32) sh.rope[tid] = p.rope[(size_t)c.pos * 32 + tid];
        consumer_sync();
        for (c.layer = 0; c.layer < p.n_layers; ++c.layer) {
            run_phase(p, c, PH_QKV, ring, sh);
            AttnItem it;
            KvRow kr, vr;
            attn_prefetch(p, c, it, kr, vr);
            grid_barrier(p, c);
            attention_phase(p, c, sh, it, kr, vr);
            grid_barrier(p, c);
            run_phase(p, c, PH_O, ring, sh);
            grid_barrier(p, c);
            run_phase(p, c, PH_GATEUP, ring, sh);
            grid_barrier(p, c);
            run_phase(p, c, PH_DOWN, ring, sh);
            grid_barrier(p, c);
            if (p.hidden_out && blockIdx.x == 0)
                for (int i = tid; i < p.hidden; i += kMkConsumers)
                    p.hidden_out[(size_t)c.layer * p.hidden_stride + i] = ld_act(p.x + i);
        }
        if (p.with_head) {
            // A9: every CTA folds its best (logit, index) into the step's slot with one packed 64-bit atomicMax
            // before the barrier; after it every CTA reads the winner = the next token.  Two slots alternate so
            // the one not in use can be cleared without a further barrier.
            c.best = 0ull;
            run_phase(p, c, PH_HEAD, ring, sh);
            unsigned long long *slot = p.best2 + (step & 1);
            if ((tid & 31) == 0) sh.wbest[warp] = c.best;   // lane 0 ran every epilogue of its warp
            consumer_sync();
            if (tid == 0) {
                unsigned long long b = sh.wbest[0];
                for (int k = 1; k < kMkConsumerWarps; ++k) b = b > sh.wbest[k] ? b : sh.wbest[k];
                if (b) atomicMax(slot, b);
            }
            grid_barrier(p, c);
            const unsigned long long win = __ldcg(slot);
            c.tok = unpack_argmax_idx(win);
            if (blockIdx.x == 0 && tid == 0) {
                *p.cur_tok = c.tok;
                p.tok_hist[c.pos + 1] = c.tok;
                *p.pos = c.pos + 1;
                p.best2[(step + 1) & 1] = 0ull;   // last read two barriers ago, next written after >= 1 more
            }
        } else {
            if (blockIdx.x == 0 && tid == 0) *p.pos = c.pos + 1;
            c.tok = 0;   // without the head the kernel runs one step (hq_prefill token walk)
        }
        c.pos += 1;
    }
    // leave the barrier counter and the argmax slots at zero for the next launch: the last CTA out resets them
    consumer_sync();
    if (tid == 0) {
        __threadfence();
        const unsigned t = atomicAdd(p.exit_ticket, 1u);
        if (t == gridDim.x - 1) {
            *p.bar = 0u;
            *p.exit_ticket = 0u;
            p.best2[0] = 0ull;
            p.best2[1] = 0ull;
        }
    }
}

// ---- host side ---------------------------------------------------------------------------------------------------
size_t mega_smem_bytes() { return (size_t)kMkStages * kMkStageBytes + sizeof(MkShared) + 128; }

bool mega_shape_supported(const hq_config &c, int n_sms) {
    // RMSNorm phases keep the whole vector in one warp (hidden <= 2048); residual phases cut K into <= 8 slices;
    // the residual rows of one CTA must fit the partial buffer; the group must fit the consumer warps
    const int q = c.n_heads * c.head_dim;
    const int units_cta = (c.hidden / 2 + n_sms - 1) / n_sms;
    return c.hidden <= kMkStagedK && q <= kMkStagedK && c.ffn <= 64 * kMkSliceChunks &&
           2 * units_cta <= kMkPartRows && c.n_heads / c.n_kv_heads <= kMkConsumerWarps && c.hidden % 8 == 0 &&
           c.ffn % 8 == 0 && c.vocab % 2 == 0 && n_sms >= c.n_kv_heads;
}

cudaError_t launch_mega(const LaunchCtx &c, const MegaParams &p, bool cooperative) {
    static bool attr_done = false;
    const size_t smem = mega_smem_bytes();
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(mega_decode_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(c.n_sms);
    cfg.blockDim = dim3(kMkThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = c.stream;
    // cooperative: the driver guarantees (and checks) that all CTAs are co-resident — the grid barrier needs it
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;
    attr[0].val.cooperative = 1;
    cfg.attrs = attr;
    cfg.numAttrs = cooperative ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, mega_decode_kernel, p);
}

}  // namespace hq
