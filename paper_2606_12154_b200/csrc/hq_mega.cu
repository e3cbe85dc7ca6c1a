// hq_mega.cu — persistent batch-1 decode: SURVEY.md §8(a) rows A1-A9 for n_steps tokens in ONE launch.
//
// Why: one token is a chain of 81 HBM-bound matrix-vector products over 2.47 GB of bf16 weights.  With one
// kernel per product the three small products of every layer (QKV, attention, O) cost more in kernel-boundary
// latency than in DRAM time (profiles/r01_decode_launches_v1.md: 53 % of the copy peak).  Here the weight
// stream never stops:
//   * grid = one CTA per SM, 9 warps.  Warp 8 is the PRODUCER: one elected thread walks the static schedule
//     (layer, phase, this CTA's rows) and streams every weight row with cp.async.bulk (TMA bulk copy,
//     mbarrier complete_tx, L2 evict-first) into a ring of kMkStages x 64 KB shared-memory stages.  Weights are
//     immutable, so the producer runs ahead of the data dependencies: while the consumers wait for another SM's
//     result or do the attention, the next phases' rows are already landing.
//   * warps 0-7 are CONSUMERS and never synchronise with one another inside a weight phase.  A stage holds
//     8/S "units" (a unit = two rows: RoPE pair (i, i+32) / gate+up pair / two adjacent rows); a row is cut
//     into S slices of <= 2048 elements and warp w owns slice w % S of unit w / S, so the slice of the
//     (normalised) input vector it needs stays in 64 registers for the whole phase.  Per stage and warp: two
//     conflict-free 16-byte shared loads per chunk, fp32 FMA, one 6-shuffle reduction for both rows, one
//     mbarrier arrive, and the fused epilogue (RoPE + KV append, SwiGLU, logits + packed argmax) from lane 0.
//   * NO GRID BARRIERS AND NO FENCES.  Measured on B200 (profiles/r01_mega_sync_microbench.md): with the ring's
//     192 KB of bulk copies in flight per SM a membar.gpu / red.release takes 3-9 us (idle: 0.35 us) and a
//     release/acquire grid barrier 10 us, i.e. more than the 1.2 us of DRAM time of a small phase.  So every vector that
//     crosses CTAs (residual x, q/k/v of the token, split-KV partials, SwiGLU output, per-CTA argmax) travels
//     as 8-byte (fp32 value, 32-bit epoch tag) words written with ONE relaxed 64-bit store each and polled by
//     the readers until every tag equals the epoch of (step, layer) — the "flag in the data" protocol of
//     latency-bound collectives.  A 64-bit aligned store is single-copy atomic, so a matching tag proves the
//     value; no ordering between different words is ever needed.  Reuse of a buffer is safe by the data
//     dependencies themselves (its next writer needs, transitively, a result from every reader of the
//     previous epoch).
//   * attention: work item = (KV head, context split); warp = (query head of the group, sub-split); LANE =
//     POSITION: every lane runs its own online softmax over its positions (K/V rows are one 128-byte line each,
//     read with 256-bit loads issued BEFORE the warp waits for its query), then the 32 lane states are merged
//     with a transposed butterfly, the sub-splits through shared memory; the split states (m, l, o) go out as
//     tagged words and every CTA merges them while it stages the input of the O projection.
#include "hq_common.cuh"
#include "hq_internal.h"

namespace hq {

constexpr int kMkConsumerWarps = 8;
constexpr int kMkConsumers = 32 * kMkConsumerWarps;
constexpr int kMkThreads = kMkConsumers + 32;
constexpr int kMkPartRows = 64;                   // residual rows of one CTA in one phase (2 * units)
constexpr int kMkStagedK = 8 * kMkConsumers;      // 2048: one 8-element chunk per consumer thread
constexpr unsigned kMaxPollSpins = 1u << 23;      // poll rounds (each >= one L2 round trip + 64 ns sleep) before a lost word traps
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
__device__ __noinline__ void mk_fail(int *err, int code) {
    atomicExch(err, code);
    __threadfence_system();
    __trap();
}
// slow path out of line: the kernel's steady-state code must fit the instruction cache (see consume_phase)
__device__ __noinline__ void mk_mbar_wait_slow(uint64_t *bar, uint32_t parity, int *err) {
    const long long t0 = clock64();
    unsigned spins = 0;
    while (!mk_mbar_try_wait(bar, parity))
        if ((++spins & 1023u) == 0 && clock64() - t0 > kSpinCycles) mk_fail(err, 1);
}
__device__ __forceinline__ void mk_mbar_wait(uint64_t *bar, uint32_t parity, int *err) {
    if (!mk_mbar_try_wait(bar, parity)) mk_mbar_wait_slow(bar, parity, err);
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
__device__ __forceinline__ void consumer_sync() { asm volatile("bar.sync 1, %0;" ::"n"(kMkConsumers) : "memory"); }
// ---- tagged words: (fp32 value | 32-bit epoch tag) in one 64-bit word -------------------------------------
typedef unsigned long long llw_t;
__device__ __forceinline__ void ll_store(llw_t *p, float v, uint32_t tag) {
    const llw_t w = ((llw_t)tag << 32) | (llw_t)__float_as_uint(v);
    asm volatile("st.global.cg.u64 [%0], %1;" ::"l"(p), "l"(w) : "memory");
}
__device__ __forceinline__ void ll_store_u32(llw_t *p, uint32_t v, uint32_t tag) {
    const llw_t w = ((llw_t)tag << 32) | (llw_t)v;
    asm volatile("st.global.cg.u64 [%0], %1;" ::"l"(p), "l"(w) : "memory");
}
__device__ __forceinline__ void ll_load2(const llw_t *p, llw_t &a, llw_t &b) {
    asm volatile("ld.volatile.global.v2.u64 {%0,%1}, [%2];" : "=l"(a), "=l"(b) : "l"(p) : "memory");
}
__device__ __forceinline__ bool ll_ok(llw_t w, uint32_t tag) { return (uint32_t)(w >> 32) == tag; }
__device__ __forceinline__ float ll_val(llw_t w) { return __uint_as_float((uint32_t)w); }
// Poll N (even) consecutive tagged words until all carry `tag`.  All loads of a round are in flight together.
template <int N>
__device__ __forceinline__ void ll_poll(const llw_t *src, uint32_t tag, float (&v)[N], int *err) {
    llw_t w[N];
    unsigned spins = 0;
    for (;;) {
#pragma unroll
        for (int i = 0; i < N; i += 2) ll_load2(src + i, w[i], w[i + 1]);
        bool ok = true;
#pragma unroll
        for (int i = 0; i < N; ++i) ok = ok && ll_ok(w[i], tag);
        if (ok) break;
        if (++spins == kMaxPollSpins) mk_fail(err, 3);
        __nanosleep(20);
    }
#pragma unroll
    for (int i = 0; i < N; ++i) v[i] = ll_val(w[i]);
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
    const int lim = chunks > kMkSliceChunks ? kMkSliceChunks / 2 : kMkSliceChunks;   // un-staged inputs: 4 chunks per lane = one poll round
    while ((chunks + g.S - 1) / g.S > lim) { g.S <<= 1; ++g.log2S; }
    g.cps = (chunks + g.S - 1) / g.S;
    g.ups = kMkConsumerWarps >> g.log2S;
    // optional (p.att_ctas > 0): the last p.att_ctas CTAs do nothing but attention and the weight rows are dealt to the
    // others.  Measured slower (1,399 -> 1,334 tok/s): the weight stream loses more than the attention gains.
    const int W = (int)gridDim.x - p.att_ctas;
    const int n = phase_units(p, ph), per = n / W, rem = n % W, b = blockIdx.x;
    g.u0 = b < W ? b * per + min(b, rem) : 0;
    g.u1 = b < W ? g.u0 + per + (b < rem ? 1 : 0) : 0;
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
    PhaseGeom geo[5];                            // this CTA's static schedule, computed once (integer divisions out of the loop)
    alignas(16) float xs[kMkStagedK];            // phase input staged once per CTA (phases with K <= kMkStagedK)
    float part[kMkPartRows][kMkConsumerWarps];   // residual phases: [row of this CTA][slice] partial sums
    float2 rope[32];
    alignas(16) kv_t kvnew[kMkConsumerWarps][2][kHeadDim];   // per warp: this step's K and V row (fp16 like the cache)
    float mrg[kMkConsumerWarps][kHeadDim + 2];   // attention: sub-split states (o[64], m, l)
    float red[kMkConsumerWarps];                 // RMSNorm: per-warp sum of squares
    unsigned long long wbest[kMkConsumerWarps];  // LM head: per-warp packed argmax
};

// ---- producer ----------------------------------------------------------------------------------------------
// One elected thread walks this CTA's static schedule and fills the shared-memory ring (TMA bulk copies, mbarrier
// complete_tx, L2 evict-first).  At most p.inflight_stages stages are issued and not yet landed: a deeper queue buys no
// bandwidth, it only delays the small exchange loads and stores (and instruction fetches) that share the memory system
// with the stream (queueing delay = bytes in flight / HBM rate, profiles/r01_mega_sync_microbench.md).
__device__ void mk_producer(const MegaParams &p, uint8_t *ring, MkShared &sh) {
    const uint64_t pol = mk_policy_evict_first();
    const int n_ph = p.n_layers * 4 + (p.with_head ? 1 : 0);
    unsigned g = 0;   // stages produced so far
    const int pi0 = p.x_plain ? p.pi_begin : 0, pi1 = p.x_plain ? p.pi_end : n_ph;
    for (int step = 0; step < p.n_steps; ++step)
        for (int pi = pi0; pi < pi1; ++pi) {
            const int layer = pi >> 2;
            const int ph = layer < p.n_layers ? (pi & 3) : PH_HEAD;
            const LayerW &w = p.layers[layer < p.n_layers ? layer : 0];
            const PhaseGeom &geo = sh.geo[ph];
            for (int s = 0; s < geo.n_stages; ++s, ++g) {
                const int slot = g % kMkStages;
                mk_mbar_wait(&sh.empty[slot], ((g / kMkStages) & 1) ^ 1, p.err);
                // the LM head has no exchange to protect: full depth there (7.1 vs 5.4 TB/s)
                const unsigned infl = ph == PH_HEAD ? (unsigned)kMkStages : (unsigned)p.inflight_stages;
                if (g >= infl) {
                    const unsigned gl = g - infl;
                    mk_mbar_wait(&sh.full[gl % kMkStages], (gl / kMkStages) & 1, p.err);
                }
                const int ub = geo.u0 + s * geo.ups;
                const int nu = min(geo.ups, geo.u1 - ub);
                mk_mbar_expect_tx(&sh.full[slot], (uint32_t)(2 * nu * geo.row_bytes));
                uint8_t *dst = ring + (size_t)slot * kMkStageBytes;
#pragma unroll 1
                for (int j = 0; j < nu; ++j) {
                    const bf16 *ra, *rb;
                    unit_row_ptrs(p, w, ph, geo.K, ub + j, ra, rb);
                    mk_bulk_g2s_hint(dst + (size_t)(2 * j) * geo.row_bytes, ra, geo.row_bytes, &sh.full[slot], pol);
                    mk_bulk_g2s_hint(dst + (size_t)(2 * j + 1) * geo.row_bytes, rb, geo.row_bytes, &sh.full[slot], pol);
                }
            }
        }
}

// ---- consumer state ------------------------------------------------------------------------------------------
struct MkCtx {
    unsigned g;          // stages consumed so far
    int pos, tok;
    int layer;
    uint32_t tag;        // epoch tag of (step, layer): every word exchanged in this layer carries it
    uint32_t tag_prev;   // tag of the previous layer of this step (input of the QKV phase / the LM head)
    uint4 gain_pre;      // attention-block launch: the layer's attn_norm gains, loaded before the dependency wait
    float rold;          // residual phases: thread tid < rows of this CTA keeps x[row] in a register
    int ti;              // trace cursor (thread 0)
    unsigned long long best;
};

// optional timeline (hq_debug_trace): every CTA's thread 0 stamps the global timer at fixed points
template <bool TRACE>
__device__ __forceinline__ void mk_trace(const MegaParams &p, MkCtx &c) {
    if (TRACE && p.trace && threadIdx.x == 0) {
        if (c.ti < p.trace_cap) p.trace[(size_t)blockIdx.x * p.trace_cap + c.ti] = mk_globaltimer();
        ++c.ti;
    }
}

// context splits per KV head at this position: one 32-position batch per warp before another split is added, at most
// p.att_splits (the attention CTAs the launch set aside).  A function of the device-resident position: graph safe.
__device__ __forceinline__ int mk_num_splits(const MegaParams &p, int n_ctx) {
    const int G = p.n_heads / p.n_kv_heads, per = 32 * (kMkConsumerWarps / G);
    const int want = (n_ctx + per - 1) / per;
    return want < p.att_splits ? want : p.att_splits;
}

// Phase input, K <= kMkStagedK: the CTA polls the tagged vector from L2 ONCE (thread t owns elements [8t, 8t+8)),
// applies the fused prologue, and leaves it in shared memory for its 8 warps.
//   QKV, gate/up, LM head: A2 RMSNorm (sum of squares reduced across the CTA, deterministic), gain multiply
//   O:                     A5 merge of the split-KV states (m, l, o) written by the attention phase
//   down (small models):   plain copy
template <bool BLOCK>
__device__ __forceinline__ void stage_input(const MegaParams &p, MkCtx &c, int ph, int K, MkShared &sh) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const bool has = tid * 8 < K;
    float v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = 0.f;
    if (ph == PH_O) {
        // A5 output: the normalised attention vector published by the split-0 CTA of every KV head.  Gate: ONE warp
        // watches one word per head with back-off while the other 7 sleep in the CTA barrier, so that the chip does not
        // poll the same 128 lines for the whole attention phase.
        if (tid < 32) {
            unsigned spins = 0;
            for (;;) {
                bool ok = true;
                for (int h = lane; h < p.n_heads; h += 32) {
                    llw_t w0;
                    asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(w0) : "l"(p.ll_attn + (size_t)h * kHeadDim + kHeadDim - 1) : "memory");
                    ok = ok && ll_ok(w0, c.tag);
                }
                if (__all_sync(0xffffffffu, ok)) break;
                if (++spins == kMaxPollSpins) mk_fail(p.err, 8);
                __nanosleep(20);
            }
        }
        consumer_sync();
        if (has) ll_poll<8>(p.ll_attn + (size_t)tid * 8, c.tag, v, p.err);
    } else if (!BLOCK && ph == PH_DOWN) {
        if (has) ll_poll<8>(p.ll_act + (size_t)tid * 8, c.tag, v, p.err);
    } else {
        const bf16 *gain = ph == PH_QKV ? p.layers[c.layer].attn_norm : (ph == PH_GATEUP ? p.layers[c.layer].ffn_norm : p.final_norm);
        uint4 gq = make_uint4(0, 0, 0, 0);
        if (BLOCK) gq = c.gain_pre;
        else if (has) gq = __ldg(reinterpret_cast<const uint4 *>(gain) + tid);
        if (has) {
            if (BLOCK) {   // attention-block launch: the residual stream is a plain vector written by the previous kernel
                const float4 a = ld_act4(p.x_plain + (size_t)tid * 8), b = ld_act4(p.x_plain + (size_t)tid * 8 + 4);
                v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
            } else if (ph == PH_QKV && c.layer == 0) {   // A1: the residual stream starts as the embedding row
                const uint4 e = __ldg(reinterpret_cast<const uint4 *>(p.emb + (size_t)c.tok * p.hidden) + tid);
                v[0] = bf16lo(e.x); v[1] = bf16hi(e.x); v[2] = bf16lo(e.y); v[3] = bf16hi(e.y);
                v[4] = bf16lo(e.z); v[5] = bf16hi(e.z); v[6] = bf16lo(e.w); v[7] = bf16hi(e.w);
            } else if (ph == PH_GATEUP) {
                ll_poll<8>(p.ll_x + (size_t)tid * 8, c.tag, v, p.err);                  // x after the O projection
            } else {
                ll_poll<8>(p.ll_x + (size_t)p.hidden + (size_t)tid * 8, c.tag_prev, v, p.err);   // x after the previous layer
                if (p.hidden_out && blockIdx.x == 0) {   // parity capture: residual after layer (c.layer - 1) / the last layer
                    const int l = (ph == PH_HEAD ? p.n_layers : c.layer) - 1;
                    float4 *dst = reinterpret_cast<float4 *>(p.hidden_out + (size_t)l * p.hidden_stride + tid * 8);
                    dst[0] = make_float4(v[0], v[1], v[2], v[3]);
                    dst[1] = make_float4(v[4], v[5], v[6], v[7]);
                }
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
// K > kMkStagedK (the down projection of the 1B model, K = 8192): every warp polls its own slice of the tagged
// SwiGLU vector straight into registers, up to four chunks (32 words) per lane and round trip
template <int NCH>
__device__ __forceinline__ void load_x_direct(const MegaParams &p, const MkCtx &c, int c0, int my_chunks, float (&xr)[NCH][8]) {
    const int lane = threadIdx.x & 31;
    constexpr int NB = NCH < 4 ? NCH : 4;
    if (my_chunks <= 0) {
#pragma unroll
        for (int j = 0; j < NCH; ++j)
#pragma unroll
            for (int i = 0; i < 8; ++i) xr[j][i] = 0.f;
        return;
    }
#pragma unroll
    for (int j0 = 0; j0 < NCH; j0 += NB) {
        llw_t w[NB][8];
        unsigned spins = 0;
        for (;;) {
#pragma unroll
            for (int k = 0; k < NB; ++k) {
                const int ch = min((j0 + k) * 32 + lane, my_chunks - 1);   // past the end: re-read a valid chunk
#pragma unroll
                for (int i = 0; i < 8; i += 2) ll_load2(p.ll_act + (size_t)(c0 + ch) * 8 + i, w[k][i], w[k][i + 1]);
            }
            bool ok = true;
#pragma unroll
            for (int k = 0; k < NB; ++k)
#pragma unroll
                for (int i = 0; i < 8; ++i) ok = ok && ll_ok(w[k][i], c.tag);
            if (ok) break;
            if (++spins == kMaxPollSpins) mk_fail(p.err, 5);
                __nanosleep(20);
        }
#pragma unroll
        for (int k = 0; k < NB; ++k) {
            const bool in = (j0 + k) * 32 + lane < my_chunks;
#pragma unroll
            for (int i = 0; i < 8; ++i) xr[j0 + k][i] = in ? ll_val(w[k][i]) : 0.f;
        }
    }
}

// fused epilogue of one finished unit (two row totals a, b) of a phase whose rows are whole in one warp
template <bool BLOCK>
__device__ __forceinline__ void finish_unit(const MegaParams &p, MkCtx &c, int ph, int u, float a, float b, const MkShared &sh) {
    if (BLOCK || ph == PH_QKV) {
        // A4: RoPE on q and k heads (pair (i, i+32)); q, k, v of the token -> tagged words; k, v also -> cache (fp16)
        const int hh = u >> 5, i = u & 31;
        float o0 = a, o1 = b;
        if (hh < p.n_heads + p.n_kv_heads) {
            const float2 cs = sh.rope[i];
            o0 = a * cs.x - b * cs.y;
            o1 = b * cs.x + a * cs.y;
        }
        ll_store(p.ll_qkv + hh * kHeadDim + i, o0, c.tag);
        ll_store(p.ll_qkv + hh * kHeadDim + i + 32, o1, c.tag);
        if (hh >= p.n_heads) {
            const bool is_k = hh < p.n_heads + p.n_kv_heads;
            const int kvh = hh - p.n_heads - (is_k ? 0 : p.n_kv_heads);
            kv_t *row = (is_k ? p.kc : p.vc) + (size_t)c.layer * p.layer_kv + ((size_t)kvh * p.max_seq + c.pos) * kHeadDim;
            row[i] = __float2half_rn(o0);
            row[i + 32] = __float2half_rn(o1);
        }
    } else if (ph == PH_GATEUP) {
        ll_store(p.ll_act + u, silu_f(a) * b, c.tag);   // A7: fused SwiGLU
    } else {
        // A9: logits + running packed argmax (lowest index wins ties)
        *reinterpret_cast<float2 *>(p.logits + 2 * u) = make_float2(a, b);
        unsigned long long ka = pack_argmax(a, 2 * u), kb = pack_argmax(b, 2 * u + 1);
        ka = ka > kb ? ka : kb;
        c.best = c.best > ka ? c.best : ka;
    }
}

// One weight phase on the consumer side: input slice -> registers, then stage by stage, no CTA-wide sync.
// ONE instantiation (NCH = 8 covers every slice of <= 256 chunks, shorter slices predicate chunks off) and ONE call site
// (the kernel loops over the phases): inlined into five call sites with four instantiations each the kernel was 352 KB of
// SASS, every phase ran code that was not in the 32 KB instruction cache, and every fetch waited in the same saturated
// memory system as the weights (0.5-1 us per straight-line section, profiles/r01_mega_timeline.md).
template <int NCH, bool TRACE, bool BLOCK>
__device__ __forceinline__ void consume_phase(const MegaParams &p, MkCtx &c, int ph, const PhaseGeom &geo, const uint8_t *ring,
                                           MkShared &sh) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int slice = warp & (geo.S - 1), pair = warp >> geo.log2S;
    const int chunks = geo.K >> 3, c0 = slice * geo.cps;
    const int my_chunks = min(chunks, c0 + geo.cps) - c0;   // may be <= 0 for a ragged tail slice
    const bool resid = (ph == PH_O || ph == PH_DOWN);
    const int n_rows_cta = 2 * (geo.u1 - geo.u0);

    float xr[NCH][8];
    if (BLOCK || geo.K <= kMkStagedK) {   // S == 1: the warp holds the whole vector, staged by run_phase
        load_x_staged<NCH>(sh, my_chunks, xr);
    } else {
        load_x_direct<NCH>(p, c, c0, my_chunks, xr);   // only the down projection has K > kMkStagedK
    }
    mk_trace<TRACE>(p, c);

    unsigned g = c.g;
    MkCtx lc = c;   // registers: c lives in the caller's frame
#pragma unroll 1
    for (int s = 0; s < geo.n_stages; ++s, ++g) {
        const int slot = g % kMkStages;
        const uint32_t par = (g / kMkStages) & 1;
        const int ub = geo.u0 + s * geo.ups;
        const int nu = min(geo.ups, geo.u1 - ub);
        mk_mbar_wait(&sh.full[slot], par, p.err);
        if (s == 0) mk_trace<TRACE>(p, c);
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
                    finish_unit<BLOCK>(p, lc, ph, ub + pair, v, w, sh);
                }
            }
        }
    }
    c.g = g;
    c.best = lc.best;
    if (resid) {
        consumer_sync();
        if (tid < n_rows_cta) {
            float t = c.rold;
#pragma unroll 1
            for (int k = 0; k < geo.S; ++k) t += sh.part[tid][k];
            c.rold = t;
            if (BLOCK) p.x_plain[2 * geo.u0 + tid] = t;   // read by the next kernel
            else ll_store(p.ll_x + (ph == PH_DOWN ? (size_t)p.hidden : 0) + 2 * geo.u0 + tid, t, c.tag);
        }
        // sh.part is next written after the next phase's stage_input (CTA syncs in between)
    }
}

template <bool TRACE, bool BLOCK>
__device__ __forceinline__ void run_phase(const MegaParams &p, MkCtx &c, int ph, const uint8_t *ring, MkShared &sh) {
    const PhaseGeom &geo = sh.geo[ph];
    if (geo.n_stages == 0) {
        mk_trace<TRACE>(p, c); mk_trace<TRACE>(p, c); mk_trace<TRACE>(p, c);
        return;
    }   // no unit of this phase here
    // A6 of layer 0: the residual stream starts as the embedding row; afterwards the owner of a row keeps it in c.rold
    if (ph == PH_O && (int)threadIdx.x < 2 * (geo.u1 - geo.u0)) {
        if (BLOCK) c.rold = ld_act(p.x_plain + 2 * geo.u0 + threadIdx.x);
        else if (c.layer == 0) c.rold = __bfloat162float(p.emb[(size_t)c.tok * p.hidden + 2 * geo.u0 + threadIdx.x]);
    }
    if (BLOCK && ph == PH_O && p.pf_grid > 0) {
        // The memory system idles while this CTA waits for the attention vector: pull the first two weight batches of the
        // gate/up GEMV CTAs 2b, 2b+1 (the next kernel; same unit split as gemv_kernel) into L2, so that its ramp starts
        // from L2 hits.  (A look-ahead like this hurt inside the persistent kernel, where it competes with the stream.)
        const LayerW &w = p.layers[c.layer];
        const int per = p.ffn / p.pf_grid, rem = p.ffn % p.pf_grid;
        for (int g = 2 * (int)blockIdx.x; g < 2 * (int)blockIdx.x + 2 && g < p.pf_grid; ++g) {
            const int u0 = g * per + min(g, rem);
            const int nu = min(p.pf_units, per + (g < rem ? 1 : 0));
            const int lines = p.hidden * 2 / 128;   // 128-byte lines per weight row
            for (int i = threadIdx.x; i < nu * lines; i += kMkConsumers) {
                const size_t off = (size_t)(u0 + i / lines) * p.hidden + (size_t)(i % lines) * 64;
                asm volatile("prefetch.global.L2 [%0];" ::"l"(w.w_gate + off));
                asm volatile("prefetch.global.L2 [%0];" ::"l"(w.w_up + off));
            }
        }
    }
    if (BLOCK || geo.K <= kMkStagedK) stage_input<BLOCK>(p, c, ph, geo.K, sh);
    consume_phase<kMkSliceChunks / 32, TRACE, BLOCK>(p, c, ph, geo, ring, sh);
    mk_trace<TRACE>(p, c);
}

// ---- A5: attention phase ---------------------------------------------------------------------------------------
// Work item of a CTA = (KV head, context split); warp = (query head of the group, sub-split); inside the warp
// lane = (position mod 4, dim octet): 8 lanes share one position (a 128-byte K or V row = 8 x 16 bytes), the score is
// an 8-FMA partial dot product + 3 shuffles, each lane keeps 8 output dims, and the 4 position streams run their own
// online softmax until one 2-shuffle merge at the end.  Compact on purpose: the earlier lane = position variant was
// ~2,000 instructions, and code that falls out of the instruction cache is refetched through the same saturated memory
// system as the weights (see consume_phase).  The K/V rows of earlier positions do not depend on this step, so the
// first batch of 32 positions is loaded BEFORE the warp polls for its query; the row of the current position comes
// from the tagged q/k/v words of this step (rounded to fp16 exactly like the cache row later steps will read).
template <bool TRACE>
__device__ __forceinline__ void attention_phase(const MegaParams &p, MkCtx &c, MkShared &sh) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = p.n_heads / p.n_kv_heads, nsub = kMkConsumerWarps / G;
    const int n_ctx = c.pos + 1;
    const int ns = mk_num_splits(p, n_ctx);
    // att_ctas > 0: the last att_ctas CTAs are set aside for attention; 0: the first CTAs do it besides their weight rows
    const int item = p.att_ctas > 0 ? (int)blockIdx.x - ((int)gridDim.x - p.att_ctas) : (int)blockIdx.x;
    if (item < 0 || item >= p.n_kv_heads * ns) { mk_trace<TRACE>(p, c); mk_trace<TRACE>(p, c); mk_trace<TRACE>(p, c); return; }
    const int len = (n_ctx + ns - 1) / ns;
    const int kvh = item / ns, split = item % ns;
    const int g = warp % G, sub = warp / G;
    const bool active = warp < G * nsub;
    const int head = kvh * G + g;
    const int s0 = split * len, s1 = min(n_ctx, s0 + len);
    const int sub_len = (max(s1 - s0, 0) + nsub - 1) / nsub;
    const int w0 = s0 + sub * sub_len, w1 = min(s1, w0 + sub_len);
    const int oct = lane & 7, grp = lane >> 3;
    const bool has_new = active && c.pos >= w0 && c.pos < w1;   // this warp covers the current position
    const uint4 *kg = reinterpret_cast<const uint4 *>(p.kc + (size_t)c.layer * p.layer_kv + (size_t)kvh * p.max_seq * kHeadDim) + oct;
    const uint4 *vg = reinterpret_cast<const uint4 *>(p.vc + (size_t)c.layer * p.layer_kv + (size_t)kvh * p.max_seq * kHeadDim) + oct;
    const uint4 *kn = reinterpret_cast<const uint4 *>(sh.kvnew[warp][0]) + oct, *vn = reinterpret_cast<const uint4 *>(sh.kvnew[warp][1]) + oct;

    uint4 kk[8], vv[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {   // first batch, cached positions only
        const int t = w0 + 4 * i + grp;
        kk[i] = vv[i] = make_uint4(0, 0, 0, 0);
        if (active && t < w1 && t < c.pos) { kk[i] = __ldcg(kg + (size_t)t * 8); vv[i] = __ldcg(vg + (size_t)t * 8); }
    }
    float q[8], M = -INFINITY, l = 0.f, o[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) { q[j] = 0.f; o[j] = 0.f; }
    if (active) {
        // the lane's octet of the query, pre-scaled by 1/sqrt(64) = 0.125 (exact); with has_new also this step's k and v of
        // the KV head (2 words of each per lane).  One poll loop: every load of a round in flight.
        const llw_t *qsrc = p.ll_qkv + (size_t)head * kHeadDim + oct * 8;
        const llw_t *ksrc = p.ll_qkv + (size_t)(p.n_heads + kvh) * kHeadDim + lane * 2;
        const llw_t *vsrc = ksrc + (size_t)p.n_kv_heads * kHeadDim;
        llw_t wq[8], wk[2], wv[2];
        unsigned spins = 0;
        for (;;) {
#pragma unroll
            for (int j = 0; j < 8; j += 2) ll_load2(qsrc + j, wq[j], wq[j + 1]);
            bool ok = true;
            if (has_new) {
                ll_load2(ksrc, wk[0], wk[1]);
                ll_load2(vsrc, wv[0], wv[1]);
                ok = ll_ok(wk[0], c.tag) && ll_ok(wk[1], c.tag) && ll_ok(wv[0], c.tag) && ll_ok(wv[1], c.tag);
            }
#pragma unroll
            for (int j = 0; j < 8; ++j) ok = ok && ll_ok(wq[j], c.tag);
            if (__all_sync(0xffffffffu, ok)) break;
            if (++spins == kMaxPollSpins) mk_fail(p.err, 6);
            __nanosleep(20);
        }
#pragma unroll
        for (int j = 0; j < 8; ++j) q[j] = 0.125f * ll_val(wq[j]);
        if (has_new) {
            reinterpret_cast<__half2 *>(sh.kvnew[warp][0])[lane] = __floats2half2_rn(ll_val(wk[0]), ll_val(wk[1]));
            reinterpret_cast<__half2 *>(sh.kvnew[warp][1])[lane] = __floats2half2_rn(ll_val(wv[0]), ll_val(wv[1]));
        }
        __syncwarp();
    }
    mk_trace<TRACE>(p, c);
    if (active) {
        float m = -INFINITY;
#pragma unroll 1
        for (int b0 = w0; b0 < w1; b0 += 32) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int t = b0 + 4 * i + grp;
                if (t < w1 && t == c.pos) { kk[i] = *kn; vv[i] = *vn; }
                else if (b0 != w0 && t < w1) { kk[i] = __ldcg(kg + (size_t)t * 8); vv[i] = __ldcg(vg + (size_t)t * 8); }
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int t = b0 + 4 * i + grp;
                const float2 k0 = h2f(kk[i].x), k1 = h2f(kk[i].y), k2 = h2f(kk[i].z), k3 = h2f(kk[i].w);
                float s = q[0] * k0.x;
                s = fmaf(q[1], k0.y, s); s = fmaf(q[2], k1.x, s); s = fmaf(q[3], k1.y, s);
                s = fmaf(q[4], k2.x, s); s = fmaf(q[5], k2.y, s); s = fmaf(q[6], k3.x, s); s = fmaf(q[7], k3.y, s);
                s += __shfl_xor_sync(0xffffffffu, s, 1);
                s += __shfl_xor_sync(0xffffffffu, s, 2);
                s += __shfl_xor_sync(0xffffffffu, s, 4);
                if (t < w1) {
                    const float m_new = fmaxf(m, s);
                    const float corr = __expf(m - m_new);   // m = -inf the first time -> 0
                    const float pr = __expf(s - m_new);
                    const float2 v0 = h2f(vv[i].x), v1 = h2f(vv[i].y), v2 = h2f(vv[i].z), v3 = h2f(vv[i].w);
                    l = l * corr + pr;
                    o[0] = fmaf(pr, v0.x, o[0] * corr); o[1] = fmaf(pr, v0.y, o[1] * corr);
                    o[2] = fmaf(pr, v1.x, o[2] * corr); o[3] = fmaf(pr, v1.y, o[3] * corr);
                    o[4] = fmaf(pr, v2.x, o[4] * corr); o[5] = fmaf(pr, v2.y, o[5] * corr);
                    o[6] = fmaf(pr, v3.x, o[6] * corr); o[7] = fmaf(pr, v3.y, o[7] * corr);
                    m = m_new;
                }
            }
        }
        // merge the 4 position streams of the warp
        M = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 8));
        M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, 16));
        const float sc = (m == -INFINITY) ? 0.f : __expf(m - M);
        l *= sc;
        l += __shfl_xor_sync(0xffffffffu, l, 8);
        l += __shfl_xor_sync(0xffffffffu, l, 16);
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            o[j] *= sc;
            o[j] += __shfl_xor_sync(0xffffffffu, o[j], 8);
            o[j] += __shfl_xor_sync(0xffffffffu, o[j], 16);
        }
        if (sub > 0 && lane < 8) {   // park the state for the sub-split 0 warp of this head
#pragma unroll
            for (int j = 0; j < 8; ++j) sh.mrg[warp][oct * 8 + j] = o[j];
            if (lane == 0) { sh.mrg[warp][kHeadDim] = M; sh.mrg[warp][kHeadDim + 1] = l; }
        }
    }
    mk_trace<TRACE>(p, c);
    if (nsub > 1) consumer_sync();
    if (active && sub == 0) {
        // every lane: the CTA's state of (head, octet) = its own plus the parked sub-splits
#pragma unroll 1
        for (int k = 1; k < nsub; ++k) {
            const float *o2 = sh.mrg[k * G + g];
            const float M2 = o2[kHeadDim], l2 = o2[kHeadDim + 1];
            const float Mn = fmaxf(M, M2);
            const float wa = (M == -INFINITY) ? 0.f : __expf(M - Mn), wb = (M2 == -INFINITY) ? 0.f : __expf(M2 - Mn);
            l = l * wa + l2 * wb;
#pragma unroll
            for (int j = 0; j < 8; ++j) o[j] = o[j] * wa + o2[oct * 8 + j] * wb;
            M = Mn;
        }
        const size_t pidx = (size_t)head * kMkMaxSplits + split;
        if (ns > 1 && split > 0) {
            // split state (unnormalised) as tagged words for the CTA of split 0 of this KV head
            if (lane < 8) {
#pragma unroll
                for (int j = 0; j < 8; ++j) ll_store(p.ll_part_o + pidx * kHeadDim + oct * 8 + j, o[j], c.tag);
                if (lane == 0) {
                    ll_store(p.ll_part_ml + pidx * 2, M, c.tag);
                    ll_store(p.ll_part_ml + pidx * 2 + 1, l, c.tag);
                }
            }
        } else {
            // Split 0 merges the other splits of its heads (second level: the ~3 KB it reads are nothing next to every
            // CTA of the chip reading every split state, 12 MB of L2 reads per layer = 3.5 us in one poll round) and
            // publishes the final, normalised attention output: the O phase of every CTA polls 8 words per thread.
            // Lane group j (8 lanes) takes splits j, j + 4 (group 0: its own state and split 4).
            if (grp > 0) {
                M = -INFINITY; l = 0.f;
#pragma unroll
                for (int j = 0; j < 8; ++j) o[j] = 0.f;
            }
#pragma unroll 1
            for (int r4 = 0; r4 < kMkMaxSplits; r4 += 4) {   // warp-uniform trip count: the poll below votes across the warp
                const int s = r4 + grp;
                const bool mine = s >= 1 && s < ns;
                if (!__any_sync(0xffffffffu, mine)) break;
                const size_t q2 = (size_t)head * kMkMaxSplits + (mine ? s : 0);
                llw_t wm[2], wo[8];
                unsigned spins = 0;
                for (;;) {
                    bool ok = true;
                    if (mine) {
                        ll_load2(p.ll_part_ml + q2 * 2, wm[0], wm[1]);
#pragma unroll
                        for (int j = 0; j < 8; j += 2) ll_load2(p.ll_part_o + q2 * kHeadDim + oct * 8 + j, wo[j], wo[j + 1]);
                        ok = ll_ok(wm[0], c.tag) && ll_ok(wm[1], c.tag);
#pragma unroll
                        for (int j = 0; j < 8; ++j) ok = ok && ll_ok(wo[j], c.tag);
                    }
                    if (__all_sync(0xffffffffu, ok)) break;
                    if (++spins == kMaxPollSpins) mk_fail(p.err, 9);
                    __nanosleep(20);
                }
                if (mine) {
                    const float M2 = ll_val(wm[0]), l2 = ll_val(wm[1]);
                    const float Mn = fmaxf(M, M2);
                    const float wa = (M == -INFINITY) ? 0.f : __expf(M - Mn), wb = (M2 == -INFINITY) ? 0.f : __expf(M2 - Mn);
                    l = l * wa + l2 * wb;
#pragma unroll
                    for (int j = 0; j < 8; ++j) o[j] = o[j] * wa + ll_val(wo[j]) * wb;
                    M = Mn;
                }
            }
            // merge the 4 lane groups
            float Mg = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, 8));
            Mg = fmaxf(Mg, __shfl_xor_sync(0xffffffffu, Mg, 16));
            const float sg = (M == -INFINITY) ? 0.f : __expf(M - Mg);
            l *= sg;
            l += __shfl_xor_sync(0xffffffffu, l, 8);
            l += __shfl_xor_sync(0xffffffffu, l, 16);
            const float inv = 1.0f / l;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                o[j] *= sg;
                o[j] += __shfl_xor_sync(0xffffffffu, o[j], 8);
                o[j] += __shfl_xor_sync(0xffffffffu, o[j], 16);
            }
            if (lane < 8) {
#pragma unroll
                for (int j = 0; j < 8; ++j) ll_store(p.ll_attn + (size_t)head * kHeadDim + oct * 8 + j, o[j] * inv, c.tag);
            }
        }
    }
    mk_trace<TRACE>(p, c);
    // sh.kvnew / sh.mrg are next written in the next layer's attention, CTA syncs (stage_input) in between
}

// ---- the kernel -----------------------------------------------------------------------------------------------
template <bool TRACE, bool BLOCK>
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
    if (tid < 5) sh.geo[tid] = phase_geom(p, tid);
    __syncthreads();

    if (warp == kMkConsumerWarps) {
        if ((tid & 31) == 0) mk_producer(p, ring, sh);
        return;
    }

    // Attention-block launches sit between per-step kernels with programmatic edges: the producer warp (above) is already
    // streaming this launch's weights (immutable), everything else waits for the previous kernel here.
    MkCtx c;
    c.gain_pre = make_uint4(0, 0, 0, 0);
    if (BLOCK && tid * 8 < p.hidden)   // immutable like the weights: its HBM latency overlaps the previous kernel's tail
        c.gain_pre = __ldg(reinterpret_cast<const uint4 *>(p.layers[p.pi_begin >> 2].attn_norm) + tid);
    pdl_launch_dependents();
    pdl_wait();
    c.g = 0;
    c.best = 0ull;
    c.ti = 0;
    c.rold = 0.f;
    c.pos = ld_act(p.pos);
    c.tok = ld_act(p.tok_src);
    // Steps run by earlier launches.  Written only by CTA 0 at its exit, which needs a result of this step from every
    // CTA, i.e. after every CTA has read it here.
    const uint32_t epoch0 = *reinterpret_cast<volatile unsigned int *>(p.epoch);
    mk_trace<TRACE>(p, c);
    for (int step = 0; step < p.n_steps; ++step) {
        if (tid < 32) sh.rope[tid] = p.rope[(size_t)c.pos * 32 + tid];
        consumer_sync();
        const uint32_t tag0 = (epoch0 + (uint32_t)step) * (uint32_t)(p.n_layers + 1) + 1u;   // >= 1: zeroed buffers never match
        const int n_ph = p.n_layers * 4 + (p.with_head ? 1 : 0);
        const int pi0 = BLOCK ? p.pi_begin : 0, pi1 = BLOCK ? p.pi_end : n_ph;
#pragma unroll 1
        for (int pi = pi0; pi < pi1; ++pi) {   // a loop, not straight-line code: one copy of every phase body (see consume_phase)
            c.layer = pi >> 2;
            const int ph = BLOCK ? (pi & 1 ? PH_O : PH_QKV) : (c.layer < p.n_layers ? (pi & 3) : PH_HEAD);
            c.tag = tag0 + (uint32_t)c.layer;
            c.tag_prev = c.tag - 1u;
            if (ph == PH_HEAD) c.best = 0ull;
            run_phase<TRACE, BLOCK>(p, c, ph, ring, sh);
            if (ph == PH_QKV) attention_phase<TRACE>(p, c, sh);
        }
        if (BLOCK) break;   // attention-block launch: one step, no head, position advanced by the LM-head kernel
        c.tag_prev = tag0 + (uint32_t)(p.n_layers - 1);
        c.tag = tag0 + (uint32_t)p.n_layers;
        if (p.with_head) {
            // A9: every CTA publishes its best (ordered logit key, index) as two tagged words; every CTA then polls all of
            // them and takes the maximum = the next token (lowest index wins ties: the packing orders ~index).
            if ((tid & 31) == 0) sh.wbest[warp] = c.best;   // lane 0 ran every epilogue of its warp
            consumer_sync();
            if (tid == 0) {
                unsigned long long b = sh.wbest[0];
                for (int k = 1; k < kMkConsumerWarps; ++k) b = b > sh.wbest[k] ? b : sh.wbest[k];
                ll_store_u32(p.ll_best + 2 * blockIdx.x, (uint32_t)(b >> 32), c.tag);
                ll_store_u32(p.ll_best + 2 * blockIdx.x + 1, (uint32_t)b, c.tag);
            }
            unsigned long long mine = 0ull;
#pragma unroll 1
            for (int i = tid; i < (int)gridDim.x; i += kMkConsumers) {
                llw_t a, b;
                unsigned spins = 0;
                for (;;) {
                    ll_load2(p.ll_best + 2 * i, a, b);
                    if (ll_ok(a, c.tag) && ll_ok(b, c.tag)) break;
                    if (++spins == kMaxPollSpins) mk_fail(p.err, 7);
                __nanosleep(20);
                }
                const unsigned long long v = ((a & 0xFFFFFFFFull) << 32) | (b & 0xFFFFFFFFull);
                mine = mine > v ? mine : v;
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const unsigned long long other = __shfl_xor_sync(0xffffffffu, mine, o);
                mine = mine > other ? mine : other;
            }
            consumer_sync();   // everyone has read sh.wbest above
            if ((tid & 31) == 0) sh.wbest[warp] = mine;
            consumer_sync();
            unsigned long long win = sh.wbest[0];
#pragma unroll
            for (int k = 1; k < kMkConsumerWarps; ++k) win = win > sh.wbest[k] ? win : sh.wbest[k];
            c.tok = unpack_argmax_idx(win);
            mk_trace<TRACE>(p, c);
            if (blockIdx.x == 0 && tid == 0) {
                *p.cur_tok = c.tok;
                p.tok_hist[c.pos + 1] = c.tok;
                *p.pos = c.pos + 1;
            }
        } else {
            // without the head the kernel runs one step (hq_prefill token walk)
            if (blockIdx.x == 0) {
                if (p.hidden_out && tid * 8 < p.hidden) {   // parity capture of the last layer
                    float v[8];
                    ll_poll<8>(p.ll_x + (size_t)p.hidden + (size_t)tid * 8, c.tag_prev, v, p.err);
                    float4 *dst = reinterpret_cast<float4 *>(p.hidden_out + (size_t)(p.n_layers - 1) * p.hidden_stride + tid * 8);
                    dst[0] = make_float4(v[0], v[1], v[2], v[3]);
                    dst[1] = make_float4(v[4], v[5], v[6], v[7]);
                }
                if (tid == 0) *p.pos = c.pos + 1;
            }
            c.tok = 0;
        }
        c.pos += 1;
    }
    if (blockIdx.x == 0 && tid == 0) *p.epoch = epoch0 + (uint32_t)p.n_steps;
}

// ---- host side ---------------------------------------------------------------------------------------------------
size_t mega_smem_bytes() { return (size_t)kMkStages * kMkStageBytes + sizeof(MkShared) + 128; }

size_t mega_ll_words(const hq_config &c) {
    const size_t H = c.n_heads, Hkv = c.n_kv_heads;
    return 2 * (size_t)c.hidden + (H + 2 * Hkv) * kHeadDim + (size_t)c.ffn + H * kMkMaxSplits * kHeadDim + H * kMkMaxSplits * 2 + H * kHeadDim +
           2 * (size_t)kMkMaxGrid;
}

// Most context splits per KV head a model will use = attention CTAs set aside per KV head: enough for max_ctx at two
// 32-position batch per warp, at most kMkMaxSplits and half of the SMs.
int mega_att_splits(const hq_config &c, int n_sms, int max_ctx) {
    const int G = c.n_heads / c.n_kv_heads, nsub = kMkConsumerWarps / (G > 0 ? G : 1);
    const int per = 32 * (nsub > 0 ? nsub : 1);
    int ns = (max_ctx + per - 1) / per;
    int cap = (n_sms / 2) / c.n_kv_heads;
    if (cap < 1) cap = 1;
    if (cap > kMkMaxSplits) cap = kMkMaxSplits;
    if (ns > cap) ns = cap;
    return ns < 1 ? 1 : ns;
}

bool mega_shape_supported(const hq_config &c, int n_sms) {
    // staged phases keep the whole vector in one warp (hidden, q <= 2048); the down projection cuts K into <= 8 slices;
    // the residual rows of one CTA must fit the partial buffer; the group must fit the consumer warps
    const int q = c.n_heads * c.head_dim;
    const int w_ctas = n_sms - mega_att_splits(c, n_sms, 1 << 30) * c.n_kv_heads;
    const int units_cta = (c.hidden / 2 + w_ctas - 1) / w_ctas;   // fewest weight CTAs a launch can have
    return c.hidden <= kMkStagedK && q <= kMkStagedK && c.ffn <= 32 * kMkSliceChunks &&
           2 * units_cta <= kMkPartRows && c.n_heads / c.n_kv_heads <= kMkConsumerWarps && c.hidden % 8 == 0 &&
           c.ffn % 8 == 0 && c.vocab % 2 == 0 && n_sms >= 2 * c.n_kv_heads && n_sms <= kMkMaxGrid && w_ctas >= 1;
}

cudaError_t launch_mega(const LaunchCtx &c, const MegaParams &p, bool cooperative) {
    static bool attr_done = false;
    const size_t smem = mega_smem_bytes();
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(mega_decode_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(mega_decode_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(mega_decode_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(mega_decode_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(c.n_sms);
    cfg.blockDim = dim3(kMkThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = c.stream;
    // cooperative: the driver guarantees (and checks) that all CTAs are co-resident — the CTAs wait on one another
    cudaLaunchAttribute attr[1];
    cfg.attrs = attr;
    if (p.x_plain) {
        // one CTA per SM (shared memory) and no dependence of the neighbouring kernels on this one's CTAs: all CTAs become
        // resident as the previous kernel drains; a programmatic edge lets the weight stream start under its tail
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.numAttrs = c.pdl ? 1 : 0;
    } else {
        attr[0].id = cudaLaunchAttributeCooperative;
        attr[0].val.cooperative = 1;
        cfg.numAttrs = cooperative ? 1 : 0;
    }
    // the timeline stamps live in their own instantiation: the production kernel's code has to stay small
    // ... and so does the attention block (its per-launch path has to stay resident in the instruction cache between
    // launches: everything it does not need is compiled out)
    if (p.x_plain) return p.trace ? cudaLaunchKernelEx(&cfg, mega_decode_kernel<true, true>, p) : cudaLaunchKernelEx(&cfg, mega_decode_kernel<false, true>, p);
    return p.trace ? cudaLaunchKernelEx(&cfg, mega_decode_kernel<true, false>, p) : cudaLaunchKernelEx(&cfg, mega_decode_kernel<false, false>, p);
}

}  // namespace hq
