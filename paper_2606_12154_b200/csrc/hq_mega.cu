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
constexpr int kMkPartRows = 64;                   // residual rows of one CTA in one phase (2 * units)
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
    float part[kMkPartRows][kMkConsumerWarps];   // residual phases: [row of this CTA][slice] partial sums
    float2 rope[32];
    float q[8][kHeadDim];                        // pre-scaled queries of the group
    float mrg[kMkConsumerWarps][kHeadDim + 2];   // attention: sub-split states (o[64], m, l)
    unsigned long long wbest[kMkConsumerWarps];  // LM head: per-warp packed argmax
    int flag;
};

// ---- producer ----------------------------------------------------------------------------------------------
__device__ void mk_producer(const MegaParams &p, uint8_t *ring, MkShared &sh) {
    unsigned g = 0;   // stages produced so far
    for (int step = 0; step < p.n_steps; ++step) {
        const int n_ph = p.n_layers * 4 + (p.with_head ? 1 : 0);
        for (int pi = 0; pi < n_ph; ++pi) {
            const int layer = pi >> 2;
            const int ph = layer < p.n_layers ? (pi & 3) : PH_HEAD;
            const LayerW &w = p.layers[layer < p.n_layers ? layer : 0];
            const PhaseGeom geo = phase_geom(p, ph);
            for (int s = 0; s < geo.n_stages; ++s, ++g) {
                const int slot = g % kMkStages;
                const uint32_t par = (g / kMkStages) & 1;
                mk_mbar_wait(&sh.empty[slot], par ^ 1, p.err);
                const int ub = geo.u0 + s * geo.ups;
                const int nu = min(geo.ups, geo.u1 - ub);
                mk_mbar_expect_tx(&sh.full[slot], (uint32_t)(2 * nu * geo.row_bytes));
                uint8_t *dst = ring + (size_t)slot * kMkStageBytes;
                for (int j = 0; j < nu; ++j) {
                    const bf16 *ra, *rb;
                    unit_row_ptrs(p, w, ph, geo.K, ub + j, ra, rb);
                    mk_bulk_g2s(dst + (size_t)(2 * j) * geo.row_bytes, ra, geo.row_bytes, &sh.full[slot]);
                    mk_bulk_g2s(dst + (size_t)(2 * j + 1) * geo.row_bytes, rb, geo.row_bytes, &sh.full[slot]);
                }
            }
        }
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

// Phase input slice -> registers.  Lane owns chunks (8 elements) c0 + j*32 + lane, j < NCH, of the row.
// Phases with a fused RMSNorm (A2) have S == 1 (hidden <= 2048): the warp holds the whole vector, so the sum of
// squares is one warp reduction, recomputed by every warp (deterministic, no atomics).
template <int NCH>
__device__ __forceinline__ void load_x(const MegaParams &p, const MkCtx &c, int ph, int K, int c0, int my_chunks,
                                       float (&xr)[NCH][8]) {
    const int lane = threadIdx.x & 31;
    const bool norm = (ph == PH_QKV || ph == PH_GATEUP || ph == PH_HEAD);
    const bool from_emb = (ph == PH_QKV && c.layer == 0);
    const float *src = ph == PH_O ? p.attn_out : (ph == PH_DOWN ? p.act : p.x);
    float ss = 0.f;
#pragma unroll
    for (int j = 0; j < NCH; ++j) {
        const int ch = j * 32 + lane;
        if (ch < my_chunks) {
            if (from_emb) {
                const uint4 e = __ldg(reinterpret_cast<const uint4 *>(p.emb + (size_t)c.tok * p.hidden) + c0 + ch);
                xr[j][0] = bf16lo(e.x); xr[j][1] = bf16hi(e.x); xr[j][2] = bf16lo(e.y); xr[j][3] = bf16hi(e.y);
                xr[j][4] = bf16lo(e.z); xr[j][5] = bf16hi(e.z); xr[j][6] = bf16lo(e.w); xr[j][7] = bf16hi(e.w);
            } else {
                const float4 a = ld_act4(src + (size_t)(c0 + ch) * 8), b = ld_act4(src + (size_t)(c0 + ch) * 8 + 4);
                xr[j][0] = a.x; xr[j][1] = a.y; xr[j][2] = a.z; xr[j][3] = a.w;
                xr[j][4] = b.x; xr[j][5] = b.y; xr[j][6] = b.z; xr[j][7] = b.w;
            }
        } else {
#pragma unroll
            for (int i = 0; i < 8; ++i) xr[j][i] = 0.f;
        }
    }
    if (norm) {
        const bf16 *gain = ph == PH_QKV ? p.layers[c.layer].attn_norm : (ph == PH_GATEUP ? p.layers[c.layer].ffn_norm : p.final_norm);
        uint4 gq[NCH];
#pragma unroll
        for (int j = 0; j < NCH; ++j) {
            const int ch = j * 32 + lane;
            gq[j] = ch < my_chunks ? __ldg(reinterpret_cast<const uint4 *>(gain) + c0 + ch) : make_uint4(0, 0, 0, 0);
#pragma unroll
            for (int i = 0; i < 8; ++i) ss = fmaf(xr[j][i], xr[j][i], ss);
        }
        ss = warp_sum(ss);
        const float inv = 1.0f / sqrtf(ss / (float)K + p.eps);
#pragma unroll
        for (int j = 0; j < NCH; ++j) {
            const uint32_t gg[4] = {gq[j].x, gq[j].y, gq[j].z, gq[j].w};
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                xr[j][2 * i] *= inv * bf16lo(gg[i]);
                xr[j][2 * i + 1] *= inv * bf16hi(gg[i]);
            }
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
    load_x<NCH>(p, c, ph, geo.K, c0, my_chunks, xr);
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
// attention split policy (device only; a function of the context length and the grid): one 32-position
// iteration per warp while the grid has CTAs to spare, then longer splits
__device__ __forceinline__ int mk_num_splits(const MegaParams &p, int n_ctx, int nsub) {
    int ns_max = (int)gridDim.x / p.n_kv_heads;
    ns_max = ns_max < 1 ? 1 : (ns_max > kMkMaxSplits ? kMkMaxSplits : ns_max);
    const int per = 32 * nsub;
    const int want = (n_ctx + per - 1) / per;
    return want < ns_max ? want : ns_max;
}

__device__ void attention_phase(const MegaParams &p, MkCtx &c, MkShared &sh) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = p.n_heads / p.n_kv_heads;
    const int nsub = kMkConsumerWarps / G;
    const int n_ctx = c.pos + 1;
    const int ns = mk_num_splits(p, n_ctx, nsub);
    const int len = (n_ctx + ns - 1) / ns;
    const int items = p.n_kv_heads * ns;
    const size_t layer_off = (size_t)c.layer * p.layer_kv;

    for (int item = blockIdx.x; item < items; item += gridDim.x) {
        const int kvh = item / ns, split = item % ns;
        const int s0 = split * len, s1 = min(n_ctx, s0 + len);
        // stage the group's queries, pre-scaled by 1/sqrt(64) = 0.125 (exact)
        for (int i = tid; i < G * kHeadDim; i += kMkConsumers)
            sh.q[i >> 6][i & 63] = 0.125f * ld_act(p.qkv + (size_t)(kvh * G) * kHeadDim + i);
        consumer_sync();
        if (item == (int)blockIdx.x) mk_trace(p, c);

        const bool active = warp < G * nsub;
        const int g = warp % G, sub = warp / G;
        const int head = kvh * G + g;
        const int r = warp_row_of_lane<32>(lane);   // the output dims (r, 32 + r) this lane holds after the merge
        float M = -INFINITY, l_tot = 0.f, o_lo = 0.f, o_hi = 0.f;
        if (active) {
            const int sub_len = (s1 - s0 + nsub - 1) / nsub;
            const int w0 = s0 + sub * sub_len, w1 = min(s1, w0 + sub_len);
            const kv_t *kg = p.kc + layer_off + (size_t)kvh * p.max_seq * kHeadDim;
            const kv_t *vg = p.vc + layer_off + (size_t)kvh * p.max_seq * kHeadDim;
            const float4 *q4 = reinterpret_cast<const float4 *>(sh.q[g]);

            float m = -INFINITY, l = 0.f, o[kHeadDim];
#pragma unroll
            for (int d = 0; d < kHeadDim; ++d) o[d] = 0.f;
            for (int t = w0 + lane; t < w1; t += 32) {
                KvRow kr, vr;
                ld_kv_row(kr, kg + (size_t)t * kHeadDim);
                ld_kv_row(vr, vg + (size_t)t * kHeadDim);
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
            if (sub > 0) {   // park the state for the sub-split 0 warp of this head
                sh.mrg[warp][r] = o_lo;
                sh.mrg[warp][32 + r] = o_hi;
                if (lane == 0) { sh.mrg[warp][kHeadDim] = M; sh.mrg[warp][kHeadDim + 1] = l_tot; }
            }
        }
        if (nsub > 1) consumer_sync();
        if (active && sub == 0) {
            for (int k = 1; k < nsub; ++k) {
                const float *o2 = sh.mrg[k * G + g];
                const float M2 = o2[kHeadDim], l2 = o2[kHeadDim + 1];
                const float Mn = fmaxf(M, M2);
                const float wa = (M == -INFINITY) ? 0.f : __expf(M - Mn), wb = (M2 == -INFINITY) ? 0.f : __expf(M2 - Mn);
                l_tot = l_tot * wa + l2 * wb;
                o_lo = o_lo * wa + o2[r] * wb;
                o_hi = o_hi * wa + o2[32 + r] * wb;
                M = Mn;
            }
            if (ns == 1) {   // the whole context in one CTA: final
                const float inv = 1.0f / l_tot;
                p.attn_out[head * kHeadDim + r] = o_lo * inv;
                p.attn_out[head * kHeadDim + 32 + r] = o_hi * inv;
            } else {
                const size_t pidx = (size_t)head * kMkMaxSplits + split;
                p.part_o[pidx * kHeadDim + r] = o_lo;
                p.part_o[pidx * kHeadDim + 32 + r] = o_hi;
                if (lane == 0) p.part_ml[pidx] = make_float2(M, l_tot);
            }
        }
        if (item == (int)blockIdx.x) mk_trace(p, c);
        if (ns > 1) {
            // the last CTA of this KV head merges the split partials (fixed slot order: deterministic)
            consumer_sync();
            if (tid == 0) {
                __threadfence();
                const unsigned t = atomicAdd(p.kv_ticket + kvh, 1u);
                sh.flag = (t == (unsigned)ns - 1u);
                if (sh.flag) {
                    p.kv_ticket[kvh] = 0u;
                    __threadfence();
                }
            }
            consumer_sync();
            if (sh.flag) {
                for (int i = tid; i < G * kHeadDim; i += kMkConsumers) {
                    const int hd = kvh * G + (i >> 6), d = i & 63;
                    const float2 *ml = p.part_ml + (size_t)hd * kMkMaxSplits;
                    float Mx = -INFINITY;
                    for (int s = 0; s < ns; ++s) Mx = fmaxf(Mx, __ldcg(&ml[s]).x);
                    float acc = 0.f, den = 0.f;
                    for (int s = 0; s < ns; ++s) {
                        const float2 v = __ldcg(&ml[s]);
                        const float wgt = (v.x == -INFINITY) ? 0.f : __expf(v.x - Mx);
                        den = fmaf(wgt, v.y, den);
                        acc = fmaf(wgt, __ldcg(p.part_o + ((size_t)hd * kMkMaxSplits + s) * kHeadDim + d), acc);
                    }
                    p.attn_out[hd * kHeadDim + d] = acc / den;
                }
            }
        }
        consumer_sync();   // sh.q / sh.mrg / sh.flag are reused by the next item
    }
    if ((int)blockIdx.x >= items) { mk_trace(p, c); mk_trace(p, c); }
    mk_trace(p, c);
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
            grid_barrier(p, c);
            attention_phase(p, c, sh);
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
    return c.hidden <= 8 * kMkSliceChunks && q <= 64 * kMkSliceChunks && c.ffn <= 64 * kMkSliceChunks &&
           2 * units_cta <= kMkPartRows && c.n_heads / c.n_kv_heads <= kMkConsumerWarps && c.hidden % 8 == 0 &&
           c.ffn % 8 == 0 && c.vocab % 2 == 0 && n_sms >= 1;
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
