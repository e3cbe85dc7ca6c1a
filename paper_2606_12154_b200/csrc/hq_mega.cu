// hq_mega.cu — persistent batch-1 decode: SURVEY.md §8(a) rows A1-A9 for n_steps tokens in ONE launch.
//
// Why: one token is a chain of 81 HBM-bound matrix-vector products over 2.47 GB of bf16 weights.  With one
// kernel per product the three small products of every layer (QKV, attention, O) cost more in kernel-boundary
// latency than in DRAM time (profiles/r01_decode_launches_v1.md: 53 % of the copy peak).  Here the weight
// stream never stops:
//   * grid = one CTA per SM, 9 warps.  Warp 8 is the PRODUCER: one elected thread walks the static schedule
//     (layer, phase, this CTA's rows) and streams every weight row with cp.async.bulk (TMA bulk copy,
//     mbarrier complete_tx) into a ring of kMkStages x 32 KB shared-memory stages.  Weights are immutable, so
//     the producer runs ahead of the phase barriers — while the consumers wait for the other SMs, do the
//     attention, or reduce, the next phases' rows are already landing.
//   * warps 0-7 are CONSUMERS: the (normalised) input vector of the phase lives in registers, a stage holds
//     R = 2, 4 or 8 rows (a "unit" = 2 rows: RoPE pair / gate+up pair / two adjacent rows), 8/R warps per row,
//     conflict-free 16-byte shared loads, fp32 FMA, warp-shuffle reduction, fused epilogues (RoPE, SwiGLU,
//     residual add, logits + packed argmax).
//   * phases are separated by a grid barrier (one release-add + acquire-poll on a global counter): per layer
//     QKV | attention | O | gate/up | down, then the LM head.  The token and the position stay on the device;
//     the kernel loops over n_steps tokens (hq_decode_run) so there is no launch gap between tokens either.
//   * attention: work item = (KV head, split); warp = (query head of the group, sub-split); LANE = POSITION:
//     every lane runs its own online softmax over its positions (K/V rows are one 128-byte line each, read
//     with 256-bit loads), then the 32 lane states are merged with a transposed butterfly.  The last CTA of a
//     KV head (ticket) merges the split partials, so the O phase reads a plain vector.  The new K/V row is
//     appended by the CTA that owns the last split, from the fp32 scratch the QKV phase wrote.
#include "hq_common.cuh"
#include "hq_internal.h"

namespace hq {

constexpr int kMkConsumerWarps = 8;
constexpr int kMkConsumers = 32 * kMkConsumerWarps;
constexpr int kMkThreads = kMkConsumers + 32;
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
// one 128-byte K or V row (64 fp16) of a cache position: read-only for the life of the kernel
struct KvRow { uint4 v[8]; };
__device__ __forceinline__ void ld_kv_row(KvRow &r, const kv_t *p) {
#pragma unroll
    for (int j = 0; j < 4; ++j)
        asm volatile("ld.global.nc.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                     : "=r"(r.v[2 * j].x), "=r"(r.v[2 * j].y), "=r"(r.v[2 * j].z), "=r"(r.v[2 * j].w),
                       "=r"(r.v[2 * j + 1].x), "=r"(r.v[2 * j + 1].y), "=r"(r.v[2 * j + 1].z), "=r"(r.v[2 * j + 1].w)
                     : "l"(p + 16 * j));
}
__device__ __forceinline__ float2 h2f(uint32_t u) { return __half22float2(*reinterpret_cast<const __half2 *>(&u)); }

// ---- static schedule shared by producer and consumers -----------------------------------------------------
struct PhaseGeom {
    int K, row_bytes;
    int u0, u1;        // this CTA's units [u0, u1)
    int ups;           // units per stage (1, 2 or 4): a stage holds 2*ups rows
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
    const int n = phase_units(p, ph), per = n / gridDim.x, rem = n % gridDim.x, b = blockIdx.x;
    g.u0 = b * per + min(b, rem);
    g.u1 = g.u0 + per + (b < rem ? 1 : 0);
    const int fit = kMkStageBytes / (2 * g.row_bytes);
    g.ups = fit >= 4 ? 4 : (fit >= 2 ? 2 : 1);
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

// attention split policy (device only; a function of the context length and the grid)
__device__ __forceinline__ int mk_num_splits(const MegaParams &p, int n_ctx) {
    int ns_max = (int)gridDim.x / p.n_kv_heads;
    ns_max = ns_max < 1 ? 1 : (ns_max > kMkMaxSplits ? kMkMaxSplits : ns_max);
    const int want = (n_ctx + 15) >> 4;   // at least 16 positions per split
    return want < ns_max ? want : ns_max;
}

struct MkShared {
    uint64_t full[kMkStages], empty[kMkStages];
    float partial[2][kMkConsumerWarps];
    float2 rope[32];
    float q[8][kHeadDim];                 // pre-scaled queries of the group
    alignas(16) __half knew[kHeadDim];    // this step's K/V row of the KV head, fp16-rounded
    alignas(16) __half vnew[kHeadDim];
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
    unsigned long long best;
};

__device__ __forceinline__ void grid_barrier(const MegaParams &p, MkCtx &c) {
    consumer_sync();   // every consumer's global stores of this phase are issued
    if (threadIdx.x == 0) {
        c.bar_target += gridDim.x;
        __threadfence();
        red_release_add(p.bar, 1u);
        const long long t0 = clock64();
        unsigned spins = 0;
        while ((int)(ld_acquire_u32(p.bar) - c.bar_target) < 0)
            if ((++spins & 1023u) == 0 && clock64() - t0 > kSpinCycles) mk_fail(p.err, 2);
        __threadfence();
    }
    consumer_sync();
}

// residual stream value i: the embedding row of the token before layer 0's O projection, x afterwards
__device__ __forceinline__ float2 resid2(const MegaParams &p, const MkCtx &c, bool from_emb, int i) {
    if (from_emb) {
        const uint32_t u = __ldg(reinterpret_cast<const uint32_t *>(p.emb + (size_t)c.tok * p.hidden + i));
        return make_float2(bf16lo(u), bf16hi(u));
    }
    return __ldcg(reinterpret_cast<const float2 *>(p.x + i));
}

// Phase input vector -> registers.  Lane owns chunks (8 elements) ks*cpw + j*32 + lane, j < NCH, of the row.
template <int NCH>
__device__ __forceinline__ void load_x(const MegaParams &p, const MkCtx &c, int ph, int K, int wpr, float (&xr)[NCH][8]) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int chunks = K >> 3, cpw = (chunks + wpr - 1) / wpr, ks = warp % wpr;
    const int c_end = min(chunks, (ks + 1) * cpw);
    const bool norm = (ph == PH_QKV || ph == PH_GATEUP || ph == PH_HEAD);
    const bool from_emb = (ph == PH_QKV && c.layer == 0);
    const float *src = ph == PH_O ? p.attn_out : (ph == PH_DOWN ? p.act : p.x);
    float ss = 0.f;
#pragma unroll
    for (int j = 0; j < NCH; ++j) {
        const int ch = ks * cpw + j * 32 + lane;
        if (ch < c_end) {
            if (from_emb) {
                const uint4 e = __ldg(reinterpret_cast<const uint4 *>(p.emb + (size_t)c.tok * p.hidden) + ch);
                xr[j][0] = bf16lo(e.x); xr[j][1] = bf16hi(e.x); xr[j][2] = bf16lo(e.y); xr[j][3] = bf16hi(e.y);
                xr[j][4] = bf16lo(e.z); xr[j][5] = bf16hi(e.z); xr[j][6] = bf16lo(e.w); xr[j][7] = bf16hi(e.w);
            } else {
                const float4 a = ld_act4(src + ch * 8), b = ld_act4(src + ch * 8 + 4);
                xr[j][0] = a.x; xr[j][1] = a.y; xr[j][2] = a.z; xr[j][3] = a.w;
                xr[j][4] = b.x; xr[j][5] = b.y; xr[j][6] = b.z; xr[j][7] = b.w;
            }
        } else {
#pragma unroll
            for (int i = 0; i < 8; ++i) xr[j][i] = 0.f;
        }
#pragma unroll
        for (int i = 0; i < 8; ++i) ss = fmaf(xr[j][i], xr[j][i], ss);
    }
    if (norm) {
        // fused RMSNorm (A2): every warp recomputes sum(x^2) of the L2-resident vector (deterministic)
        if (wpr == 1) {
            ss = warp_sum(ss);
        } else {
            ss = 0.f;
            for (int ch = lane; ch < chunks; ch += 32) {
                float v[8];
                if (from_emb) {
                    const uint4 e = __ldg(reinterpret_cast<const uint4 *>(p.emb + (size_t)c.tok * p.hidden) + ch);
                    v[0] = bf16lo(e.x); v[1] = bf16hi(e.x); v[2] = bf16lo(e.y); v[3] = bf16hi(e.y);
                    v[4] = bf16lo(e.z); v[5] = bf16hi(e.z); v[6] = bf16lo(e.w); v[7] = bf16hi(e.w);
                } else {
                    const float4 a = ld_act4(src + ch * 8), b = ld_act4(src + ch * 8 + 4);
                    v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
                }
#pragma unroll
                for (int i = 0; i < 8; ++i) ss = fmaf(v[i], v[i], ss);
            }
            ss = warp_sum(ss);
        }
        const float inv = 1.0f / sqrtf(ss / (float)K + p.eps);
        const bf16 *gain = ph == PH_QKV ? p.layers[c.layer].attn_norm : (ph == PH_GATEUP ? p.layers[c.layer].ffn_norm : p.final_norm);
#pragma unroll
        for (int j = 0; j < NCH; ++j) {
            const int ch = ks * cpw + j * 32 + lane;
            if (ch < c_end) {
                const uint4 gq = __ldg(reinterpret_cast<const uint4 *>(gain) + ch);
                const uint32_t gg[4] = {gq.x, gq.y, gq.z, gq.w};
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    xr[j][2 * i] *= inv * bf16lo(gg[i]);
                    xr[j][2 * i + 1] *= inv * bf16hi(gg[i]);
                }
            }
        }
    }
}

// One weight phase on the consumer side: input vector -> registers, then stage by stage.
template <int NCH>
__device__ __forceinline__ void consume_phase(const MegaParams &p, MkCtx &c, int ph, const PhaseGeom &geo, const uint8_t *ring,
                                              MkShared &sh) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int R = 2 * geo.ups, wpr = kMkConsumerWarps / R;
    const int chunks = geo.K >> 3, cpw = (chunks + wpr - 1) / wpr;
    const int row = warp / wpr, ks = warp % wpr;
    const int my_chunks = min(chunks, (ks + 1) * cpw) - ks * cpw;   // may be <= 0 for a ragged tail slice

    float xr[NCH][8];
    load_x<NCH>(p, c, ph, geo.K, wpr, xr);
    const bool from_emb = (ph == PH_O && c.layer == 0);
    const bool resid = (ph == PH_O || ph == PH_DOWN);

    for (int s = 0; s < geo.n_stages; ++s, ++c.g) {
        const int slot = c.g % kMkStages;
        const uint32_t par = (c.g / kMkStages) & 1;
        const int ub = geo.u0 + s * geo.ups;
        const int nu = min(geo.ups, geo.u1 - ub);
        // epilogue lanes fetch the old residual values while the stage is computed
        float2 rold = make_float2(0.f, 0.f);
        const bool epi = (warp == 0 && lane < nu);
        if (resid && epi) rold = resid2(p, c, from_emb, 2 * (ub + lane));

        mk_mbar_wait(&sh.full[slot], par, p.err);
        float acc[NCH];
#pragma unroll
        for (int j = 0; j < NCH; ++j) acc[j] = 0.f;
        if (row < 2 * nu) {
            const uint4 *rp = reinterpret_cast<const uint4 *>(ring + (size_t)slot * kMkStageBytes + (size_t)row * geo.row_bytes) +
                              ks * cpw;
#pragma unroll
            for (int j = 0; j < NCH; ++j) {
                const int ch = j * 32 + lane;
                if (ch < my_chunks) acc[j] = dot8(rp[ch], xr[j], 0.f);
            }
        }
        float tot = acc[0];
#pragma unroll
        for (int j = 1; j < NCH; ++j) tot += acc[j];
        tot = warp_sum(tot);
        if (lane == 0) {
            sh.partial[s & 1][warp] = tot;
            mk_mbar_arrive(&sh.empty[slot]);   // warp_sum ordered every lane's shared loads before this
        }
        consumer_sync();
        if (epi) {
            const int u = ub + lane;
            float a = 0.f, b = 0.f;
            for (int k = 0; k < wpr; ++k) {
                a += sh.partial[s & 1][(2 * lane) * wpr + k];
                b += sh.partial[s & 1][(2 * lane + 1) * wpr + k];
            }
            if (ph == PH_QKV) {
                const int hh = u >> 5, i = u & 31;
                float o0 = a, o1 = b;
                if (hh < p.n_heads + p.n_kv_heads) {
                    const float2 cs = sh.rope[i];
                    o0 = a * cs.x - b * cs.y;
                    o1 = b * cs.x + a * cs.y;
                }
                p.qkv[hh * kHeadDim + i] = o0;
                p.qkv[hh * kHeadDim + i + 32] = o1;
            } else if (ph == PH_GATEUP) {
                p.act[u] = silu_f(a) * b;
            } else if (resid) {
                *reinterpret_cast<float2 *>(p.x + 2 * u) = make_float2(rold.x + a, rold.y + b);
            } else {
                *reinterpret_cast<float2 *>(p.logits + 2 * u) = make_float2(a, b);
                unsigned long long ka = pack_argmax(a, 2 * u), kb = pack_argmax(b, 2 * u + 1);
                ka = ka > kb ? ka : kb;
                c.best = c.best > ka ? c.best : ka;
            }
        }
    }
}

__device__ __forceinline__ void run_phase(const MegaParams &p, MkCtx &c, int ph, const uint8_t *ring, MkShared &sh) {
    const PhaseGeom geo = phase_geom(p, ph);
    const int wpr = kMkConsumerWarps / (2 * geo.ups);
    const int cpw = ((geo.K >> 3) + wpr - 1) / wpr;
    const int nch = (cpw + 31) / 32;
    if (nch <= 1) consume_phase<1>(p, c, ph, geo, ring, sh);
    else if (nch <= 2) consume_phase<2>(p, c, ph, geo, ring, sh);
    else if (nch <= 4) consume_phase<4>(p, c, ph, geo, ring, sh);
    else consume_phase<8>(p, c, ph, geo, ring, sh);
}

// ---- A5: attention phase ---------------------------------------------------------------------------------------
__device__ void attention_phase(const MegaParams &p, MkCtx &c, MkShared &sh) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = p.n_heads / p.n_kv_heads;
    const int nsub = kMkConsumerWarps / G;
    const int n_ctx = c.pos + 1;
    const int ns = mk_num_splits(p, n_ctx);
    const int len = (n_ctx + ns - 1) / ns;
    const int items = p.n_kv_heads * ns;
    const size_t layer_off = (size_t)c.layer * p.layer_kv;

    for (int item = blockIdx.x; item < items; item += gridDim.x) {
        const int kvh = item / ns, split = item % ns;
        const int s0 = split * len, s1 = min(n_ctx, s0 + len);
        const bool owns_new = (split == ns - 1);
        // stage the group's queries (pre-scaled by 1/sqrt(64) = 0.125, exact) and the new K/V row
        for (int i = tid; i < G * kHeadDim; i += kMkConsumers)
            sh.q[i >> 6][i & 63] = 0.125f * ld_act(p.qkv + (size_t)(kvh * G) * kHeadDim + i);
        if (owns_new && tid < 2 * kHeadDim) {
            const int i = tid & 63;
            const int hh = p.n_heads + (tid < kHeadDim ? 0 : p.n_kv_heads) + kvh;
            const __half hv = __float2half_rn(ld_act(p.qkv + (size_t)hh * kHeadDim + i));
            kv_t *cache = (tid < kHeadDim ? p.kc : p.vc) + layer_off + ((size_t)kvh * p.max_seq + c.pos) * kHeadDim;
            (tid < kHeadDim ? sh.knew : sh.vnew)[i] = hv;
            cache[i] = hv;   // KV append (A4): read again only by later steps
        }
        consumer_sync();

        if (warp < G * nsub) {
            const int g = warp % G, sub = warp / G;
            const int head = kvh * G + g;
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
                if (t == c.pos) {
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        kr.v[j] = reinterpret_cast<const uint4 *>(sh.knew)[j];
                        vr.v[j] = reinterpret_cast<const uint4 *>(sh.vnew)[j];
                    }
                } else {
                    ld_kv_row(kr, kg + (size_t)t * kHeadDim);
                    ld_kv_row(vr, vg + (size_t)t * kHeadDim);
                }
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
            const float M = warp_max(m);
            const float sc = (m == -INFINITY) ? 0.f : __expf(m - M);
            const float l_tot = warp_sum(l * sc);
#pragma unroll
            for (int d = 0; d < kHeadDim; ++d) o[d] *= sc;
            float(&h0)[32] = *reinterpret_cast<float(*)[32]>(&o[0]);
            float(&h1)[32] = *reinterpret_cast<float(*)[32]>(&o[32]);
            warp_reduce_rows<32>(h0, lane);
            warp_reduce_rows<32>(h1, lane);
            const int r = warp_row_of_lane<32>(lane);
            const size_t pidx = (size_t)head * kMkMaxParts + split * nsub + sub;
            p.part_o[pidx * kHeadDim + r] = h0[0];
            p.part_o[pidx * kHeadDim + 32 + r] = h1[0];
            if (lane == 0) p.part_ml[pidx] = make_float2(M, l_tot);
        }
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
            const int n_parts = ns * nsub;
            for (int i = tid; i < G * kHeadDim; i += kMkConsumers) {
                const int head = kvh * G + (i >> 6), d = i & 63;
                const float2 *ml = p.part_ml + (size_t)head * kMkMaxParts;
                float M = -INFINITY;
                for (int s = 0; s < n_parts; ++s) M = fmaxf(M, __ldcg(&ml[s]).x);
                float acc = 0.f, den = 0.f;
                for (int s = 0; s < n_parts; ++s) {
                    const float2 v = __ldcg(&ml[s]);
                    const float wgt = (v.x == -INFINITY) ? 0.f : __expf(v.x - M);
                    den = fmaf(wgt, v.y, den);
                    acc = fmaf(wgt, __ldcg(p.part_o + ((size_t)head * kMkMaxParts + s) * kHeadDim + d), acc);
                }
                p.attn_out[head * kHeadDim + d] = acc / den;
            }
        }
        consumer_sync();   // sh.q / sh.flag are reused by the next item
    }
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
    for (int step = 0; step < p.n_steps; ++step) {
        c.pos = ld_act(p.pos);
        c.tok = ld_act(step == 0 ? p.tok_src : p.cur_tok);
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
            c.best = 0ull;
            run_phase(p, c, PH_HEAD, ring, sh);
            // fused argmax (A9): per-CTA best -> one packed 64-bit atomicMax; the last CTA publishes the token
            if (warp == 0) {
                unsigned long long b = c.best;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    const unsigned long long other = __shfl_xor_sync(0xffffffffu, b, o);
                    b = b > other ? b : other;
                }
                if (tid == 0) {
                    if (b) atomicMax(p.best, b);
                    __threadfence();
                    const unsigned t = atomicAdd(p.head_ticket, 1u);
                    if (t == gridDim.x - 1) {
                        __threadfence();
                        const unsigned long long win = atomicExch(p.best, 0ull);
                        const int tok = unpack_argmax_idx(win);
                        *p.cur_tok = tok;
                        p.tok_hist[c.pos + 1] = tok;
                        *p.pos = c.pos + 1;
                        *p.head_ticket = 0u;
                    }
                }
            }
            if (step + 1 < p.n_steps) grid_barrier(p, c);   // the next step reads the token and the position
        } else if (blockIdx.x == 0 && tid == 0) {
            *p.pos = c.pos + 1;   // every CTA read the position before the first barrier of this step
        }
    }
    // leave the barrier counter at zero for the next launch: the last CTA out resets it
    consumer_sync();
    if (tid == 0) {
        __threadfence();
        const unsigned t = atomicAdd(p.exit_ticket, 1u);
        if (t == gridDim.x - 1) {
            *p.bar = 0u;
            *p.exit_ticket = 0u;
        }
    }
}

// ---- host side ---------------------------------------------------------------------------------------------------
size_t mega_smem_bytes() { return (size_t)kMkStages * kMkStageBytes + sizeof(MkShared) + 128; }

bool mega_shape_supported(const hq_config &c) {
    // a unit (two rows) must fit one stage; the group must fit the consumer warps
    const int kmax = c.ffn > c.hidden ? c.ffn : c.hidden;
    const int q = c.n_heads * c.head_dim;
    return 2 * 2 * (kmax > q ? kmax : q) <= kMkStageBytes && c.n_heads / c.n_kv_heads <= kMkConsumerWarps &&
           c.hidden % 8 == 0 && c.ffn % 8 == 0 && c.vocab % 2 == 0;
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
