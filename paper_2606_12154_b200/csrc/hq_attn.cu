// hq_attn.cu — batch-1 decode, rows A2-A6 of one layer in ONE launch: RMSNorm, QKV GEMV, RoPE + KV
// append, GQA split-KV attention, split merge, O GEMV, residual add.
//
// Why one launch: the three small products of a layer (QKV 12.6 MB, attention, O 8.4 MB for the 1B shape) stream for
// ~3 us but form a chain of dependent steps; as three kernels they cost ~17 us, as one kernel whose CTAs exchange five
// vectors through L2 (round 1) 15 us.  Here the chain stays inside thread-block clusters:
//   * grid = n_kv_heads clusters of 8 CTAs (portable cluster size; 8 clusters are co-resident on every B200 probed,
//     16-CTA clusters are not: 7 fit).  Cluster kappa owns KV head kappa: its 8 CTAs compute the (G + 2) * 64 rows of
//     W_q (G query heads of the group) | W_k | W_v, exchange q, k, v through DISTRIBUTED SHARED MEMORY (st.shared::cluster
//     + remote mbarrier arrive: no global round trip, no polling), split the context of the head 8 ways, and merge the
//     8 split states with remote shared-memory loads.
//   * one exchange through L2 is left: the merged attention vector (n_heads * 64 floats) goes out as (fp32 value | 32-bit
//     epoch tag) 64-bit words, single-copy atomic, polled by every CTA ("flag in the data": no fence, no barrier); then
//     every CTA computes its rows of the O projection and adds them to the residual stream.
//   * weights never wait for data: warp 8 is a producer that requests every row of this CTA with cp.async.bulk (TMA bulk
//     copy, mbarrier complete_tx, L2 evict-first) into a 3 x 64 KB ring BEFORE griddepcontrol.wait, i.e. under the tail of
//     the previous kernel; the first K/V tile of the CTA's context chunk follows right after the wait.
//   * the launch uses 8 * n_kv_heads SMs (64 for the 1B shape); the CTAs of the following gate/up GEMV become resident on
//     the others at once (programmatic dependent launch) and prefetch their first weight batch meanwhile.
#include "hq_common.cuh"
#include "hq_internal.h"
#include "hq_attn_tile.cuh"

namespace hq {

constexpr int kAbWarps = 8;                       // consumer warps
constexpr int kAbConsumers = 32 * kAbWarps;
constexpr int kAbThreads = kAbConsumers + 32;     // + producer warp
constexpr int kAbStageBytes = 16 * 2 * 2048;      // ring stage: 16 rows of <= 4 KB back to back (ONE or two bulk copies: an SM pulls 4 KB copies at
                                                  // ~58 GB/s, 32-64 KB ones at 135-160 GB/s), or 256 cached positions (K | V)
constexpr int kAbStages = 3;
constexpr int kAbUnitsPerStage = 8;
constexpr int kAbTile0 = 56;                      // cached positions of the first K/V tile (own buffer, requested right after the wait)
constexpr int kAbRingTile = 256;                  // cached positions per ring stage (long contexts)
constexpr int kAbMaxK = 2048;                     // longest weight row (elements): hidden and n_heads * 64
constexpr int kAbMaxPhaseStages = 5;              // ring stages of one weight phase: (G + 2) / 2 <= 5 for QKV, rows / 16 for O
constexpr int kAbMaxORows = 16 * kAbMaxPhaseStages;   // rows of W_o per CTA
constexpr unsigned kAbMaxSpins = 1u << 24;        // poll rounds before a lost word / arrival traps instead of hanging the GPU

typedef unsigned long long llw_t;

struct AbShared {
    uint64_t full[kAbStages], empty[kAbStages];
    uint64_t kv_bar;                              // first K/V tile landed
    uint64_t qkv_bar;                             // q, k, v of the KV head complete in this CTA (bytes pushed by the whole cluster)
    uint64_t part_bar;                            // this CTA's slice of the split states of all 8 ranks complete
    alignas(16) bf16 xh[kAbMaxK], xl[kAbMaxK];    // phase input as two bf16 planes x = hi + lo (16 mantissa bits): normalised x, later
                                                  // the attention vector
    alignas(16) float2 qkv[(8 + 2) * 32];         // RoPE pairs (dim i, dim i + 32) of the G query heads | k | v of this token
    alignas(16) float part[8][kHeadDim + 4];      // this CTA's split state per query head: o[64] (unnormalised), m, l
    alignas(16) float mrg[kAbWarps][kHeadDim + 4];// sub-split states of the warps
    union {
        float recv[kAbCluster][10 * 8];           // from every rank: (m, l) of the G heads, then the 8 G output dims this CTA merges
        float dpart[kAbMaxPhaseStages][kAbWarps][16];   // weight phases: per stage, warp (K slice) and row, partial dot products
    };                                            // (never live together: see the notes at the phase loop)
    float xo[kAbMaxORows];                        // residual values of this CTA's O rows
    float red[kAbWarps];
    alignas(128) kv_t kst[kAbTile0 * kHeadDim];
    alignas(128) kv_t vst[kAbTile0 * kHeadDim];
};

static_assert((size_t)kAbStages * kAbStageBytes + sizeof(AbShared) + 128 <= 232448, "attention block: over the 227 KB of shared memory per CTA");

__device__ __noinline__ void ab_fail(int *err, int code) {
    atomicExch(err, code);
    __threadfence_system();
    __trap();
}
__device__ __forceinline__ void ab_wait(uint64_t *bar, uint32_t parity, int *err) {
    unsigned spins = 0;
    while (!mbar_try_wait(bar, parity))
        if (++spins == kAbMaxSpins) ab_fail(err, 21);
}
__device__ __forceinline__ void ab_consumer_sync() { asm volatile("bar.sync 1, %0;" ::"n"(kAbConsumers) : "memory"); }
__device__ __forceinline__ float2 ab_h2f(uint32_t u) { return __half22float2(*reinterpret_cast<const __half2 *>(&u)); }
__device__ __forceinline__ float ab_round_kv(float v) { return __half2float(__float2half_rn(v)); }

// geometry of one CTA (uniform over the grid apart from rank / kvh)
struct AbGeom {
    int G, K, qdim, rank, kvh;
    int q_units, q_u0, q_stages;      // QKV: units (RoPE pairs) of this CTA within the cluster's (G + 2) * 32
    int o_rows, o_row0, o_stages;     // O: rows of W_o of this CTA
};
__device__ __forceinline__ AbGeom ab_geom(const AttnBlockParams &p) {
    AbGeom g;
    g.G = p.n_heads / p.n_kv_heads;
    g.K = p.hidden;
    g.qdim = p.n_heads * kHeadDim;
    g.rank = (int)cluster_ctarank();
    g.kvh = (int)cluster_id_x();
    g.q_units = 4 * (g.G + 2);
    g.q_u0 = g.rank * g.q_units;
    g.q_stages = (g.q_units + kAbUnitsPerStage - 1) / kAbUnitsPerStage;
    g.o_rows = p.hidden / (p.n_kv_heads * kAbCluster);
    g.o_row0 = (g.kvh * kAbCluster + g.rank) * g.o_rows;
    g.o_stages = (g.o_rows / 2 + kAbUnitsPerStage - 1) / kAbUnitsPerStage;
    return g;
}
// context chunk of a rank: positions [c0, c1) of the n_ctx = pos + 1 visible ones; the current position is not in the
// cache yet (it comes from the q/k/v exchange), so the cached part is [c0, c0 + n_cached)
struct AbChunk { int c0, c1, n_cached; bool has_new; };
__device__ __forceinline__ AbChunk ab_chunk(int pos, int rank) {
    const int n_ctx = pos + 1, len = (n_ctx + kAbCluster - 1) / kAbCluster;
    AbChunk c;
    c.c0 = rank * len;
    c.c1 = min(n_ctx, c.c0 + len);
    c.has_new = pos >= c.c0 && pos < c.c1;
    const int cached_end = min(c.c1, pos);
    c.n_cached = cached_end > c.c0 ? cached_end - c.c0 : 0;
    return c;
}

// ---- producer warp: walks the static schedule QKV stages | K/V tiles | O stages -------------------------------------
// Lane r issues row r of a stage (address arithmetic for 16 rows in parallel: one thread issuing 48 copies serially took
// microseconds); lane 0 posts the byte count first.
__device__ void ab_producer(const AttnBlockParams &p, const AbGeom &g, uint8_t *ring, AbShared &sh) {
    const int lane = threadIdx.x & 31;
    const uint64_t pol = l2_policy_evict_first();
    unsigned n = 0;   // stages produced
    auto slot_wait = [&](unsigned i) { ab_wait(&sh.empty[i % kAbStages], ((i / kAbStages) & 1) ^ 1, p.err); };
    const uint32_t qrb = (uint32_t)g.K * 2;
    for (int s = 0; s < g.q_stages; ++s, ++n) {
        slot_wait(n);
        const int ub = s * kAbUnitsPerStage, nu = min(kAbUnitsPerStage, g.q_units - ub);
        uint64_t *bar = &sh.full[n % kAbStages];
        uint8_t *dst = ring + (size_t)(n % kAbStages) * kAbStageBytes;
        if (lane == 0) {
            // stage rows 0-7: row i of the units' RoPE pairs, rows 8-15: row i + 32.  Consecutive units are consecutive rows
            // of one head, so each half is one copy (two where the 8 units straddle a head boundary).
            mbar_expect_tx(bar, 2u * nu * qrb);
            for (int j = 0; j < nu;) {
                const int cu = g.q_u0 + ub + j, hh = cu >> 5, i = cu & 31;
                const int run = min(nu - j, 32 - i);
                const bf16 *row = hh < g.G ? p.wq + (size_t)((g.kvh * g.G + hh) * kHeadDim + i) * g.K
                                           : (hh == g.G ? p.wk : p.wv) + (size_t)(g.kvh * kHeadDim + i) * g.K;
                bulk_g2s_hint(dst + (size_t)j * qrb, row, (uint32_t)run * qrb, bar, pol);
                bulk_g2s_hint(dst + (size_t)(8 + j) * qrb, row + (size_t)32 * g.K, (uint32_t)run * qrb, bar, pol);
                j += run;
            }
        }
    }
    // this CTA's rows of W_o are one contiguous range: into L2 now (behind the QKV rows), so that the ring loads issued
    // later are L2 hits
    if (lane == 0 && g.q_stages >= kAbStages) bulk_prefetch_l2(p.wo + (size_t)g.o_row0 * g.qdim, (uint32_t)g.o_rows * (uint32_t)g.qdim * 2u);
    // everything below depends on the position / the cache rows written by earlier kernels
    pdl_wait();
    const int pos = ld_act(p.pos);
    const AbChunk c = ab_chunk(pos, g.rank);
    const kv_t *kg = p.kc + ((size_t)g.kvh * p.max_seq + c.c0) * kHeadDim;
    const kv_t *vg = p.vc + ((size_t)g.kvh * p.max_seq + c.c0) * kHeadDim;
    const int n0 = min(c.n_cached, kAbTile0);
    if (lane == 0) {
        if (n0 > 0) {
            const uint32_t bytes = (uint32_t)n0 * kHeadDim * sizeof(kv_t);
            mbar_expect_tx(&sh.kv_bar, 2 * bytes);
            bulk_g2s(sh.kst, kg, bytes, &sh.kv_bar);
            bulk_g2s(sh.vst, vg, bytes, &sh.kv_bar);
        } else {
            mbar_arrive(&sh.kv_bar);
        }
    }
    for (int t = kAbTile0; t < c.n_cached; t += kAbRingTile, ++n) {
        slot_wait(n);
        if (lane == 0) {
            const uint32_t bytes = (uint32_t)min(kAbRingTile, c.n_cached - t) * kHeadDim * sizeof(kv_t);
            uint64_t *bar = &sh.full[n % kAbStages];
            uint8_t *dst = ring + (size_t)(n % kAbStages) * kAbStageBytes;
            mbar_expect_tx(bar, 2 * bytes);
            bulk_g2s(dst, kg + (size_t)t * kHeadDim, bytes, bar);
            bulk_g2s(dst + kAbStageBytes / 2, vg + (size_t)t * kHeadDim, bytes, bar);
        }
    }
    const uint32_t orb = (uint32_t)g.qdim * 2;
    for (int s = 0; s < g.o_stages; ++s, ++n) {
        slot_wait(n);
        const int nr = min(16, g.o_rows - 16 * s);   // rows of W_o of this stage: one contiguous copy
        if (lane == 0) {
            uint64_t *bar = &sh.full[n % kAbStages];
            mbar_expect_tx(bar, (uint32_t)nr * orb);
            bulk_g2s_hint(ring + (size_t)(n % kAbStages) * kAbStageBytes, p.wo + (size_t)(g.o_row0 + 16 * s) * g.qdim, (uint32_t)nr * orb, bar, pol);
        }
    }
}

// ---- consumers ---------------------------------------------------------------------------------------------------
// The 16 rows of a stage against the input vector on the tensor cores (mma.sync m16n8k16 bf16, fp32 accumulate): the
// launch is bound by instruction issue, not by bytes, and two LDS.128 + two MMAs replace ~100 load / convert / FMA
// instructions.  Fragment scheme of hq_stream.cu: the rows of a stage lie back to back (a multiple of 128 bytes apart), lane
// (g, t) loads elements [8t, 8t + 8) of a 32-element K block of A rows g and g + 8 — words 0, 1 feed the first k-tile, words
// 2, 3 the second (a permutation of K, applied to B alike) — and odd rows take the neighbouring 64-byte block, so a
// quarter-warp covers all 32 banks.  B = the input as bf16 planes hi | lo in columns 0, 1 (block order of the even rows)
// and 2, 3 (block order of the odd rows); row m reads D[m][2 (m & 1)] + D[m][2 (m & 1) + 1].  Warp w owns K blocks
// [w * nb, (w + 1) * nb): the 8 partial sums of a row meet in shared memory.
__device__ __forceinline__ void ab_mma_bf16(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
    asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint4 ab_lds128(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
constexpr int kAbMaxBlocks = kAbMaxK / 32 / kAbWarps;   // 32-element K blocks per warp at the longest row
// K blocks per row (even: odd rows read block b ^ 1) and per warp
__device__ __forceinline__ int ab_nblk(int K) { return 2 * ((K + 63) / 64); }
// B fragments of this warp's K blocks: lane = (column n = lane >> 2, t = lane & 3); n: plane n & 1, block order n >> 1
__device__ __forceinline__ void ab_load_b(const AbShared &sh, int K, int nb, int warp, int lane, uint4 (&bq)[kAbMaxBlocks]) {
    const int n = lane >> 2, t = lane & 3, nblk = ab_nblk(K);
    const bf16 *src = (n & 1) ? sh.xl : sh.xh;
#pragma unroll
    for (int i = 0; i < kAbMaxBlocks; ++i) {
        const int blk = warp * nb + i, ks = (blk ^ (n >> 1)) * 32 + t * 8;
        const bool ok = n < 4 && i < nb && blk < nblk && ks < K;
        bq[i] = ok ? *reinterpret_cast<const uint4 *>(src + ks) : make_uint4(0, 0, 0, 0);
    }
}
__device__ __forceinline__ void ab_dot16(uint32_t stage_addr, uint32_t row_bytes, int K, int nb, int warp, int lane,
                                         const uint4 (&bq)[kAbMaxBlocks], float (&c)[4]) {
    float cc[4][4];   // four chains: an MMA waits ~30 cycles for its accumulator
#pragma unroll
    for (int i = 0; i < 4; ++i) cc[i][0] = cc[i][1] = cc[i][2] = cc[i][3] = 0.f;
    const int g = lane >> 2, t = lane & 3, nblk = ab_nblk(K);
    const uint32_t a_base = stage_addr + (uint32_t)g * row_bytes + (uint32_t)t * 16u;
    uint4 a0[kAbMaxBlocks], a1[kAbMaxBlocks];
#pragma unroll
    for (int i = 0; i < kAbMaxBlocks; ++i) {
        const int blk = warp * nb + i;
        if (i < nb && blk < nblk) {   // warp-uniform
            const uint32_t off = (uint32_t)(blk ^ (g & 1)) * 64u;
            a0[i] = ab_lds128(a_base + off);
            a1[i] = ab_lds128(a_base + 8u * row_bytes + off);
        } else {
            a0[i] = a1[i] = make_uint4(0, 0, 0, 0);
        }
    }
#pragma unroll
    for (int i = 0; i < kAbMaxBlocks; ++i) {
        if (i < nb) {
            ab_mma_bf16(cc[(2 * i) & 3], a0[i].x, a1[i].x, a0[i].y, a1[i].y, bq[i].x, bq[i].y);
            ab_mma_bf16(cc[(2 * i + 1) & 3], a0[i].z, a1[i].z, a0[i].w, a1[i].w, bq[i].z, bq[i].w);
        }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) c[i] = (cc[0][i] + cc[1][i]) + (cc[2][i] + cc[3][i]);
}
// 8 fp32 of the phase input -> the two bf16 planes in shared memory
__device__ __forceinline__ void ab_stage_x(AbShared &sh, int e0, const float (&v)[8]) {
    uint32_t h[4], l[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) split_bf16x2(v[2 * i], v[2 * i + 1], h[i], l[i]);
    *reinterpret_cast<uint4 *>(sh.xh + e0) = make_uint4(h[0], h[1], h[2], h[3]);
    *reinterpret_cast<uint4 *>(sh.xl + e0) = make_uint4(l[0], l[1], l[2], l[3]);
}
__device__ __forceinline__ void ll_store(llw_t *p, float v, uint32_t tag) {
    const llw_t w = ((llw_t)tag << 32) | (llw_t)__float_as_uint(v);
    asm volatile("st.global.cg.u64 [%0], %1;" ::"l"(p), "l"(w) : "memory");
}
__device__ __forceinline__ void ll_load2(const llw_t *p, llw_t &a, llw_t &b) {
    asm volatile("ld.volatile.global.v2.u64 {%0,%1}, [%2];" : "=l"(a), "=l"(b) : "l"(p) : "memory");
}

// online-softmax state of one lane: its position stream (lane >> 3) and its dim octet (lane & 7)
struct AbState { float m, l, o[8]; };
__device__ __forceinline__ float ab_score(const float (&q)[8], const uint4 &kk) {
    const float2 k0 = ab_h2f(kk.x), k1 = ab_h2f(kk.y), k2 = ab_h2f(kk.z), k3 = ab_h2f(kk.w);
    float s = q[0] * k0.x;
    s = fmaf(q[1], k0.y, s); s = fmaf(q[2], k1.x, s); s = fmaf(q[3], k1.y, s);
    s = fmaf(q[4], k2.x, s); s = fmaf(q[5], k2.y, s); s = fmaf(q[6], k3.x, s); s = fmaf(q[7], k3.y, s);
    s += __shfl_xor_sync(0xffffffffu, s, 1);
    s += __shfl_xor_sync(0xffffffffu, s, 2);
    s += __shfl_xor_sync(0xffffffffu, s, 4);
    return s;
}
// n positions of a shared-memory tile (rows of 64 fp16): sub-split `sub` of `nsub` takes groups of 16 positions round robin.
// Four positions per lane group and iteration: their scores are independent (loads, FMAs and shuffles overlap), one
// rescale of the running state per iteration.
__device__ __forceinline__ void ab_tile(AbState &st, const float (&q)[8], const kv_t *kt, const kv_t *vt, int n, int sub, int nsub,
                                        int lane) {
    const int oct = lane & 7, grp = lane >> 3;
    const uint4 *k4 = reinterpret_cast<const uint4 *>(kt) + oct, *v4 = reinterpret_cast<const uint4 *>(vt) + oct;
#pragma unroll 1
    for (int t0 = sub * 16; t0 < n; t0 += 16 * nsub) {   // warp-uniform trip count
        uint4 kk[4], vv[4];
        float sc[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int t = t0 + 4 * u + grp;
            const bool ok = t < n;
            kk[u] = ok ? k4[(size_t)t * 8] : make_uint4(0, 0, 0, 0);
            vv[u] = ok ? v4[(size_t)t * 8] : make_uint4(0, 0, 0, 0);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const float s = ab_score(q, kk[u]);
            sc[u] = (t0 + 4 * u + grp < n) ? s : -INFINITY;
        }
        const float m_new = fmaxf(fmaxf(st.m, fmaxf(sc[0], sc[1])), fmaxf(sc[2], sc[3]));
        if (m_new != -INFINITY) {
            const float corr = __expf(st.m - m_new);   // m = -inf the first time -> 0
            float pr[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) pr[u] = __expf(sc[u] - m_new);   // -inf -> 0
            st.l = st.l * corr + ((pr[0] + pr[1]) + (pr[2] + pr[3]));
#pragma unroll
            for (int j = 0; j < 8; ++j) st.o[j] *= corr;
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const float2 v0 = ab_h2f(vv[u].x), v1 = ab_h2f(vv[u].y), v2 = ab_h2f(vv[u].z), v3 = ab_h2f(vv[u].w);
                st.o[0] = fmaf(pr[u], v0.x, st.o[0]); st.o[1] = fmaf(pr[u], v0.y, st.o[1]);
                st.o[2] = fmaf(pr[u], v1.x, st.o[2]); st.o[3] = fmaf(pr[u], v1.y, st.o[3]);
                st.o[4] = fmaf(pr[u], v2.x, st.o[4]); st.o[5] = fmaf(pr[u], v2.y, st.o[5]);
                st.o[6] = fmaf(pr[u], v3.x, st.o[6]); st.o[7] = fmaf(pr[u], v3.y, st.o[7]);
            }
            st.m = m_new;
        }
    }
}
// merge state b into a (same dim octet)
__device__ __forceinline__ void ab_merge(float &M, float &l, float (&o)[8], float M2, float l2, const float *o2) {
    const float Mn = fmaxf(M, M2);
    const float wa = (M == -INFINITY) ? 0.f : __expf(M - Mn), wb = (M2 == -INFINITY) ? 0.f : __expf(M2 - Mn);
    l = l * wa + l2 * wb;
#pragma unroll
    for (int j = 0; j < 8; ++j) o[j] = o[j] * wa + o2[j] * wb;
    M = Mn;
}

// optional timeline (hq_debug_trace): thread 0 of every CTA stamps the GPU global timer at fixed points
template <bool TRACE>
__device__ __forceinline__ void ab_trace(const AttnBlockParams &p, int &ti) {
    if (TRACE && threadIdx.x == 0) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        if (ti < p.trace_cap) p.trace[(size_t)blockIdx.x * p.trace_cap + ti] = t;
        ++ti;
    }
}

// A5 on this rank's chunk of the context + the two exchanges that follow it: split states -> cluster (pushed), merged
// slice of the attention vector -> L2 (tagged words), whole vector polled into sh.xs.  Ring stages consumed: returned in n.
template <bool TRACE>
__device__ __forceinline__ void ab_attention(const AttnBlockParams &p, const AbGeom &g, const uint8_t *ring, AbShared &sh, int pos,
                                             uint32_t tag, unsigned &n, int &ti) {
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const AbChunk c = ab_chunk(pos, g.rank);
    const int nsub = kAbWarps / g.G, hg = warp % g.G, sub = warp / g.G;
    const bool active = warp < g.G * nsub;
    const int oct = lane & 7, grp = lane >> 3;
    ab_wait(&sh.qkv_bar, 0, p.err);
    ab_trace<TRACE>(p, ti);   // q, k, v of the head here
    AbState st;
    st.m = -INFINITY;
    st.l = 0.f;
#pragma unroll
    for (int j = 0; j < 8; ++j) st.o[j] = 0.f;
    float q[8];
    {
        // dims [8 oct, 8 oct + 8) of the head: pairs hold (dim i, dim i + 32); pre-scaled by 1/sqrt(64) = 0.125 (exact)
        const float2 *qp = sh.qkv + hg * 32 + (oct & 3) * 8;
#pragma unroll
        for (int j = 0; j < 8; ++j) q[j] = 0.125f * (oct < 4 ? qp[j].x : qp[j].y);
    }
    ab_wait(&sh.kv_bar, 0, p.err);
    ab_trace<TRACE>(p, ti);   // first K/V tile here
    // tile 0 sits in its own buffer, later tiles (long contexts) come through the ring
#pragma unroll 1
    for (int t = 0; t < c.n_cached; t += (t == 0 ? kAbTile0 : kAbRingTile)) {
        const kv_t *kt = sh.kst, *vt = sh.vst;
        int nt = min(c.n_cached, kAbTile0), slot = 0;
        if (t > 0) {
            slot = n % kAbStages;
            ab_wait(&sh.full[slot], (n / kAbStages) & 1, p.err);
            kt = reinterpret_cast<const kv_t *>(ring + (size_t)slot * kAbStageBytes);
            vt = kt + kAbStageBytes / 2 / sizeof(kv_t);
            nt = min(kAbRingTile, c.n_cached - t);
        }
        if (active) ab_tile(st, q, kt, vt, nt, sub, nsub, lane);
        if (t > 0) {
            __syncwarp();
            if (lane == 0) mbar_arrive(&sh.empty[slot]);
            ++n;
        }
    }
    if (c.has_new && active && sub == 0) {
        // the current position: k and v of this step, rounded to fp16 exactly like the cache row later steps will read
        const float2 *kp = sh.qkv + g.G * 32 + (oct & 3) * 8, *vp = sh.qkv + (g.G + 1) * 32 + (oct & 3) * 8;
        float s = 0.f, vn[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            s = fmaf(q[j], ab_round_kv(oct < 4 ? kp[j].x : kp[j].y), s);
            vn[j] = ab_round_kv(oct < 4 ? vp[j].x : vp[j].y);
        }
        s += __shfl_xor_sync(0xffffffffu, s, 1);
        s += __shfl_xor_sync(0xffffffffu, s, 2);
        s += __shfl_xor_sync(0xffffffffu, s, 4);
        if (grp == 0) {
            const float m_new = fmaxf(st.m, s);
            const float corr = __expf(st.m - m_new), pr = __expf(s - m_new);
            st.l = st.l * corr + pr;
#pragma unroll
            for (int j = 0; j < 8; ++j) st.o[j] = fmaf(pr, vn[j], st.o[j] * corr);
            st.m = m_new;
        }
    }
    {
        // merge the 4 position streams of the warp, then the sub-splits of the head through shared memory
        float M = fmaxf(st.m, __shfl_xor_sync(0xffffffffu, st.m, 8));
        M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, 16));
        const float sc = (st.m == -INFINITY) ? 0.f : __expf(st.m - M);
        float l = st.l * sc;
        l += __shfl_xor_sync(0xffffffffu, l, 8);
        l += __shfl_xor_sync(0xffffffffu, l, 16);
        float o[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            o[j] = st.o[j] * sc;
            o[j] += __shfl_xor_sync(0xffffffffu, o[j], 8);
            o[j] += __shfl_xor_sync(0xffffffffu, o[j], 16);
        }
        if (active && sub > 0 && lane < 8) {
#pragma unroll
            for (int j = 0; j < 8; ++j) sh.mrg[warp][oct * 8 + j] = o[j];
            if (lane == 0) { sh.mrg[warp][kHeadDim] = M; sh.mrg[warp][kHeadDim + 1] = l; }
        }
        ab_consumer_sync();
        if (active && sub == 0 && lane < 8) {
#pragma unroll 1
            for (int k = 1; k < nsub; ++k) {
                const float *o2 = sh.mrg[k * g.G + hg];
                ab_merge(M, l, o, o2[kHeadDim], o2[kHeadDim + 1], o2 + oct * 8);
            }
#pragma unroll
            for (int j = 0; j < 8; ++j) sh.part[hg][oct * 8 + j] = o[j];
            if (lane == 0) { sh.part[hg][kHeadDim] = M; sh.part[hg][kHeadDim + 1] = l; }
        }
        ab_consumer_sync();
    }
    ab_trace<TRACE>(p, ti);   // attention of this chunk done
    // this CTA's split states are complete: push to every rank (m, l) of the G heads and the 8 G output dims it merges
    {
        const int per = 5 * g.G;   // float pairs per destination
        const uint32_t recv_base = smem_addr_u32(&sh.recv[g.rank][0]), bar_addr = smem_addr_u32(&sh.part_bar);
        for (int t = tid; t < kAbCluster * per; t += kAbConsumers) {
            const int dst = t / per, k = t - dst * per;
            float a, b;
            if (k < g.G) {
                a = sh.part[k][kHeadDim];
                b = sh.part[k][kHeadDim + 1];
            } else {
                const int e = dst * 8 * g.G + 2 * (k - g.G);   // even: both dims in the same head
                a = sh.part[e >> 6][e & 63];
                b = sh.part[e >> 6][(e & 63) + 1];
            }
            st_async_f32x2(cluster_map(recv_base + (uint32_t)k * 8u, (uint32_t)dst), a, b, cluster_map(bar_addr, (uint32_t)dst));
        }
    }
    // split merge: thread t < 8 G merges output dim rank * 8 G + t of the group over the 8 ranks
    ab_wait(&sh.part_bar, 0, p.err);
    ab_trace<TRACE>(p, ti);   // split states of all ranks here
    if (tid < 8 * g.G) {
        const int e = g.rank * 8 * g.G + tid, h2 = e >> 6, d = e & 63;
        float M = -INFINITY;
#pragma unroll
        for (int r = 0; r < kAbCluster; ++r) M = fmaxf(M, sh.recv[r][2 * h2]);
        float num = 0.f, den = 0.f;
#pragma unroll
        for (int r = 0; r < kAbCluster; ++r) {
            const float mr = sh.recv[r][2 * h2];
            const float w = (mr == -INFINITY) ? 0.f : __expf(mr - M);
            num = fmaf(w, sh.recv[r][2 * g.G + tid], num);
            den = fmaf(w, sh.recv[r][2 * h2 + 1], den);
        }
        ll_store(p.ll_attn + (size_t)(g.kvh * g.G + h2) * kHeadDim + d, num / den, tag);
    }
    ab_trace<TRACE>(p, ti);   // merged slice published
    // the one exchange through L2: every CTA polls the whole attention vector (tagged words)
    if (tid * 8 < g.qdim) {
        const llw_t *src = p.ll_attn + (size_t)tid * 8;
        llw_t w[8];
        unsigned spins = 0;
        for (;;) {
#pragma unroll
            for (int i = 0; i < 8; i += 2) ll_load2(src + i, w[i], w[i + 1]);
            bool ok = true;
#pragma unroll
            for (int i = 0; i < 8; ++i) ok = ok && (uint32_t)(w[i] >> 32) == tag;
            if (ok) break;
            if (++spins == kAbMaxSpins) ab_fail(p.err, 23);
            __nanosleep(32);
        }
        float v[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) v[i] = __uint_as_float((uint32_t)w[i]);
        ab_stage_x(sh, tid * 8, v);
    }
    ab_consumer_sync();
    ab_trace<TRACE>(p, ti);   // attention vector polled and staged
}

template <bool TRACE>
__global__ void __launch_bounds__(kAbThreads, 1) attn_block_kernel(const __grid_constant__ AttnBlockParams p) {
    extern __shared__ __align__(128) uint8_t ab_smem[];
    int ti = 0;
    ab_trace<TRACE>(p, ti);   // CTA started
    if (threadIdx.x == 0) { step_stamp(p.step_trace, p.step_slot, 0); step_stamp(p.step_trace, p.step_slot, 3); }
    uint8_t *ring = ab_smem;
    AbShared &sh = *reinterpret_cast<AbShared *>(ab_smem + (size_t)kAbStages * kAbStageBytes);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const AbGeom g = ab_geom(p);

    if (tid == 0) {
        for (int s = 0; s < kAbStages; ++s) {
            mbar_init(&sh.full[s], 1);
            mbar_init(&sh.empty[s], kAbWarps);
        }
        mbar_init(&sh.kv_bar, 1);
        mbar_init(&sh.qkv_bar, 1);
        mbar_init(&sh.part_bar, 1);
        mbar_fence_init();
        // bytes the cluster will push into this CTA (st.async complete_tx): 8 bytes per RoPE pair of the (G + 2) heads;
        // from every rank (m, l) of the G heads + this CTA's 8 G output dims
        mbar_expect_tx(&sh.qkv_bar, (uint32_t)(kAbCluster * g.q_units * 8));
        mbar_expect_tx(&sh.part_bar, (uint32_t)(kAbCluster * 10 * g.G * 4));
    }
    // the barriers of every CTA of the cluster exist before anyone pushes into them
    cluster_sync_all();
    ab_trace<TRACE>(p, ti);   // cluster up

    if (warp == kAbWarps) {
        ab_producer(p, g, ring, sh);
        return;
    }

    // ---- A2: residual stream -> RMSNorm -> shared memory (thread t owns elements [8t, 8t + 8)) ------------------
    const bool has = tid * 8 < g.K;
    uint4 gq = make_uint4(0, 0, 0, 0);
    if (has) gq = __ldg(reinterpret_cast<const uint4 *>(p.gain) + tid);   // immutable: its latency overlaps the previous kernel
    pdl_launch_dependents();
    pdl_wait();
    ab_trace<TRACE>(p, ti);   // dependency wait over
    if (tid == 0) step_stamp(p.step_trace, p.step_slot, 1);
    const int pos = ld_act(p.pos);
    const uint32_t tag = *reinterpret_cast<volatile unsigned int *>(p.epoch);
    float v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = 0.f;
    if (has) {
        const float4 a = ld_act4(p.x + (size_t)tid * 8), b = ld_act4(p.x + (size_t)tid * 8 + 4);
        v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
    }
    for (int r = tid; r < g.o_rows; r += kAbConsumers) sh.xo[r] = ld_act(p.x + g.o_row0 + r);
    {
        float ss = 0.f;
#pragma unroll
        for (int i = 0; i < 8; ++i) ss = fmaf(v[i], v[i], ss);
        ss = warp_sum(ss);
        if (lane == 0) sh.red[warp] = ss;
        ab_consumer_sync();
        float tot = 0.f;
#pragma unroll
        for (int k = 0; k < kAbWarps; ++k) tot += sh.red[k];
        const float inv = 1.0f / sqrtf(tot / (float)g.K + p.eps);
        const uint32_t gg[4] = {gq.x, gq.y, gq.z, gq.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            v[2 * i] *= inv * bf16lo(gg[i]);
            v[2 * i + 1] *= inv * bf16hi(gg[i]);
        }
        if (has) ab_stage_x(sh, tid * 8, v);
        ab_consumer_sync();
    }
    ab_trace<TRACE>(p, ti);   // x normalised and staged

    // ---- the two weight phases, one loop (one copy of the stage body: the launch runs every instruction once, so code
    //      size is instruction-fetch time).  Phase 0 = A3 + A4: QKV rows, RoPE, q/k/v -> every CTA of the cluster, k/v ->
    //      cache.  Between the phases: A5.  Phase 1 = A6: this CTA's rows of the O projection + residual.
    unsigned n = 0;   // ring stages consumed
    const uint32_t qkv_base = smem_addr_u32(sh.qkv), qkv_bar_addr = smem_addr_u32(&sh.qkv_bar);
    // sh.dpart shares its memory with sh.recv.  Phase 0: another rank pushes split states into recv only after it has
    // received every q/k/v push of this CTA, i.e. after every thread here has read dpart.  Phase 1: the CTA-wide barrier
    // after the poll follows the last read of recv.
#pragma unroll 1
    for (int ph = 0; ph < 2; ++ph) {
        if (ph == 1) ab_attention<TRACE>(p, g, ring, sh, pos, tag, n, ti);
        const int K = ph ? g.qdim : g.K, units = ph ? g.o_rows / 2 : g.q_units;
        const int nb = (ab_nblk(K) + kAbWarps - 1) / kAbWarps;
        uint4 bq[kAbMaxBlocks];
        ab_load_b(sh, K, nb, warp, lane, bq);
        // RoPE factors of the units this thread finishes (phase 0): loaded now, needed after the barrier below
        float2 cs[kAbMaxPhaseStages];
#pragma unroll
        for (int s = 0; s < kAbMaxPhaseStages; ++s) {
            const int cu = g.q_u0 + s * kAbUnitsPerStage + (tid >> 3);
            cs[s] = (ph == 0 && tid < 64 && s * kAbUnitsPerStage + (tid >> 3) < units) ? p.rope[(size_t)pos * 32 + (cu & 31)] : make_float2(1.f, 0.f);
        }
        // every stage: 16 rows x this warp's K slice on the tensor cores; the accumulators stay in registers, so the stages
        // only wait for their bytes, not for one another's epilogue
        float c[kAbMaxPhaseStages][4];
#pragma unroll
        for (int s = 0; s < kAbMaxPhaseStages; ++s) {
            if (s * kAbUnitsPerStage < units) {   // uniform
                const int slot = n % kAbStages;
                ab_wait(&sh.full[slot], (n / kAbStages) & 1, p.err);
                ab_dot16(smem_addr_u32(ring + (size_t)slot * kAbStageBytes), (uint32_t)(K * 2), K, nb, warp, lane, bq, c[s]);
                __syncwarp();
                if (lane == 0) mbar_arrive(&sh.empty[slot]);
                ++n;
                // C fragment: lane holds (row lane >> 2, cols 2 (lane & 3), +1) in c0, c1 and row + 8 in c2, c3; a row reads the
                // (hi, lo) column pair of its block order
                if ((lane & 3) == ((lane >> 2) & 1)) {
                    sh.dpart[s][warp][lane >> 2] = c[s][0] + c[s][1];
                    sh.dpart[s][warp][(lane >> 2) + 8] = c[s][2] + c[s][3];
                }
            }
        }
        ab_trace<TRACE>(p, ti);   // this warp's dots done
        ab_consumer_sync();
        // epilogue: thread t = (u = t >> 3, destination rank t & 7) sums the 8 K slices of stage rows u and u + 8: the RoPE
        // pair of unit u (phase 0), rows 16 s + u and 16 s + u + 8 of this CTA's slice of W_o (phase 1)
        if (tid < 64) {
            const int u = tid >> 3, dst = tid & 7;
#pragma unroll
            for (int s = 0; s < kAbMaxPhaseStages; ++s) {
                if (s * kAbUnitsPerStage + u < units || (ph == 1 && s * kAbUnitsPerStage < units)) {
                    float a = 0.f, b = 0.f;
#pragma unroll
                    for (int w = 0; w < kAbWarps; ++w) {
                        a += sh.dpart[s][w][u];
                        b += sh.dpart[s][w][u + 8];
                    }
                    if (ph == 0) {
                        const int cu = g.q_u0 + s * kAbUnitsPerStage + u, hh = cu >> 5, i = cu & 31;
                        float o0 = a, o1 = b;
                        if (hh <= g.G) {   // query heads and k: rotate the pair (i, i + 32)
                            o0 = a * cs[s].x - b * cs[s].y;
                            o1 = b * cs[s].x + a * cs[s].y;
                        }
                        st_async_f32x2(cluster_map(qkv_base + (uint32_t)(hh * 32 + i) * 8u, (uint32_t)dst), o0, o1,
                                       cluster_map(qkv_bar_addr, (uint32_t)dst));
                        if (dst == 0 && hh >= g.G) {
                            kv_t *row = (hh == g.G ? p.kc : p.vc) + ((size_t)g.kvh * p.max_seq + pos) * kHeadDim;
                            row[i] = __float2half_rn(o0);
                            row[i + 32] = __float2half_rn(o1);
                        }
                    } else if (dst == 0) {
                        const int r = 16 * s + u;
                        if (r < g.o_rows) p.x[g.o_row0 + r] = sh.xo[r] + a;
                        if (r + 8 < g.o_rows) p.x[g.o_row0 + r + 8] = sh.xo[r + 8] + b;
                    }
                }
            }
        }
        ab_trace<TRACE>(p, ti);   // phase done
    }
    // Every word polled above was published after its writer had received everything other CTAs push into its shared
    // memory, and every CTA read the epoch before it published: no CTA needs this one's shared memory or the old epoch.
    if (g.kvh == 0 && g.rank == 0 && tid == 0) *p.epoch = tag + 1u == 0u ? 1u : tag + 1u;
    if (tid == 0) step_stamp(p.step_trace, p.step_slot, 2);
}

// ---- host side ---------------------------------------------------------------------------------------------------
size_t attn_block_smem_bytes() { return (size_t)kAbStages * kAbStageBytes + sizeof(AbShared) + 128; }

bool attn_block_shape_supported(const hq_config &c) {
    const int G = c.n_kv_heads > 0 ? c.n_heads / c.n_kv_heads : 0, qdim = c.n_heads * c.head_dim;
    const int o_den = c.n_kv_heads * kAbCluster;
    return c.head_dim == kHeadDim && G >= 1 && G <= 8 && c.hidden % 8 == 0 && c.hidden <= kAbMaxK && qdim <= kAbMaxK &&
           c.hidden % 64 == 0 && c.hidden % (2 * o_den) == 0 && c.hidden / o_den <= kAbMaxORows;   // % 64: whole K block pairs (ab_dot16)
}

static void attn_block_config(cudaLaunchConfig_t &cfg, cudaLaunchAttribute *attr, const LaunchCtx &c, int n_kv_heads) {
    cfg = {};
    cfg.gridDim = dim3(n_kv_heads * kAbCluster);
    cfg.blockDim = dim3(kAbThreads);
    cfg.dynamicSmemBytes = attn_block_smem_bytes();
    cfg.stream = c.stream;
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = kAbCluster;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = c.pdl ? 2 : 1;
}

// Opt in to the shared-memory size on the current device and prove that all n_kv_heads clusters can be resident at once
// (the CTAs of different clusters wait for one another's attention vector).
cudaError_t attn_block_prepare(int n_kv_heads, bool *co_resident) {
    *co_resident = false;
    cudaError_t e = cudaFuncSetAttribute(attn_block_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)attn_block_smem_bytes());
    if (e == cudaSuccess) e = cudaFuncSetAttribute(attn_block_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)attn_block_smem_bytes());
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute attr[2];
    attn_block_config(cfg, attr, LaunchCtx{nullptr, false, 0}, n_kv_heads);
    int n = 0;
    e = cudaOccupancyMaxActiveClusters(&n, attn_block_kernel<false>, &cfg);
    if (e != cudaSuccess) return e;
    *co_resident = n >= n_kv_heads;
    return cudaSuccess;
}

cudaError_t launch_attn_block(const LaunchCtx &c, const AttnBlockParams &p) {
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute attr[2];
    attn_block_config(cfg, attr, c, p.n_kv_heads);
    return p.trace ? cudaLaunchKernelEx(&cfg, attn_block_kernel<true>, p) : cudaLaunchKernelEx(&cfg, attn_block_kernel<false>, p);
}

}  // namespace hq
