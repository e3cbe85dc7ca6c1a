// hq_stream.cu — the streaming matrix-vector kernel of batch-1 decode: gate/up + SwiGLU (A2 + A7), down + residual
// (A8), final norm + LM head + argmax (A9) of SURVEY.md §8(a).
//
// These three products are 97 % of the bytes of a token (2.4 GB of bf16 weights) and pure HBM streams; the design
// keeps the stream independent of everything else the CTA does:
//   * grid = one CTA per SM; a producer warp copies weight rows with cp.async.bulk (TMA bulk copy, mbarrier
//     complete_tx, L2 evict-first) into a shared-memory ring of ~200 KB.  Weights are immutable, so the ring is filled
//     BEFORE griddepcontrol.wait: the CTA becomes resident under programmatic dependent launch while the previous
//     kernel still runs, and the first ~200 KB per SM (up to 29 MB chip-wide) are already on chip when its input vector
//     arrives.  Behind the attention block, which streams little and occupies 64 of the 148 SMs, that is HBM time that
//     would otherwise idle.
//   * a ring stage holds one "group" of 16 weight rows x kc columns (kc = K when K <= 2048, else 1024), rows 16 bytes
//     apart from a multiple of 128 bytes so that ldmatrix reads are conflict free.  The 8 consumer warps each own a
//     K slice of the stage and run it on the tensor cores: mma.sync m16n8k16 bf16 with A = 16 rows x 16 columns of the
//     stage and B = the input vector as two bf16 planes (x = hi + lo, 16 mantissa bits) in columns 0 and 1 of the
//     16 x 8 operand.  One ldmatrix + one MMA per 256 weights instead of ~20 load/convert/FMA instructions: the
//     consumers can drain a full ring several times faster than HBM refills it, so they never limit the stream.
//   * per group the 8 K-slice partial sums of a row meet in shared memory (one named barrier per 16 rows — every
//     ~1.4 us at stream rate — while the producer keeps the ring full), then 16 threads run the fused epilogue.
//   * groups beyond the first ring-full of every CTA are handed out dynamically (one atomicAdd per group by the
//     producer, one group ahead): CTAs that start late — behind the attention block's clusters — take fewer groups.
//     One counter serves every launch of the stream: the CTA that draws the last ticket of a launch zeroes it.
#include <stdlib.h>
#include "hq_common.cuh"
#include "hq_internal.h"

namespace hq {

constexpr int kSgWarps = 8;                      // consumer warps
constexpr int kSgConsumers = 32 * kSgWarps;
constexpr int kSgThreads = kSgConsumers + 32;    // + producer warp
constexpr int kSgRowPad = 16;                    // bytes between the rows of a stage
constexpr int kSgMaxStages = 8;
constexpr int kSgSmemBudget = 232448 - 1024;     // 227 KB per CTA minus slack for alignment

struct SgShared {
    uint64_t full[kSgMaxStages], empty[kSgMaxStages];
    int group_of_stage[kSgMaxStages];            // which group the stage belongs to (dynamic hand-out), -1 = end of work
    float dpart[2][kSgWarps][16];                // per group parity, warp (K slice) and row: partial dot products
    float red[kSgWarps];
    unsigned long long best;                     // LM head: CTA-wide packed argmax
};

__device__ __forceinline__ void sg_consumer_sync() { asm volatile("bar.sync 1, %0;" ::"n"(kSgConsumers) : "memory"); }
__device__ __forceinline__ void sg_ldmatrix_x4(uint32_t (&r)[4], uint32_t addr) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];" : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void sg_mma_bf16(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void sg_red_add(float *p, float v) { asm volatile("red.global.add.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory"); }
__device__ __forceinline__ void sg_stamp(const SgemvParams &p, int which, bool is_min) {
    if (p.trace) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        if (is_min) atomicMin(p.trace + 4 * p.trace_slot + which, t);
        else atomicMax(p.trace + 4 * p.trace_slot + which, t);
    }
}

// geometry shared by producer and consumers
struct SgGeom {
    int n_groups, n_chunks, kc, stages, rows_per_group;
    uint32_t row_stride, stage_bytes;
    int static_groups;       // groups [cta * static_groups, ...) belong to this CTA; the rest are handed out dynamically
};
__device__ __forceinline__ SgGeom sg_geom(const SgemvParams &p) {
    SgGeom g;
    g.rows_per_group = p.mode == SGEMV_GATEUP ? 8 : 16;
    g.n_groups = (p.n_rows + g.rows_per_group - 1) / g.rows_per_group;
    g.kc = p.kc;
    g.n_chunks = (p.K + p.kc - 1) / p.kc;
    g.stages = p.stages;
    g.row_stride = (uint32_t)p.kc * 2u + (uint32_t)p.row_pad;
    g.stage_bytes = 16u * g.row_stride;
    g.static_groups = p.static_groups;
    return g;
}

// ---- producer warp ------------------------------------------------------------------------------------------------
// Walks this CTA's groups: first its static ones, then tickets from the dynamic counter.  Lane r copies row r of a stage.
__device__ void sg_producer(const SgemvParams &p, const SgGeom &g, uint8_t *ring, SgShared &sh) {
    const int lane = threadIdx.x & 31;
    const uint64_t pol = l2_policy_evict_first();
    unsigned n = 0;                                  // stages produced
    const int first = (int)blockIdx.x * g.static_groups;
    int s_left = min(g.static_groups, max(0, g.n_groups - first));
    const int dyn_base = min(g.n_groups, (int)gridDim.x * g.static_groups);
    const int n_dyn = g.n_groups - dyn_base;
    bool waited = false;
    int grp = s_left > 0 ? first : -1;
    int next_ticket = -1;                            // lane 0: dynamic ticket fetched one group ahead (-1 = none yet)
    for (;;) {
        if (grp < 0) {
            if (!p.ticket) break;
            // static share done: dynamic hand-out.  The counter is shared by every launch of the stream and is back at zero
            // once the previous launch has completed, i.e. it may be touched only after the dependency wait.
            if (!waited) { pdl_wait(); waited = true; }
            int t = next_ticket;
            if (lane == 0 && t < 0) t = (int)atomicAdd(p.ticket, 1u);
            t = __shfl_sync(0xffffffffu, t, 0);
            // every CTA fetches until its first out-of-range ticket: n_dyn + gridDim.x fetches per launch in all; whoever
            // draws the last one puts the counter back to zero for the next launch
            if (lane == 0 && t == n_dyn + (int)gridDim.x - 1) atomicExch(p.ticket, 0u);
            if (t >= n_dyn) break;
            grp = dyn_base + t;
            if (lane == 0) next_ticket = (int)atomicAdd(p.ticket, 1u);   // consumed one group later: its latency is hidden
        }
        const int rows_valid = min(g.rows_per_group, p.n_rows - grp * g.rows_per_group);
        for (int c = 0; c < g.n_chunks; ++c, ++n) {
            const int slot = n % g.stages;
            unsigned spins = 0;
            while (!mbar_try_wait(&sh.empty[slot], ((n / g.stages) & 1) ^ 1))
                if (++spins == (1u << 26)) __trap();
            const int k0 = c * g.kc;
            const uint32_t bytes = (uint32_t)min(g.kc, p.K - k0) * 2u;
            uint8_t *dst = ring + (size_t)slot * g.stage_bytes;
            if (lane == 0) {
                sh.group_of_stage[slot] = grp;
                mbar_expect_tx(&sh.full[slot], (p.mode == SGEMV_GATEUP ? 2u : 1u) * (uint32_t)rows_valid * bytes);
            }
            __syncwarp();
            if (p.mode == SGEMV_GATEUP) {
                if (lane < 16 && (lane & 7) < rows_valid) {
                    const bf16 *row = (lane < 8 ? p.w0 : p.w1) + (size_t)(grp * 8 + (lane & 7)) * p.K + k0;
                    bulk_g2s_hint(dst + (size_t)lane * g.row_stride, row, bytes, &sh.full[slot], pol);
                }
            } else if (lane < rows_valid) {
                bulk_g2s_hint(dst + (size_t)lane * g.row_stride, p.w0 + (size_t)(grp * 16 + lane) * p.K + k0, bytes, &sh.full[slot], pol);
            }
        }
        if (s_left > 1) { --s_left; ++grp; } else { s_left = 0; grp = -1; }
    }
    // end marker: one more stage that only tells the consumers to stop
    {
        const int slot = n % g.stages;
        unsigned spins = 0;
        while (!mbar_try_wait(&sh.empty[slot], ((n / g.stages) & 1) ^ 1))
            if (++spins == (1u << 26)) __trap();
        if (lane == 0) {
            sh.group_of_stage[slot] = -1;
            mbar_arrive(&sh.full[slot]);
        }
    }
}

// ---- the kernel ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kSgThreads, 1) sgemv_kernel(const __grid_constant__ SgemvParams p) {
    extern __shared__ __align__(128) uint8_t sg_smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const SgGeom g = sg_geom(p);
    uint8_t *ring = sg_smem;
    bf16 *xh = reinterpret_cast<bf16 *>(sg_smem + (size_t)g.stages * g.stage_bytes);
    bf16 *xl = xh + p.K;
    SgShared &sh = *reinterpret_cast<SgShared *>(reinterpret_cast<uint8_t *>(xl + p.K) + ((16 - ((2 * p.K * 2) & 15)) & 15));

    if (tid == 0) {
        for (int s = 0; s < g.stages; ++s) {
            mbar_init(&sh.full[s], 1);
            mbar_init(&sh.empty[s], kSgWarps);
        }
        sh.best = 0ull;
        mbar_fence_init();
    }
    // the 16-byte pads are read by the last k-tile of a row whose length is 8 mod 16: they must hold zeros
    for (int i = tid; i < g.stages * 16; i += kSgThreads)
        *reinterpret_cast<uint4 *>(ring + (size_t)(i >> 4) * g.stage_bytes + (size_t)(i & 15) * g.row_stride + (size_t)g.kc * 2) = make_uint4(0, 0, 0, 0);
    __syncthreads();
    if (tid == 0) sg_stamp(p, 0, true);
    pdl_launch_dependents();

    if (warp == kSgWarps) {
        sg_producer(p, g, ring, sh);
        return;
    }

    // ---- input vector -> two bf16 planes in shared memory (after the dependency wait) --------------------------------
    uint4 gq[4];
    if (p.xin_mode == SGEMV_XIN_NORM) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int e0 = (tid + j * kSgConsumers) * 8;
            gq[j] = e0 < p.K ? __ldg(reinterpret_cast<const uint4 *>(p.gain + e0)) : make_uint4(0, 0, 0, 0);   // immutable
        }
    }
    pdl_wait();
    if (tid == 0) sg_stamp(p, 1, true);
    int pos = 0;
    if (p.mode == SGEMV_LMHEAD) pos = ld_act(p.pos);
    if (p.xin_mode == SGEMV_XIN_NORM) {
        float v[4][8];
        float ss = 0.f;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int e0 = (tid + j * kSgConsumers) * 8;
#pragma unroll
            for (int i = 0; i < 8; ++i) v[j][i] = 0.f;
            if (e0 < p.K) {
                const float4 a = ld_act4(p.xin + e0), b = ld_act4(p.xin + e0 + 4);
                v[j][0] = a.x; v[j][1] = a.y; v[j][2] = a.z; v[j][3] = a.w; v[j][4] = b.x; v[j][5] = b.y; v[j][6] = b.z; v[j][7] = b.w;
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) ss = fmaf(v[j][i], v[j][i], ss);
        }
        ss = warp_sum(ss);
        if (lane == 0) sh.red[warp] = ss;
        sg_consumer_sync();
        float tot = 0.f;
#pragma unroll
        for (int k = 0; k < kSgWarps; ++k) tot += sh.red[k];
        const float inv = 1.0f / sqrtf(tot / (float)p.K + p.eps);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int e0 = (tid + j * kSgConsumers) * 8;
            if (e0 < p.K) {
                const uint32_t gg[4] = {gq[j].x, gq[j].y, gq[j].z, gq[j].w};
                uint32_t h[4], l[4];
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    split_bf16x2(v[j][2 * i] * (inv * bf16lo(gg[i])), v[j][2 * i + 1] * (inv * bf16hi(gg[i])), h[i], l[i]);
                *reinterpret_cast<uint4 *>(xh + e0) = make_uint4(h[0], h[1], h[2], h[3]);
                *reinterpret_cast<uint4 *>(xl + e0) = make_uint4(l[0], l[1], l[2], l[3]);
            }
        }
    } else {
        // the SwiGLU vector arrives as two bf16 planes already (written by the gate/up epilogue)
        const uint4 *src = reinterpret_cast<const uint4 *>(p.xin);
        const int n16 = 2 * (p.K / 8);
        for (int i0 = 0; i0 < n16; i0 += 8 * kSgConsumers) {
            uint4 v[8];   // all loads in flight before the first store
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int i = i0 + j * kSgConsumers + tid;
                v[j] = i < n16 ? __ldcg(src + i) : make_uint4(0, 0, 0, 0);
            }
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int i = i0 + j * kSgConsumers + tid;
                if (i < n16) reinterpret_cast<uint4 *>(xh)[i] = v[j];
            }
        }
    }
    sg_consumer_sync();

    // ---- stages ---------------------------------------------------------------------------------------------------
    const int nkt_stage = (g.kc + 15) / 16, nkt = (nkt_stage + kSgWarps - 1) / kSgWarps;   // k-tiles per stage / per warp
    const int bn = lane >> 2, bk = (lane & 3) * 2;
    const bf16 *bsrc = bn == 0 ? xh : xl;
    const bool b_on = bn < 2;
    const uint32_t a_lane = (uint32_t)((lane & 7) + ((lane >> 3) & 1) * 8) * g.row_stride + (uint32_t)(lane >> 4) * 16u + (uint32_t)(warp * nkt) * 32u;
    const uint32_t ring_addr = smem_addr_u32(ring);
    unsigned long long my_best = 0ull;
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    int chunk = 0, par = 0;
    for (unsigned n = 0;; ++n) {
        const int slot = n % g.stages;
        {
            unsigned spins = 0;
            while (!mbar_try_wait(&sh.full[slot], (n / g.stages) & 1))
                if (++spins == (1u << 26)) __trap();
        }
        const int grp = sh.group_of_stage[slot];
        if (grp < 0) break;
        {
            float cc[4][4];
#pragma unroll
            for (int i = 0; i < 4; ++i) cc[i][0] = cc[i][1] = cc[i][2] = cc[i][3] = 0.f;
            const int k_base = chunk * g.kc;
            const int kt_end = (min(g.kc, p.K - k_base) + 15) / 16;   // valid k-tiles of this chunk
            const uint32_t a_base = ring_addr + (uint32_t)slot * g.stage_bytes + a_lane;
            const int t0 = warp * nkt;
            // batches of 4 k-tiles, software pipelined: the fragments of batch b + 1 are requested before the MMAs of batch
            // b are issued (an MMA right behind its own ldmatrix waits ~30 cycles for it, 16 times per stage)
            uint32_t fa[2][4][4], fb[2][4][2];
            auto load_batch = [&](uint32_t (&A)[4][4], uint32_t (&B)[4][2], int i4) {
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int i = i4 + j;
                    const int k0 = k_base + (t0 + i) * 16 + bk;
                    const bool on = i < nkt && t0 + i < kt_end;   // warp-uniform
                    B[j][0] = (on && b_on && k0 < p.K) ? *reinterpret_cast<const uint32_t *>(bsrc + k0) : 0u;
                    B[j][1] = (on && b_on && k0 + 8 < p.K) ? *reinterpret_cast<const uint32_t *>(bsrc + k0 + 8) : 0u;
                    if (on) sg_ldmatrix_x4(A[j], a_base + (uint32_t)i * 32u);
                    else A[j][0] = A[j][1] = A[j][2] = A[j][3] = 0u;
                }
            };
            auto mma_batch = [&](const uint32_t (&A)[4][4], const uint32_t (&B)[4][2]) {
#pragma unroll
                for (int j = 0; j < 4; ++j) sg_mma_bf16(cc[j], A[j], B[j][0], B[j][1]);   // zero fragments add nothing
            };
            load_batch(fa[0], fb[0], 0);
#pragma unroll 1
            for (int i4 = 0; i4 < nkt; i4 += 8) {
                if (i4 + 4 < nkt) load_batch(fa[1], fb[1], i4 + 4);
                mma_batch(fa[0], fb[0]);
                if (i4 + 4 < nkt) {
                    if (i4 + 8 < nkt) load_batch(fa[0], fb[0], i4 + 8);
                    mma_batch(fa[1], fb[1]);
                }
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) acc[i] += (cc[0][i] + cc[1][i]) + (cc[2][i] + cc[3][i]);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&sh.empty[slot]);
        if (++chunk < g.n_chunks) continue;
        chunk = 0;
        // group complete: C fragment holds (row lane >> 2, cols 2 (lane & 3), +1) in acc[0], acc[1] and row + 8 in acc[2], acc[3];
        // columns 0 and 1 are the two planes of the input
        if ((lane & 3) == 0) {
            sh.dpart[par][warp][lane >> 2] = acc[0] + acc[1];
            sh.dpart[par][warp][(lane >> 2) + 8] = acc[2] + acc[3];
        }
        acc[0] = acc[1] = acc[2] = acc[3] = 0.f;
        sg_consumer_sync();
        if (tid < 16) {
            float tot = 0.f;
#pragma unroll
            for (int w = 0; w < kSgWarps; ++w) tot += sh.dpart[par][w][tid];
            if (p.mode == SGEMV_GATEUP) {
                // rows 0-7 gate, 8-15 up of units 8 grp .. 8 grp + 7
                const float up = __shfl_down_sync(0x0000ffffu, tot, 8);
                const int u = grp * 8 + tid;
                if (tid < 8 && u < p.n_rows) {
                    const float a = silu_f(tot) * up;
                    bf16 hi, lo;
                    split_bf16(a, hi, lo);
                    p.out_planes[u] = hi;
                    p.out_planes[p.n_rows + u] = lo;
                }
            } else {
                const int r = grp * 16 + tid;
                if (r < p.n_rows) {
                    if (p.mode == SGEMV_RESID) {
                        sg_red_add(p.out + r, tot);   // exactly one add per element and launch: order independent
                    } else {
                        p.out[r] = tot;
                        const unsigned long long key = pack_argmax(tot, r);
                        my_best = my_best > key ? my_best : key;
                    }
                }
            }
        }
        par ^= 1;
    }
    if (tid == 0) sg_stamp(p, 2, false);

    if (p.mode == SGEMV_LMHEAD && warp == 0) {
        // fused argmax (A9): per-CTA best -> one packed 64-bit atomicMax; the last CTA to finish publishes the token and
        // advances the position (device-resident step state)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const unsigned long long other = __shfl_xor_sync(0xffffffffu, my_best, o);
            my_best = my_best > other ? my_best : other;
        }
        if (lane == 0) {
            if (my_best) atomicMax(p.best, my_best);
            __threadfence();
            const unsigned int ticket = atomicAdd(p.counter, 1u);
            if (ticket == gridDim.x - 1) {
                __threadfence();
                const unsigned long long win = atomicExch(p.best, 0ull);
                const int tok = unpack_argmax_idx(win);
                *p.cur_tok = tok;
                p.tok_hist[pos + p.pos_inc] = tok;
                *p.pos_rw = pos + p.pos_inc;
                *p.counter = 0u;
            }
        }
    }
}

// ---- host side ------------------------------------------------------------------------------------------------------
// K <= 2048: one chunk per row, the zeroed pad behind it covers a half k-tile; longer rows must be whole k-tiles
bool sgemv_shape_supported(int K) { return K > 0 && K % 8 == 0 && K <= 8192 && (K <= 2048 || K % 16 == 0); }

// ring geometry for an input length K: chunk length, stages, dynamic shared memory
static void sgemv_plan(int K, int *kc, int *stages, size_t *smem) {
    *kc = K <= 2048 ? K : 1024;
    const size_t stage = 16 * ((size_t)*kc * 2 + 128);
    const size_t fixed = (size_t)K * 4 + 16 + sizeof(SgShared) + 128;
    int s = (int)((kSgSmemBudget - fixed) / stage);
    if (s > kSgMaxStages) s = kSgMaxStages;
    *stages = s;
    *smem = (size_t)s * stage + fixed;
}

cudaError_t sgemv_prepare() {
    return cudaFuncSetAttribute(sgemv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSgSmemBudget);
}

cudaError_t launch_sgemv(const LaunchCtx &c, SgemvParams p) {
    size_t smem;
    sgemv_plan(p.K, &p.kc, &p.stages, &smem);
    p.row_pad = getenv("HQ_SG_PAD") ? atoi(getenv("HQ_SG_PAD")) : kSgRowPad;
    p.dbg = getenv("HQ_SG_DBG") ? atoi(getenv("HQ_SG_DBG")) : 0;
    const int rpg = p.mode == SGEMV_GATEUP ? 8 : 16;
    const int n_groups = (p.n_rows + rpg - 1) / rpg;
    const int n_chunks = (p.K + p.kc - 1) / p.kc;
    int grid = c.n_sms < n_groups ? c.n_sms : n_groups;
    // static share: what one ring holds (requested before the dependency wait), at most an even split
    int sg = p.stages / n_chunks;
    if (sg < 1) sg = 1;
    if (!p.ticket || sg * grid > n_groups) sg = p.ticket ? n_groups / grid : (n_groups + grid - 1) / grid;
    p.static_groups = sg;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(kSgThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = c.stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = c.pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, sgemv_kernel, p);
}

}  // namespace hq
