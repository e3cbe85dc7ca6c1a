// hq_stream.cu — the streaming matrix-vector kernel of batch-1 decode: gate/up + SwiGLU (A2 + A7), down + residual
// (A8), final norm + LM head + argmax (A9) of SURVEY.md §8(a).
//
// These three products are 97 % of the bytes of a token (2.4 GB of bf16 weights) and pure HBM streams; the design
// keeps the stream independent of everything else the CTA does:
//   * grid = one CTA per SM; one producer thread copies weights with cp.async.bulk (TMA bulk copy, mbarrier complete_tx,
//     L2 evict-first) into a ring of 3 x 64 KB shared-memory stages.  A stage is ONE copy of 64 KB of consecutive weight
//     rows (two of 32 KB for gate | up): measured on B200 (bench.py --probes, profiles/r02_copy_size.md), an SM pulls
//     33 GB/s through 1 KB bulk copies, ~105 through 4 KB ones (58 next to busy consumer warps) and ~180 through >= 16 KB
//     ones, and the chip-wide stream rises from 6.85 to 7.26 TB/s.
//     The high per-SM rate matters behind the attention block: its 64 SMs join the following gate/up stream ~11 us
//     late and have to catch up with the 84 SMs whose CTAs were resident — and pre-filled their rings — meanwhile.
//   * weights are immutable, so the ring is filled BEFORE griddepcontrol.wait: under programmatic dependent launch the
//     CTA becomes resident while the previous kernel still runs and up to 192 KB per SM are on chip when the input
//     vector arrives.
//   * the 8 consumer warps each own a K slice of every stage and run it on the tensor cores: mma.sync m16n8k16 bf16,
//     A = weights, B = the input vector as two bf16 planes (x = hi + lo, 16 mantissa bits).  Rows of a stage lie a
//     multiple of 128 bytes apart (no padding: one contiguous copy), so ldmatrix would be 8-way bank conflicted.
//     Instead every lane loads 16 bytes of its two A rows with LDS.128 and the K index is PERMUTED (the dot product does
//     not care, as long as B is permuted alike): lane (g, t) of the fragment takes elements [8t, 8t + 8) of a 32-element
//     block of row g — words 0, 1 for the first k-tile, words 2, 3 for the second — and rows with odd g take the
//     neighbouring 64-byte block, which puts the two rows of a quarter-warp into different bank halves: conflict free.
//     The "different order for odd rows" is paid for with B columns: the 8 columns of the 16 x 8 operand hold up to four
//     (hi, lo) pairs of differently ordered / offset copies of x ("segments"), and a row's result is read from the pair
//     of D columns of its segment.  With rows longer than 2048 (down projection: 8192) a stage is 4 rows x 4 quarters of
//     K, one segment per quarter.  B lives in registers for the whole launch (32 per thread).
//   * per stage the 8 K-slice partial sums of a row meet in shared memory (one named barrier per 64 KB — every ~1.4 us
//     at stream rate, while the producer keeps the ring full), then <= 16 threads run the fused epilogue: SwiGLU -> bf16
//     hi/lo planes, residual add (one red.global.add.f32 per element and launch: order independent, bit reproducible),
//     or logits + packed-atomicMax argmax + step bookkeeping by the last CTA.
#include "hq_common.cuh"
#include "hq_internal.h"

namespace hq {

constexpr int kSgWarps = 8;                      // consumer warps
constexpr int kSgConsumers = 32 * kSgWarps;
constexpr int kSgThreads = kSgConsumers + 32;    // + producer warp
constexpr int kSgStages = 3;
constexpr int kSgStageBytes = 65536;
constexpr int kSgMaxBlocks = 8;                  // 32-element K blocks per warp and segment (segment <= 2048 elements)

struct SgShared {
    uint64_t full[kSgStages], empty[kSgStages];
    float dpart[2][kSgWarps][16];                // per stage parity, warp (K slice) and A row: partial dot products
    float red[kSgWarps];
};

__device__ __forceinline__ void sg_consumer_sync() { asm volatile("bar.sync 1, %0;" ::"n"(kSgConsumers) : "memory"); }
__device__ __forceinline__ void sg_mma_bf16(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
    asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint4 sg_lds128(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sg_red_add(float *p, float v) { asm volatile("red.global.add.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory"); }

// Geometry.  Q = 1 (K <= 2048): a stage is 16 rows x K (gate/up: 8 + 8); segments 0 / 1 = even / odd A rows (normal /
// swapped block order).  Q = 4 (K > 2048): a stage is 4 rows x K; A row m < 8 holds (weight row (m >> 1) & 3, K quarter
// m & 1), A row m + 8 the quarter 2 + (m & 1); segment = quarter, odd quarters in swapped block order.
struct SgGeom {
    int Q, rows_per_stage, n_stages_total, kseg, nblk, nb;   // kseg: K elements per segment; nblk: blocks per segment (even); nb: per warp
    uint32_t row_bytes;
};
__host__ __device__ inline int sg_rows_per_stage(int K, int mode) { return K > 2048 ? 4 : (mode == SGEMV_GATEUP ? 8 : 16); }
__device__ __forceinline__ SgGeom sg_geom(const SgemvParams &p) {
    SgGeom g;
    g.Q = p.K > 2048 ? 4 : 1;
    g.rows_per_stage = sg_rows_per_stage(p.K, p.mode);
    g.n_stages_total = (p.n_rows + g.rows_per_stage - 1) / g.rows_per_stage;
    g.kseg = p.K / g.Q;
    g.nblk = 2 * ((g.kseg + 63) / 64);
    g.nb = (g.nblk + kSgWarps - 1) / kSgWarps;
    g.row_bytes = (uint32_t)p.K * 2u;
    return g;
}

__global__ void __launch_bounds__(kSgThreads, 1) sgemv_kernel(const __grid_constant__ SgemvParams p) {
    extern __shared__ __align__(128) uint8_t sg_smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const SgGeom g = sg_geom(p);
    uint8_t *ring = sg_smem;
    SgShared &sh = *reinterpret_cast<SgShared *>(sg_smem + (size_t)kSgStages * kSgStageBytes);
    bf16 *xh = reinterpret_cast<bf16 *>(sg_smem + (size_t)kSgStages * kSgStageBytes + ((sizeof(SgShared) + 15) & ~(size_t)15));
    bf16 *xl = xh + p.K;                         // XIN_NORM only: the normalised input as two bf16 planes
    // contiguous share of the stages.  The first n_early CTAs are expected to be resident (and to have pre-filled their rings)
    // while the previous kernel still holds the other SMs: they take late_deficit stages more than the rest.
    int s0, s1;
    {
        const int S = g.n_stages_total, G = (int)gridDim.x, b = (int)blockIdx.x;
        const int ne = min(p.n_early, G);
        const float l = fmaxf(0.f, (float)S - (float)ne * p.late_deficit) / (float)G, e = ((float)S - l * (float)(G - ne)) / (float)max(ne, 1);
        auto cum = [&](int i) { return i >= G ? S : min(S, (int)((i <= ne ? (float)i * e : (float)ne * e + (float)(i - ne) * l) + 0.5f)); };
        s0 = cum(b);
        s1 = cum(b + 1);
    }

    if (tid == 0) {
        for (int s = 0; s < kSgStages; ++s) {
            mbar_init(&sh.full[s], 1);
            mbar_init(&sh.empty[s], kSgWarps);
        }
        mbar_fence_init();
        step_stamp(p.trace, p.trace_slot, 0);
        step_stamp(p.trace, p.trace_slot, 3);
    }
    // a segment whose length is not a multiple of 64 elements is read up to 126 bytes past its end (against zeros of B):
    // what lies there must not be uninitialised shared memory (NaN x 0).  Odd shapes only (e.g. ffn = 688).
    if (g.kseg % 64 != 0)
        for (int i = tid; i < kSgStages * kSgStageBytes / 16; i += kSgThreads) reinterpret_cast<uint4 *>(ring)[i] = make_uint4(0, 0, 0, 0);
    __syncthreads();
    pdl_launch_dependents();

    if (warp == kSgWarps) {
        // ---- producer: one thread, one bulk copy per stage (two for gate | up); never waits for the dependency ----------
        if (lane == 0) {
            const uint64_t pol = l2_policy_evict_first();
            unsigned n = 0;
            for (int st = s0; st < s1; ++st, ++n) {
                const int slot = n % kSgStages;
                unsigned spins = 0;
                while (!mbar_try_wait(&sh.empty[slot], ((n / kSgStages) & 1) ^ 1))
                    if (++spins == (1u << 26)) __trap();
                const int r0 = st * g.rows_per_stage;
                const uint32_t bytes = (uint32_t)min(g.rows_per_stage, p.n_rows - r0) * g.row_bytes;
                uint8_t *dst = ring + (size_t)slot * kSgStageBytes;
                if (p.mode == SGEMV_GATEUP) {
                    mbar_expect_tx(&sh.full[slot], 2u * bytes);
                    bulk_g2s_hint(dst, p.w0 + (size_t)r0 * p.K, bytes, &sh.full[slot], pol);
                    bulk_g2s_hint(dst + 8u * g.row_bytes, p.w1 + (size_t)r0 * p.K, bytes, &sh.full[slot], pol);
                } else {
                    mbar_expect_tx(&sh.full[slot], bytes);
                    bulk_g2s_hint(dst, p.w0 + (size_t)r0 * p.K, bytes, &sh.full[slot], pol);
                }
            }
        }
        return;
    }

    // ---- consumers ------------------------------------------------------------------------------------------------
    const int fg = lane >> 2, ft = lane & 3;      // fragment coordinates: A rows fg, fg + 8; B column fg; k pairs of ft
    // B: column n = fg -> segment n >> 1, plane n & 1
    const int b_seg = fg >> 1, b_plane = fg & 1;
    const bool b_on = g.Q == 4 || fg < 4;
    const int b_swap = b_seg & 1;
    const int b_xoff = g.Q == 4 ? b_seg * g.kseg : 0;
    // A: rows fg and fg + 8 of the fragment
    const int a_swap = fg & 1;
    uint32_t a_off0, a_off1;
    if (g.Q == 4) {
        a_off0 = (uint32_t)((fg >> 1) & 3) * g.row_bytes + (uint32_t)(fg & 1) * (uint32_t)g.kseg * 2u;
        a_off1 = a_off0 + 2u * (uint32_t)g.kseg * 2u;
    } else {
        a_off0 = (uint32_t)fg * g.row_bytes;
        a_off1 = a_off0 + 8u * g.row_bytes;
    }

    // XIN_NORM: thread t owns elements [8 (t + 256 j), + 8), j < 4, of the fp32 residual
    uint4 gq[4];
    if (p.xin_mode == SGEMV_XIN_NORM) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int e0 = (tid + j * kSgConsumers) * 8;
            gq[j] = e0 < p.K ? __ldg(reinterpret_cast<const uint4 *>(p.gain + e0)) : make_uint4(0, 0, 0, 0);   // immutable: before the wait
        }
    }
    pdl_wait();
    if (tid == 0) step_stamp(p.trace, p.trace_slot, 1);
    int pos = 0;
    if (p.mode == SGEMV_LMHEAD) pos = ld_act(p.pos);

    // B fragments of this warp's K blocks, in registers for the whole launch
    uint4 bq[kSgMaxBlocks];
    if (p.xin_mode == SGEMV_XIN_NORM) {
        // A2: RMSNorm of the fp32 residual -> two bf16 planes in shared memory
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
        sg_consumer_sync();
        const bf16 *plane = b_plane ? xl : xh;
#pragma unroll
        for (int i = 0; i < kSgMaxBlocks; ++i) {
            const int kb = (warp * g.nb + i) ^ b_swap, ks = kb * 32 + ft * 8;
            const bool ok = b_on && i < g.nb && warp * g.nb + i < g.nblk && ks < g.kseg;
            bq[i] = ok ? *reinterpret_cast<const uint4 *>(plane + b_xoff + ks) : make_uint4(0, 0, 0, 0);
        }
    } else {
        // the SwiGLU vector arrives as two bf16 planes (hi [K], lo [K]) written by the gate/up epilogue: straight from L2
        const bf16 *plane = reinterpret_cast<const bf16 *>(p.xin) + (b_plane ? p.K : 0);
#pragma unroll
        for (int i = 0; i < kSgMaxBlocks; ++i) {
            const int kb = (warp * g.nb + i) ^ b_swap, ks = kb * 32 + ft * 8;
            const bool ok = b_on && i < g.nb && warp * g.nb + i < g.nblk && ks < g.kseg;
            bq[i] = ok ? __ldcg(reinterpret_cast<const uint4 *>(plane + b_xoff + ks)) : make_uint4(0, 0, 0, 0);
        }
    }

    const uint32_t ring_addr = smem_addr_u32(ring);
    unsigned long long my_best = 0ull;
    int par = 0;
    unsigned n = 0;
    for (int st = s0; st < s1; ++st, ++n) {
        const int slot = n % kSgStages;
        {
            unsigned spins = 0;
            while (!mbar_try_wait(&sh.full[slot], (n / kSgStages) & 1))
                if (++spins == (1u << 26)) __trap();
        }
        float cc[4][4];
#pragma unroll
        for (int i = 0; i < 4; ++i) cc[i][0] = cc[i][1] = cc[i][2] = cc[i][3] = 0.f;
        const uint32_t base = ring_addr + (uint32_t)slot * kSgStageBytes + (uint32_t)ft * 16u;
        // all loads of the stage first (16 x LDS.128 per lane at most), then the MMAs on four accumulator chains
        uint4 a0[kSgMaxBlocks], a1[kSgMaxBlocks];
#pragma unroll
        for (int i = 0; i < kSgMaxBlocks; ++i) {
            const int blk = warp * g.nb + i;
            if (i < g.nb && blk < g.nblk) {   // warp-uniform
                const uint32_t off = (uint32_t)(blk ^ a_swap) * 64u;
                a0[i] = sg_lds128(base + a_off0 + off);
                a1[i] = sg_lds128(base + a_off1 + off);
            } else {
                a0[i] = a1[i] = make_uint4(0, 0, 0, 0);
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&sh.empty[slot]);   // the stage is in registers: the producer may refill the slot
#pragma unroll
        for (int i = 0; i < kSgMaxBlocks; ++i) {
            if (i < g.nb) {
                sg_mma_bf16(cc[(2 * i) & 3], a0[i].x, a1[i].x, a0[i].y, a1[i].y, bq[i].x, bq[i].y);
                sg_mma_bf16(cc[(2 * i + 1) & 3], a0[i].z, a1[i].z, a0[i].w, a1[i].w, bq[i].z, bq[i].w);
            }
        }
        float c[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) c[i] = (cc[0][i] + cc[1][i]) + (cc[2][i] + cc[3][i]);
        // C fragment: lane (fg, ft) holds D[fg][2 ft], D[fg][2 ft + 1], D[fg + 8][2 ft], D[fg + 8][2 ft + 1]; A row m reads
        // the (hi, lo) column pair of its segment
        if (g.Q == 4) {
            if (ft == (fg & 1)) sh.dpart[par][warp][fg] = c[0] + c[1];
            if (ft == 2 + (fg & 1)) sh.dpart[par][warp][fg + 8] = c[2] + c[3];
        } else if (ft == (fg & 1)) {
            sh.dpart[par][warp][fg] = c[0] + c[1];
            sh.dpart[par][warp][fg + 8] = c[2] + c[3];
        }
        sg_consumer_sync();
        if (tid < 16) {
            float tot = 0.f;
            if (g.Q == 4) {
                if (tid < 4) {
#pragma unroll
                    for (int w = 0; w < kSgWarps; ++w)
                        tot += (sh.dpart[par][w][2 * tid] + sh.dpart[par][w][2 * tid + 1]) + (sh.dpart[par][w][8 + 2 * tid] + sh.dpart[par][w][9 + 2 * tid]);
                }
            } else {
#pragma unroll
                for (int w = 0; w < kSgWarps; ++w) tot += sh.dpart[par][w][tid];
            }
            if (p.mode == SGEMV_GATEUP) {
                // A rows 0-7 gate, 8-15 up of units 8 st .. 8 st + 7
                const float up = __shfl_down_sync(0x0000ffffu, tot, 8);
                const int u = st * 8 + tid;
                if (tid < 8 && u < p.n_rows) {
                    const float a = silu_f(tot) * up;
                    bf16 hi, lo;
                    split_bf16(a, hi, lo);
                    p.out_planes[u] = hi;
                    p.out_planes[p.n_rows + u] = lo;
                }
            } else {
                const int r = st * g.rows_per_stage + tid;
                if (tid < g.rows_per_stage && r < p.n_rows) {
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
    if (tid == 0) step_stamp(p.trace, p.trace_slot, 2);

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
// K <= 2048: any multiple of 8 (blocks past the end of a row read the next row's weights against zeros of B); longer rows
// are cut into four quarters of whole 64-element block pairs and must fit one 64 KB stage four rows at a time
bool sgemv_shape_supported(int K) { return K > 0 && K % 8 == 0 && (K <= 2048 || (K % 256 == 0 && K <= 8192)); }

static size_t sgemv_smem_bytes(int norm_k) {
    return (size_t)kSgStages * kSgStageBytes + ((sizeof(SgShared) + 15) & ~(size_t)15) + (size_t)norm_k * 4 + 128;
}

cudaError_t sgemv_prepare() {
    return cudaFuncSetAttribute(sgemv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sgemv_smem_bytes(8192));
}

cudaError_t launch_sgemv(const LaunchCtx &c, const SgemvParams &p) {
    if (p.q0) return launch_sgemv_q4(c, p);
    if (!sgemv_shape_supported(p.K)) return cudaErrorInvalidValue;
    const int rps = sg_rows_per_stage(p.K, p.mode);
    const int n_stages = (p.n_rows + rps - 1) / rps;
    int grid = c.n_sms < n_stages ? c.n_sms : n_stages;
    if (p.max_ctas > 0 && p.max_ctas < grid) grid = p.max_ctas;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(kSgThreads);
    cfg.dynamicSmemBytes = sgemv_smem_bytes(p.xin_mode == SGEMV_XIN_NORM ? p.K : 0);
    cfg.stream = c.stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = c.pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, sgemv_kernel, p);
}

}  // namespace hq
