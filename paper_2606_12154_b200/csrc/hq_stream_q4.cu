// hq_stream_q4.cu — 4-bit weight-only streaming GEMV and the "hq4" quantiser.
//
// The paper's mouth model runs at 4-bit quantisation; its runtime's format is neither described
// nor used.  hq4 is this library's own group format (include/hq.h):
//   * a weight row of K elements (K % 32 == 0) is cut into groups of 32 consecutive elements;
//   * group exponent e = the smallest integer with max|w| <= 7 * 2^e (-126 for an all-zero group), stored as E = e + 127;
//   * code q = round-half-to-even(w / 2^e) in [-8, 7], stored as the nibble q + 8: element 2j of a row in the low nibble
//     of byte j, element 2j + 1 in the high nibble (a 32-bit word = 8 consecutive elements, nibble i = element i);
//   * the weight computed with is w' = q * 2^e, exactly representable in bf16 — so the tensor-core paths (prefill,
//     batched decode) run unchanged on a dequantised bf16 copy and see the same numbers as this kernel.
//
// The kernel is hq_stream.cu's with 4.25 bits per weight in the ring: a stage is 16 weight rows (gate/up: 8 + 8; rows
// longer than 2048: 4 rows x 4 quarters of K) = 16 KB of codes + 1 KB of exponent bytes, fetched by one bulk copy each
// (two each for gate | up) into a ring of 10 stages.  Lane (g, t) of the MMA fragment loads 16 bytes = one whole group of
// 32 codes of A rows g and g + 8 and expands them in registers: (word >> s) & 0x000F000F | 0x43004300 is the bf16 pair
// (128 + v_a, 128 + v_b) of two nibbles, and one fma.rn.bf16x2 with (2^e, 2^e) and (-136 * 2^e, -136 * 2^e) turns it into
// (q_a * 2^e, q_b * 2^e) — exact, since every intermediate has <= 8 significant bits.  Which nibbles feed which k-tile is a
// permutation of K applied to the B operand alike (B: the input vector as bf16 planes hi | lo, gathered once per launch
// into registers); odd rows take the neighbouring 64-byte block (bank conflicts), paid for with B columns as in hq_stream.cu.
#include "hq_common.cuh"
#include "hq_internal.h"

namespace hq {

constexpr int kQ4Warps = 8;
constexpr int kQ4Consumers = 32 * kQ4Warps;
constexpr int kQ4Threads = kQ4Consumers + 32;
constexpr int kQ4Stages = 10;
constexpr int kQ4CodeBytes = 16384;              // codes of one stage: 16 rows x 2048 elements / 2 (or 4 rows x 8192 / 2)
constexpr int kQ4ExpBytes = 1024;                // exponent bytes of one stage
constexpr int kQ4StageBytes = kQ4CodeBytes + kQ4ExpBytes;
constexpr int kQ4Batch = 4;                      // stages between two consumer barriers (a 17 KB stage is too little work per barrier)
constexpr int kQ4MaxSb = 2;                      // 128-element superblocks per warp and segment (segment <= 2048 elements)

struct Q4Shared {
    uint64_t full[kQ4Stages], empty[kQ4Stages];
    float dpart[2][kQ4Batch][kQ4Warps][16];
    float red[kQ4Warps];
};

__device__ __forceinline__ void q4_consumer_sync() { asm volatile("bar.sync 1, %0;" ::"n"(kQ4Consumers) : "memory"); }
__device__ __forceinline__ void q4_mma_bf16(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
    asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint4 q4_lds128(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint32_t q4_lds8(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}
// two nibbles of w (bits s .. s+3 and s+16 .. s+19) -> bf16x2 (q_lo * 2^e, q_hi * 2^e): (128 + v) * 2^e - 136 * 2^e, exact
__device__ __forceinline__ uint32_t q4_expand(uint32_t w, int s, uint32_t scale2, uint32_t off2) {
    uint32_t m;   // ((w >> s) & 0x000F000F) | 0x43004300 in one LOP3 (truth table (a & b) | c = 0xEA)
    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(m) : "r"(w >> s), "r"(0x000F000Fu), "r"(0x43004300u));
    uint32_t r;
    asm("fma.rn.bf16x2 %0, %1, %2, %3;" : "=r"(r) : "r"(m), "r"(scale2), "r"(off2));
    return r;
}
__device__ __forceinline__ void q4_red_add(float *p, float v) { asm volatile("red.global.add.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory"); }

struct Q4Geom {
    int Q, rows_per_stage, n_stages_total, kseg, nsb, nb;   // kseg: elements per segment; nsb: superblocks per segment (even); nb: per warp
    uint32_t row_code_bytes, row_exp_bytes;
};
__host__ __device__ inline int q4_rows_per_stage(int K, int mode) { return K > 2048 ? 4 : (mode == SGEMV_GATEUP ? 8 : 16); }
__device__ __forceinline__ Q4Geom q4_geom(const SgemvParams &p) {
    Q4Geom g;
    g.Q = p.K > 2048 ? 4 : 1;
    g.rows_per_stage = q4_rows_per_stage(p.K, p.mode);
    g.n_stages_total = (p.n_rows + g.rows_per_stage - 1) / g.rows_per_stage;
    g.kseg = p.K / g.Q;
    g.nsb = 2 * ((g.kseg + 255) / 256);
    g.nb = (g.nsb + kQ4Warps - 1) / kQ4Warps;
    g.row_code_bytes = (uint32_t)p.K / 2u;
    g.row_exp_bytes = (uint32_t)p.K / 32u;
    return g;
}

__global__ void __launch_bounds__(kQ4Threads, 1) sgemv_q4_kernel(const __grid_constant__ SgemvParams p) {
    extern __shared__ __align__(128) uint8_t q4_smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const Q4Geom g = q4_geom(p);
    uint8_t *ring = q4_smem;
    Q4Shared &sh = *reinterpret_cast<Q4Shared *>(q4_smem + (size_t)kQ4Stages * kQ4StageBytes);
    bf16 *xh = reinterpret_cast<bf16 *>(q4_smem + (size_t)kQ4Stages * kQ4StageBytes + ((sizeof(Q4Shared) + 15) & ~(size_t)15));
    bf16 *xl = xh + p.K;
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
        for (int s = 0; s < kQ4Stages; ++s) {
            mbar_init(&sh.full[s], 1);
            mbar_init(&sh.empty[s], kQ4Warps);
        }
        mbar_fence_init();
        step_stamp(p.trace, p.trace_slot, 0);
        step_stamp(p.trace, p.trace_slot, 3);
    }
    // segments that are not whole 256-element superblock pairs are read past their end (against zeros of B): the ring must not
    // hold uninitialised bit patterns there (an exponent byte of 255 would expand to NaN).  Odd shapes only.
    if (g.kseg % 256 != 0)
        for (int i = tid; i < kQ4Stages * kQ4StageBytes / 16; i += kQ4Threads) reinterpret_cast<uint4 *>(ring)[i] = make_uint4(0x88888888u, 0x88888888u, 0x88888888u, 0x88888888u);
    __syncthreads();
    pdl_launch_dependents();

    if (warp == kQ4Warps) {
        if (lane == 0) {
            const uint64_t pol = l2_policy_evict_first();
            unsigned n = 0;
            for (int st = s0; st < s1; ++st, ++n) {
                const int slot = n % kQ4Stages;
                unsigned spins = 0;
                while (!mbar_try_wait(&sh.empty[slot], ((n / kQ4Stages) & 1) ^ 1))
                    if (++spins == (1u << 26)) __trap();
                const int r0 = st * g.rows_per_stage;
                const uint32_t rows = (uint32_t)min(g.rows_per_stage, p.n_rows - r0);
                const uint32_t cb = rows * g.row_code_bytes, eb = rows * g.row_exp_bytes;
                uint8_t *dst = ring + (size_t)slot * kQ4StageBytes;
                if (p.mode == SGEMV_GATEUP) {
                    mbar_expect_tx(&sh.full[slot], 2u * (cb + eb));
                    bulk_g2s_hint(dst, p.q0 + (size_t)r0 * g.row_code_bytes, cb, &sh.full[slot], pol);
                    bulk_g2s_hint(dst + 8u * g.row_code_bytes, p.q1 + (size_t)r0 * g.row_code_bytes, cb, &sh.full[slot], pol);
                    bulk_g2s_hint(dst + kQ4CodeBytes, p.e0 + (size_t)r0 * g.row_exp_bytes, eb, &sh.full[slot], pol);
                    bulk_g2s_hint(dst + kQ4CodeBytes + 8u * g.row_exp_bytes, p.e1 + (size_t)r0 * g.row_exp_bytes, eb, &sh.full[slot], pol);
                } else {
                    mbar_expect_tx(&sh.full[slot], cb + eb);
                    bulk_g2s_hint(dst, p.q0 + (size_t)r0 * g.row_code_bytes, cb, &sh.full[slot], pol);
                    bulk_g2s_hint(dst + kQ4CodeBytes, p.e0 + (size_t)r0 * g.row_exp_bytes, eb, &sh.full[slot], pol);
                }
            }
        }
        return;
    }

    // ---- consumers ------------------------------------------------------------------------------------------------
    const int fg = lane >> 2, ft = lane & 3;
    const int b_seg = fg >> 1, b_plane = fg & 1;
    const bool b_on = g.Q == 4 || fg < 4;
    const int b_swap = b_seg & 1;
    const int b_xoff = g.Q == 4 ? b_seg * g.kseg : 0;
    const int a_swap = fg & 1;
    // byte offsets of A rows fg and fg + 8 inside the stage: codes and exponent bytes
    uint32_t a_c0, a_c1, a_e0, a_e1;
    if (g.Q == 4) {
        a_c0 = (uint32_t)((fg >> 1) & 3) * g.row_code_bytes + (uint32_t)(fg & 1) * (uint32_t)(g.kseg / 2);
        a_c1 = a_c0 + 2u * (uint32_t)(g.kseg / 2);
        a_e0 = (uint32_t)((fg >> 1) & 3) * g.row_exp_bytes + (uint32_t)(fg & 1) * (uint32_t)(g.kseg / 32);
        a_e1 = a_e0 + 2u * (uint32_t)(g.kseg / 32);
    } else {
        a_c0 = (uint32_t)fg * g.row_code_bytes;
        a_c1 = a_c0 + 8u * g.row_code_bytes;
        a_e0 = (uint32_t)fg * g.row_exp_bytes;
        a_e1 = a_e0 + 8u * g.row_exp_bytes;
    }

    uint4 gq[4];
    if (p.xin_mode == SGEMV_XIN_NORM) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int e0 = (tid + j * kQ4Consumers) * 8;
            gq[j] = e0 < p.K ? __ldg(reinterpret_cast<const uint4 *>(p.gain + e0)) : make_uint4(0, 0, 0, 0);
        }
    }
    pdl_wait();
    if (tid == 0) step_stamp(p.trace, p.trace_slot, 1);
    int pos = 0;
    if (p.mode == SGEMV_LMHEAD) pos = ld_act(p.pos);

    // the input as two bf16 planes in shared memory (XIN_NORM: RMSNorm first; XIN_PLANES: copied from the gate/up epilogue's output)
    if (p.xin_mode == SGEMV_XIN_NORM) {
        float v[4][8];
        float ss = 0.f;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int e0 = (tid + j * kQ4Consumers) * 8;
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
        q4_consumer_sync();
        float tot = 0.f;
#pragma unroll
        for (int k = 0; k < kQ4Warps; ++k) tot += sh.red[k];
        const float inv = 1.0f / sqrtf(tot / (float)p.K + p.eps);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int e0 = (tid + j * kQ4Consumers) * 8;
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
    }
    q4_consumer_sync();

    // B fragments, gathered once: superblock sb, word i, half h feeds MMA 2 i + h with the elements (8 i + 2 h, + 4) and
    // (8 i + 2 h + 1, + 5) of this lane's group (the same permutation the nibble extraction applies to A)
    uint32_t bq[kQ4MaxSb][8][2];
    {
        // XIN_NORM: from the planes just written to shared memory; XIN_PLANES: straight from the gate/up epilogue's output in L2
        const bf16 *plane = p.xin_mode == SGEMV_XIN_NORM ? (b_plane ? xl : xh) : reinterpret_cast<const bf16 *>(p.xin) + (b_plane ? p.K : 0);
#pragma unroll
        for (int s = 0; s < kQ4MaxSb; ++s) {
            const int sb = warp * g.nb + s;
            const int base = ((sb ^ b_swap) * 4 + ft) * 32;             // first element of the group inside the segment
            const bool ok = b_on && s < g.nb && sb < g.nsb && base < g.kseg;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                uint4 u = make_uint4(0, 0, 0, 0);                       // elements 8 i .. 8 i + 7 of the group
                if (ok) {
                    const uint4 *src = reinterpret_cast<const uint4 *>(plane + b_xoff + base + 8 * i);
                    u = p.xin_mode == SGEMV_XIN_NORM ? *src : __ldcg(src);
                }
                bq[s][2 * i][0] = __byte_perm(u.x, u.z, 0x5410);        // (e0, e4)
                bq[s][2 * i][1] = __byte_perm(u.x, u.z, 0x7632);        // (e1, e5)
                bq[s][2 * i + 1][0] = __byte_perm(u.y, u.w, 0x5410);    // (e2, e6)
                bq[s][2 * i + 1][1] = __byte_perm(u.y, u.w, 0x7632);    // (e3, e7)
            }
        }
    }

    const uint32_t ring_addr = smem_addr_u32(ring);
    unsigned long long my_best = 0ull;
    int par = 0;
    unsigned n = 0;
    for (int st0 = s0; st0 < s1; st0 += kQ4Batch) {
        const int nbatch = min(kQ4Batch, s1 - st0);
#pragma unroll 1
        for (int j = 0; j < nbatch; ++j, ++n) {
            const int slot = n % kQ4Stages;
            {
                unsigned spins = 0;
                while (!mbar_try_wait(&sh.full[slot], (n / kQ4Stages) & 1))
                    if (++spins == (1u << 26)) __trap();
            }
            const uint32_t base = ring_addr + (uint32_t)slot * kQ4StageBytes;
            uint4 c0[kQ4MaxSb], c1[kQ4MaxSb];
            uint32_t x0[kQ4MaxSb], x1[kQ4MaxSb];
#pragma unroll
            for (int s = 0; s < kQ4MaxSb; ++s) {
                const int sb = warp * g.nb + s;
                if (s < g.nb && sb < g.nsb) {   // warp-uniform
                    const uint32_t blk = (uint32_t)(sb ^ a_swap);
                    c0[s] = q4_lds128(base + a_c0 + blk * 64u + (uint32_t)ft * 16u);
                    c1[s] = q4_lds128(base + a_c1 + blk * 64u + (uint32_t)ft * 16u);
                    x0[s] = q4_lds8(base + kQ4CodeBytes + a_e0 + blk * 4u + (uint32_t)ft);
                    x1[s] = q4_lds8(base + kQ4CodeBytes + a_e1 + blk * 4u + (uint32_t)ft);
                } else {
                    c0[s] = c1[s] = make_uint4(0x88888888u, 0x88888888u, 0x88888888u, 0x88888888u);
                    x0[s] = x1[s] = 1u;
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&sh.empty[slot]);
            float cc[4][4];
#pragma unroll
            for (int i = 0; i < 4; ++i) cc[i][0] = cc[i][1] = cc[i][2] = cc[i][3] = 0.f;
#pragma unroll
            for (int s = 0; s < kQ4MaxSb; ++s) {
                if (s < g.nb) {
                    // (2^e, 2^e) and (-136 * 2^e, -136 * 2^e) as bf16 pairs: exponent field E, resp. sign | E + 7 | mantissa 0001000
                    const uint32_t s0b = x0[s] << 7, s1b = x1[s] << 7;
                    const uint32_t sc0 = s0b | (s0b << 16), sc1 = s1b | (s1b << 16);
                    const uint32_t o0b = 0x8008u | ((x0[s] + 7u) << 7), o1b = 0x8008u | ((x1[s] + 7u) << 7);
                    const uint32_t of0 = o0b | (o0b << 16), of1 = o1b | (o1b << 16);
                    const uint32_t w0[4] = {c0[s].x, c0[s].y, c0[s].z, c0[s].w}, w1[4] = {c1[s].x, c1[s].y, c1[s].z, c1[s].w};
#pragma unroll
                    for (int i = 0; i < 4; ++i)
#pragma unroll
                        for (int h = 0; h < 2; ++h)
                            q4_mma_bf16(cc[(2 * i + h) & 3], q4_expand(w0[i], 8 * h, sc0, of0), q4_expand(w1[i], 8 * h, sc1, of1),
                                        q4_expand(w0[i], 8 * h + 4, sc0, of0), q4_expand(w1[i], 8 * h + 4, sc1, of1), bq[s][2 * i + h][0],
                                        bq[s][2 * i + h][1]);
                }
            }
            float c[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) c[i] = (cc[0][i] + cc[1][i]) + (cc[2][i] + cc[3][i]);
            if (g.Q == 4) {
                if (ft == (fg & 1)) sh.dpart[par][j][warp][fg] = c[0] + c[1];
                if (ft == 2 + (fg & 1)) sh.dpart[par][j][warp][fg + 8] = c[2] + c[3];
            } else if (ft == (fg & 1)) {
                sh.dpart[par][j][warp][fg] = c[0] + c[1];
                sh.dpart[par][j][warp][fg + 8] = c[2] + c[3];
            }
        }
        q4_consumer_sync();
        if (warp < 2) {   // 64 epilogue threads: (stage j = tid >> 4 of the batch, row tid & 15); whole warps, for the shuffle
            const int j = tid >> 4, t16 = tid & 15, st = st0 + j;
            const bool live = j < nbatch;
            float tot = 0.f;
            if (live) {
                if (g.Q == 4) {
                    if (t16 < 4) {
#pragma unroll
                        for (int w = 0; w < kQ4Warps; ++w)
                            tot += (sh.dpart[par][j][w][2 * t16] + sh.dpart[par][j][w][2 * t16 + 1]) + (sh.dpart[par][j][w][8 + 2 * t16] + sh.dpart[par][j][w][9 + 2 * t16]);
                    }
                } else {
#pragma unroll
                    for (int w = 0; w < kQ4Warps; ++w) tot += sh.dpart[par][j][w][t16];
                }
            }
            const float up = __shfl_down_sync(0xffffffffu, tot, 8);   // rows 8-15 of a gate | up stage are the up rows
            if (live) {
                if (p.mode == SGEMV_GATEUP) {
                    const int u = st * 8 + t16;
                    if (t16 < 8 && u < p.n_rows) {
                        const float a = silu_f(tot) * up;
                        bf16 hi, lo;
                        split_bf16(a, hi, lo);
                        p.out_planes[u] = hi;
                        p.out_planes[p.n_rows + u] = lo;
                    }
                } else {
                    const int r = st * g.rows_per_stage + t16;
                    if (t16 < g.rows_per_stage && r < p.n_rows) {
                        if (p.mode == SGEMV_RESID) {
                            q4_red_add(p.out + r, tot);
                        } else {
                            p.out[r] = tot;
                            const unsigned long long key = pack_argmax(tot, r);
                            my_best = my_best > key ? my_best : key;
                        }
                    }
                }
            }
        }
        par ^= 1;
    }
    if (tid == 0) step_stamp(p.trace, p.trace_slot, 2);

    if (p.mode == SGEMV_LMHEAD && warp < 2) {   // the epilogue threads (tid < 64) hold the candidates
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const unsigned long long other = __shfl_xor_sync(0xffffffffu, my_best, o);
            my_best = my_best > other ? my_best : other;
        }
        if (lane == 0 && my_best) atomicMax(p.best, my_best);
        asm volatile("bar.sync 2, 64;" ::: "memory");   // both warps' candidates are out before the ticket
        if (warp == 0 && lane == 0) {
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

// ---- quantiser / dequantiser --------------------------------------------------------------------------------------
// one thread per group of 32 elements
__global__ void __launch_bounds__(256) q4_quantize_kernel(const bf16 *__restrict__ w, size_t n_groups, uint8_t *__restrict__ codes,
                                                          uint8_t *__restrict__ exps) {
    const size_t gi = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gi >= n_groups) return;
    const uint4 *src = reinterpret_cast<const uint4 *>(w + gi * 32);
    uint32_t u[16];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const uint4 v = src[i];
        u[4 * i] = v.x; u[4 * i + 1] = v.y; u[4 * i + 2] = v.z; u[4 * i + 3] = v.w;
    }
    // max |w| as fp32 bits: bf16 -> fp32 is a 16-bit shift, and |x| orders like its bit pattern
    uint32_t m = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        m = max(m, (u[i] << 16) & 0x7FFFFFFFu);
        m = max(m, u[i] & 0x7FFF0000u);
    }
    // smallest e with m <= 7 * 2^e = 1.75 * 2^(e + 2): exponent of m minus 2 when its mantissa is <= 0.75, else minus 1
    int e;
    if (m == 0u) {
        e = -126;
    } else {
        const int ex = (int)(m >> 23) - 127;
        e = ((m & 0x007FFFFFu) <= 0x00600000u) ? ex - 2 : ex - 1;
        e = max(-126, min(120, e));
    }
    const float inv = __uint_as_float((uint32_t)(127 - e) << 23);   // 2^-e, exact
    uint32_t packed[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        uint32_t wv = 0;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t pr = u[4 * i + j];
            const int q0 = max(-8, min(7, (int)rintf(bf16lo(pr) * inv))), q1 = max(-8, min(7, (int)rintf(bf16hi(pr) * inv)));
            wv |= (uint32_t)(q0 + 8) << (8 * j) | (uint32_t)(q1 + 8) << (8 * j + 4);
        }
        packed[i] = wv;
    }
    *reinterpret_cast<uint4 *>(codes + gi * 16) = make_uint4(packed[0], packed[1], packed[2], packed[3]);
    exps[gi] = (uint8_t)(e + 127);
}

__global__ void __launch_bounds__(256) q4_dequantize_kernel(const uint8_t *__restrict__ codes, const uint8_t *__restrict__ exps,
                                                            size_t n_groups, bf16 *__restrict__ w) {
    const size_t gi = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gi >= n_groups) return;
    const uint4 c = *reinterpret_cast<const uint4 *>(codes + gi * 16);
    const float s = __uint_as_float((uint32_t)exps[gi] << 23);      // 2^e
    const uint32_t wv[4] = {c.x, c.y, c.z, c.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        uint32_t o[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float a = (float)((int)((wv[i] >> (8 * j)) & 15u) - 8) * s, b = (float)((int)((wv[i] >> (8 * j + 4)) & 15u) - 8) * s;
            const __nv_bfloat162 hb = __floats2bfloat162_rn(a, b);   // exact: <= 4 significant bits
            o[j] = *reinterpret_cast<const uint32_t *>(&hb);
        }
        reinterpret_cast<uint4 *>(w + gi * 32)[i] = make_uint4(o[0], o[1], o[2], o[3]);
    }
}

// ---- host side ------------------------------------------------------------------------------------------------------
// whole groups of 32; rows longer than 2048 are cut into four quarters of whole 256-element superblock pairs
bool sgemv_q4_shape_supported(int K) { return K > 0 && K % 32 == 0 && (K <= 2048 || (K % 1024 == 0 && K <= 8192)); }

static size_t q4_smem_bytes(int norm_k) {   // norm_k: input length when the kernel normalises it into shared-memory planes, else 0
    return (size_t)kQ4Stages * kQ4StageBytes + ((sizeof(Q4Shared) + 15) & ~(size_t)15) + (size_t)norm_k * 4 + 128;
}

cudaError_t sgemv_q4_prepare() {
    return cudaFuncSetAttribute(sgemv_q4_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)q4_smem_bytes(2048));
}

cudaError_t launch_sgemv_q4(const LaunchCtx &c, const SgemvParams &p) {
    if (!sgemv_q4_shape_supported(p.K) || !p.q0 || !p.e0) return cudaErrorInvalidValue;
    const int rps = q4_rows_per_stage(p.K, p.mode);
    if ((size_t)(p.mode == SGEMV_GATEUP ? 16 : rps) * (p.K / 2) > (size_t)kQ4CodeBytes) return cudaErrorInvalidValue;
    const int n_stages = (p.n_rows + rps - 1) / rps;
    int grid = c.n_sms < n_stages ? c.n_sms : n_stages;
    if (p.max_ctas > 0 && p.max_ctas < grid) grid = p.max_ctas;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(kQ4Threads);
    if (p.xin_mode == SGEMV_XIN_NORM && p.K > 2048) return cudaErrorInvalidValue;
    cfg.dynamicSmemBytes = q4_smem_bytes(p.xin_mode == SGEMV_XIN_NORM ? p.K : 0);
    cfg.stream = c.stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = c.pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, sgemv_q4_kernel, p);
}

cudaError_t launch_q4_quantize(cudaStream_t stream, const bf16 *w, size_t n_rows, int K, uint8_t *codes, uint8_t *exps) {
    const size_t n_groups = n_rows * (size_t)(K / 32);
    q4_quantize_kernel<<<(unsigned)((n_groups + 255) / 256), 256, 0, stream>>>(w, n_groups, codes, exps);
    return cudaGetLastError();
}
cudaError_t launch_q4_dequantize(cudaStream_t stream, const uint8_t *codes, const uint8_t *exps, size_t n_rows, int K, bf16 *w) {
    const size_t n_groups = n_rows * (size_t)(K / 32);
    q4_dequantize_kernel<<<(unsigned)((n_groups + 255) / 256), 256, 0, stream>>>(codes, exps, n_groups, w);
    return cudaGetLastError();
}

}  // namespace hq
