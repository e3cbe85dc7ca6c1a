// hq_prefill.cu — row-batched kernels around the tcgen05 GEMMs: envelope prefill (SURVEY.md §8(a)
// P2-P4) and batched decode (B1-B2).  "Rows" are tokens m = b * Tc + t of the current pass.
//   embed_rows      x[m] = float(E[tok[m]])                                          (A1 for many rows)
//   rmsnorm_rows    hn[m] = hi/lo bf16 of x[m] * rsqrt(mean(x[m]^2) + eps) * g       (tensor-core operand)
//   rope_append     qkv fp32 -> RoPE(q) as fp16 (+ fp32 copy for decode), RoPE(k), v -> fp16 KV cache   (P4)
//   flash_prefill   causal GQA flash attention, mma.sync m16n8k16 fp16, fp32 online softmax           (P2)
//   attn_combine    merge split-KV partials of the decode attention -> o hi/lo bf16                         (B2)
//   argmax_rows     greedy token per sequence from fp32 logits + device-resident step state           (A9/B1)
#include "hq_common.cuh"
#include "hq_internal.h"

namespace hq {

// =====================================================================================================
__global__ void __launch_bounds__(256) embed_rows_kernel(const bf16 *__restrict__ emb, const int *tok,
                                                         float *__restrict__ x, int hidden) {
    pdl_launch_dependents();
    pdl_wait();
    const int m = blockIdx.x;
    const bf16 *row = emb + (size_t)ld_act(tok + m) * hidden;
    for (int c = threadIdx.x; c < (hidden >> 3); c += blockDim.x) {
        const uint4 w = ld_weight16(row + c * 8);
        float4 *dst = reinterpret_cast<float4 *>(x + (size_t)m * hidden + c * 8);
        dst[0] = make_float4(bf16lo(w.x), bf16hi(w.x), bf16lo(w.y), bf16hi(w.y));
        dst[1] = make_float4(bf16lo(w.z), bf16hi(w.z), bf16lo(w.w), bf16hi(w.w));
    }
}

// one CTA per row; x row stays in L1/L2 between the two passes
// delta (n_parts > 0): the deferred output of the previous residual projection as n_parts split-K partial buffers,
// part_stride floats apart: x += delta[0] + delta[1] + ... first, in that order, written back.  Keeps split-K of those
// projections bit-reproducible without atomics: every split stores its own partial, the consumer adds them in order.
__global__ void __launch_bounds__(256) rmsnorm_rows_kernel(float *x, const float *delta, int n_parts, size_t part_stride, const bf16 *__restrict__ gain,
                                                           act_t *__restrict__ out, size_t lo_offset, int hidden,
                                                           float eps, const int *row_index, int x_stride_rows, float *zero, int zero_per_row) {
    pdl_launch_dependents();
    pdl_wait();
    __shared__ float red[8];
    const int m = blockIdx.x;
    // zero (optional): row m of a buffer the NEXT kernel accumulates into with atomics (the Q|K|V projections of a batched
    // decode step).  Cleared here instead of by a memset node, which would cut the programmatic launch edge to that kernel.
    if (zero)
        for (int c = threadIdx.x; c < (zero_per_row >> 2); c += blockDim.x)
            reinterpret_cast<float4 *>(zero + (size_t)m * zero_per_row)[c] = make_float4(0.f, 0.f, 0.f, 0.f);
    // row_index (optional) gathers rows (e.g. last position of every sequence)
    const size_t src = row_index ? (size_t)row_index[m] : (size_t)m;
    float *xr = x + src * x_stride_rows;
    const float *dr = (delta && n_parts > 0) ? delta + src * x_stride_rows : nullptr;
    // Every load of a thread is issued before the first value is used (4 float4 of x and up to 4 partials of each: 20 L2
    // round trips in flight instead of one after the other -- the row kernels are latency, not bandwidth), and the summed
    // row stays in registers for the second pass.  Rows longer than 4 x 1024 floats take the plain loop below.
    constexpr int kChunks = 4, kParts = 4;
    float ss = 0.f;
    if (hidden <= kChunks * 1024 && blockDim.x == 256 && n_parts <= kParts) {
        const int n4 = hidden >> 2;
        float4 v[kChunks], dv[kChunks][kParts];
#pragma unroll
        for (int k = 0; k < kChunks; ++k) {
            const int c = threadIdx.x + k * 256;
            v[k] = c < n4 ? ld_act4(xr + c * 4) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
            for (int sp = 0; sp < kParts; ++sp)
                dv[k][sp] = (dr && sp < n_parts && c < n4) ? ld_act4(dr + (size_t)sp * part_stride + c * 4) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int k = 0; k < kChunks; ++k) {
            const int c = threadIdx.x + k * 256;
#pragma unroll
            for (int sp = 0; sp < kParts; ++sp)
                if (dr && sp < n_parts) { v[k].x += dv[k][sp].x; v[k].y += dv[k][sp].y; v[k].z += dv[k][sp].z; v[k].w += dv[k][sp].w; }   // fixed order
            if (dr && c < n4) *reinterpret_cast<float4 *>(xr + c * 4) = v[k];
            ss += v[k].x * v[k].x + v[k].y * v[k].y + v[k].z * v[k].z + v[k].w * v[k].w;
        }
        ss = warp_sum(ss);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = ss;
        __syncthreads();
        float tot = 0.f;
#pragma unroll
        for (int w = 0; w < 8; ++w) tot += red[w];
        const float inv = 1.0f / sqrtf(tot / (float)hidden + eps);
#pragma unroll
        for (int k = 0; k < kChunks; ++k) {
            const int c = threadIdx.x + k * 256;
            if (c < n4) {
                const uint2 g = *reinterpret_cast<const uint2 *>(gain + c * 4);
                uint2 oh, ol;
                split_bf16x2(v[k].x * inv * bf16lo(g.x), v[k].y * inv * bf16hi(g.x), oh.x, ol.x);
                split_bf16x2(v[k].z * inv * bf16lo(g.y), v[k].w * inv * bf16hi(g.y), oh.y, ol.y);
                *reinterpret_cast<uint2 *>(out + (size_t)m * hidden + c * 4) = oh;
                *reinterpret_cast<uint2 *>(out + lo_offset + (size_t)m * hidden + c * 4) = ol;
            }
        }
        return;
    }
    for (int c = threadIdx.x; c < (hidden >> 2); c += blockDim.x) {
        float4 v = ld_act4(xr + c * 4);
        if (dr) {
            for (int sp = 0; sp < n_parts; ++sp) {
                const float4 dv = ld_act4(dr + (size_t)sp * part_stride + c * 4);
                v.x += dv.x; v.y += dv.y; v.z += dv.z; v.w += dv.w;
            }
            *reinterpret_cast<float4 *>(xr + c * 4) = v;
        }
        ss += v.x * v.x + v.y * v.y + v.z * v.z + v.w * v.w;
    }
    ss = warp_sum(ss);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = ss;
    __syncthreads();
    float tot = 0.f;
#pragma unroll
    for (int w = 0; w < 8; ++w) tot += red[w];
    const float inv = 1.0f / sqrtf(tot / (float)hidden + eps);
    for (int c = threadIdx.x; c < (hidden >> 2); c += blockDim.x) {
        const float4 v = dr ? *reinterpret_cast<const float4 *>(xr + c * 4) : ld_act4(xr + c * 4);   // own store above
        const uint2 g = *reinterpret_cast<const uint2 *>(gain + c * 4);
        uint2 oh, ol;
        split_bf16x2(v.x * inv * bf16lo(g.x), v.y * inv * bf16hi(g.x), oh.x, ol.x);
        split_bf16x2(v.z * inv * bf16lo(g.y), v.w * inv * bf16hi(g.y), oh.y, ol.y);
        *reinterpret_cast<uint2 *>(out + (size_t)m * hidden + c * 4) = oh;
        *reinterpret_cast<uint2 *>(out + lo_offset + (size_t)m * hidden + c * 4) = ol;
    }
}

// qkv fp32 [M][(H + 2 Hkv) * 64] -> q (fp16 [M][H*64], optional fp32 copy), K/V cache rows.
// grid (M), block 256: thread handles (head-any hh, i) pairs in a loop.
__global__ void __launch_bounds__(256) rope_append_kernel(const float *qkv, int n_parts, size_t part_stride, __half *q16, float *q32, kv_t *kc, kv_t *vc,
                                                          const float2 *__restrict__ rope, const int *pos_ptr, int Tc,
                                                          int n_heads, int n_kv_heads, int max_seq) {
    pdl_launch_dependents();
    pdl_wait();
    const int m = blockIdx.x;
    const int b = m / Tc, t = m % Tc;
    const int pos = ld_act(pos_ptr) + t;
    const int nh = n_heads + 2 * n_kv_heads;
    const float *src = qkv + (size_t)m * nh * kHeadDim;
    // three (head, pair) units per thread and round, every load of the round (and of every split-K partial) issued before
    // the first use: the kernel is a chain of L2 round trips otherwise (6 units x 2 partials one after the other)
    constexpr int kU = 3;
    const int lim = nh * 32;
    for (int idx0 = threadIdx.x; idx0 < lim; idx0 += kU * blockDim.x) {
        float a[kU], c[kU];
#pragma unroll
        for (int u = 0; u < kU; ++u) {
            const int idx = idx0 + u * (int)blockDim.x, hh = idx >> 5, i = idx & 31;
            const bool ok = idx < lim;
            a[u] = ok ? ld_act(src + hh * kHeadDim + i) : 0.f;
            c[u] = ok ? ld_act(src + hh * kHeadDim + i + 32) : 0.f;
        }
        for (int sp = 1; sp < n_parts; sp += 2) {   // split-K partials of the projection, fixed order, two at a time
            float pa[2][kU], pc[2][kU];
#pragma unroll
            for (int s2 = 0; s2 < 2; ++s2)
#pragma unroll
                for (int u = 0; u < kU; ++u) {
                    const int idx = idx0 + u * (int)blockDim.x, hh = idx >> 5, i = idx & 31;
                    const bool ok = idx < lim && sp + s2 < n_parts;
                    pa[s2][u] = ok ? ld_act(src + (size_t)(sp + s2) * part_stride + hh * kHeadDim + i) : 0.f;
                    pc[s2][u] = ok ? ld_act(src + (size_t)(sp + s2) * part_stride + hh * kHeadDim + i + 32) : 0.f;
                }
#pragma unroll
            for (int s2 = 0; s2 < 2; ++s2)
                if (sp + s2 < n_parts) {
#pragma unroll
                    for (int u = 0; u < kU; ++u) { a[u] += pa[s2][u]; c[u] += pc[s2][u]; }
                }
        }
#pragma unroll
        for (int u = 0; u < kU; ++u) {
            const int idx = idx0 + u * (int)blockDim.x, hh = idx >> 5, i = idx & 31;
            if (idx >= lim) continue;
            if (hh < n_heads + n_kv_heads) {
                const float2 cs = rope[(size_t)pos * 32 + i];
                const float ra = a[u] * cs.x - c[u] * cs.y, rc = c[u] * cs.x + a[u] * cs.y;
                if (hh < n_heads) {
                    const size_t o = ((size_t)m * n_heads + hh) * kHeadDim + i;
                    q16[o] = __float2half_rn(ra);
                    q16[o + 32] = __float2half_rn(rc);
                    if (q32) { q32[o] = ra; q32[o + 32] = rc; }
                } else {
                    kv_t *dst = kc + (((size_t)b * n_kv_heads + (hh - n_heads)) * max_seq + pos) * kHeadDim;
                    dst[i] = __float2half_rn(ra);
                    dst[i + 32] = __float2half_rn(rc);
                }
            } else {
                kv_t *dst = vc + (((size_t)b * n_kv_heads + (hh - n_heads - n_kv_heads)) * max_seq + pos) * kHeadDim;
                dst[i] = __float2half_rn(a[u]);
                dst[i + 32] = __float2half_rn(c[u]);
            }
        }
    }
}

// =====================================================================================================
// P2: causal flash attention for a pass of Tc query positions per sequence starting at position p0.
// grid (ceil(Tc/64), H, B), 128 threads: warp w owns query rows 16w..16w+15 of the 64-row tile.
// =====================================================================================================
constexpr int kFaTile = 64;

__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gmem_src, bool valid) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    const int sz = valid ? 16 : 0;   // src-size 0 -> zero fill
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(gmem_src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ void ldmatrix_x4(uint32_t (&r)[4], const void *smem) {
    const uint32_t a = (uint32_t)__cvta_generic_to_shared(smem);
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(a));
}
__device__ __forceinline__ void ldmatrix_x4_trans(uint32_t (&r)[4], const void *smem) {
    const uint32_t a = (uint32_t)__cvta_generic_to_shared(smem);
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(a));
}
__device__ __forceinline__ void mma_f16(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
// element (row, col) of a [64][64] fp16 tile with 16-byte chunks XOR-swizzled by the row
__device__ __forceinline__ __half *tile_ptr(__half *tile, int row, int col) {
    return tile + row * 64 + ((((col >> 3) ^ (row & 7)) << 3) | (col & 7));
}
__device__ __forceinline__ uint32_t pack_half2(float a, float b) {
    __half2 h = __floats2half2_rn(a, b);
    return *reinterpret_cast<uint32_t *>(&h);
}

__global__ void __launch_bounds__(128) flash_prefill_kernel(const __half *q16, const kv_t *kc, const kv_t *vc,
                                                            act_t *out, size_t lo_offset, const int *pos_ptr, int Tc,
                                                            int n_heads,
                                                            int n_kv_heads, int max_seq) {
    __shared__ __align__(128) __half Qs[kFaTile * 64];
    __shared__ __align__(128) __half Ks[2][kFaTile * 64];
    __shared__ __align__(128) __half Vs[2][kFaTile * 64];
    pdl_launch_dependents();
    pdl_wait();

    const int qt = blockIdx.x, h = blockIdx.y, b = blockIdx.z;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 2, tig = lane & 3;
    const int p0 = ld_act(pos_ptr);
    const int kvh = h / (n_heads / n_kv_heads);
    const int q_lo = qt * kFaTile;                        // first local query of the tile
    const int q_hi = min(Tc, q_lo + kFaTile);             // one past the last valid local query
    const int n_keys = p0 + q_hi;                         // keys 0 .. n_keys-1 can be visible
    const int n_kt = (n_keys + kFaTile - 1) / kFaTile;
    const kv_t *kg = kc + ((size_t)b * n_kv_heads + kvh) * max_seq * kHeadDim;
    const kv_t *vg = vc + ((size_t)b * n_kv_heads + kvh) * max_seq * kHeadDim;

    auto load_kv = [&](int buf, int kt) {
        for (int c = threadIdx.x; c < kFaTile * 8; c += 128) {
            const int r = c >> 3, ch = c & 7;
            const int key = kt * kFaTile + r;
            const bool ok = key < n_keys;
            const size_t off = (size_t)(ok ? key : 0) * kHeadDim + ch * 8;
            cp_async16(tile_ptr(Ks[buf], r, ch * 8), kg + off, ok);
            cp_async16(tile_ptr(Vs[buf], r, ch * 8), vg + off, ok);
        }
    };
    // Q tile
    for (int c = threadIdx.x; c < kFaTile * 8; c += 128) {
        const int r = c >> 3, ch = c & 7;
        const bool ok = q_lo + r < Tc;
        const size_t m = (size_t)b * Tc + (ok ? q_lo + r : 0);
        cp_async16(tile_ptr(Qs, r, ch * 8), q16 + (m * n_heads + h) * kHeadDim + ch * 8, ok);
    }
    load_kv(0, 0);
    cp_async_commit();
    cp_async_wait<0>();
    __syncthreads();

    // Q fragments: 4 k-steps (dims 16kk..16kk+15) for rows 16*warp .. +15
    uint32_t qf[4][4];
#pragma unroll
    for (int kk = 0; kk < 4; ++kk)
        ldmatrix_x4(qf[kk], tile_ptr(Qs, 16 * warp + (lane & 15), kk * 16 + (lane >> 4) * 8));

    float o[8][4];
#pragma unroll
    for (int j = 0; j < 8; ++j) { o[j][0] = o[j][1] = o[j][2] = o[j][3] = 0.f; }
    float m_run[2] = {-INFINITY, -INFINITY}, l_run[2] = {0.f, 0.f};
    const float sl2 = 0.125f * 1.4426950408889634f;       // softmax scale * log2(e)
    const int qpos0 = p0 + q_lo + 16 * warp + g;           // global position of fragment row g (row g+8: +8)

    for (int kt = 0; kt < n_kt; ++kt) {
        const int buf = kt & 1;
        if (kt + 1 < n_kt) load_kv(buf ^ 1, kt + 1);
        cp_async_commit();
        // S = Q K^T for 64 keys: 8 n-tiles of 8 keys
        float s[8][4];
#pragma unroll
        for (int j = 0; j < 8; ++j) { s[j][0] = s[j][1] = s[j][2] = s[j][3] = 0.f; }
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
#pragma unroll
            for (int jp = 0; jp < 4; ++jp) {   // pairs of n-tiles
                uint32_t kf[4];
                const int mi = lane >> 3;
                ldmatrix_x4(kf, tile_ptr(Ks[buf], jp * 16 + (mi >> 1) * 8 + (lane & 7), kk * 16 + (mi & 1) * 8));
                mma_f16(s[2 * jp], qf[kk], kf[0], kf[1]);
                mma_f16(s[2 * jp + 1], qf[kk], kf[2], kf[3]);
            }
        }
        // causal mask + online softmax (rows g and g+8 of this warp's 16)
        const int key0 = kt * kFaTile;
        float mx[2] = {m_run[0], m_run[1]};
#pragma unroll
        for (int j = 0; j < 8; ++j) {
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int key = key0 + j * 8 + tig * 2 + (e & 1);
                const int qp = qpos0 + (e >> 1) * 8;
                if (key > qp) s[j][e] = -INFINITY;
                mx[e >> 1] = fmaxf(mx[e >> 1], s[j][e]);
            }
        }
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            mx[r] = fmaxf(mx[r], __shfl_xor_sync(0xffffffffu, mx[r], 1));
            mx[r] = fmaxf(mx[r], __shfl_xor_sync(0xffffffffu, mx[r], 2));
        }
        float corr[2], rs[2] = {0.f, 0.f};
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            // a fully masked row (padding rows beyond Tc) keeps m = -inf: use 0 to avoid inf - inf
            const float mref = (mx[r] == -INFINITY) ? 0.f : mx[r];
            corr[r] = exp2f((m_run[r] - mref) * sl2);
            m_run[r] = mx[r];
            mx[r] = mref;
        }
        uint32_t pf[4][4];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const float p0v = exp2f((s[j][0] - mx[0]) * sl2), p1v = exp2f((s[j][1] - mx[0]) * sl2);
            const float p2v = exp2f((s[j][2] - mx[1]) * sl2), p3v = exp2f((s[j][3] - mx[1]) * sl2);
            rs[0] += p0v + p1v;
            rs[1] += p2v + p3v;
            pf[j >> 1][(j & 1) * 2 + 0] = pack_half2(p0v, p1v);
            pf[j >> 1][(j & 1) * 2 + 1] = pack_half2(p2v, p3v);
        }
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            rs[r] += __shfl_xor_sync(0xffffffffu, rs[r], 1);
            rs[r] += __shfl_xor_sync(0xffffffffu, rs[r], 2);
            l_run[r] = l_run[r] * corr[r] + rs[r];
        }
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            o[j][0] *= corr[0]; o[j][1] *= corr[0]; o[j][2] *= corr[1]; o[j][3] *= corr[1];
        }
        // O += P V : k-steps over keys (16 each), n-tiles over dims
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
#pragma unroll
            for (int jp = 0; jp < 4; ++jp) {
                uint32_t vf[4];
                const int mi = lane >> 3;
                ldmatrix_x4_trans(vf, tile_ptr(Vs[buf], kk * 16 + (mi & 1) * 8 + (lane & 7), jp * 16 + (mi >> 1) * 8));
                mma_f16(o[2 * jp], pf[kk], vf[0], vf[1]);
                mma_f16(o[2 * jp + 1], pf[kk], vf[2], vf[3]);
            }
        }
        cp_async_wait<0>();
        __syncthreads();
    }

    // normalise and store o as hi/lo bf16 planes [m][H*64]
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        const int ql = q_lo + 16 * warp + g + r * 8;
        if (ql < Tc) {
            const float inv = 1.0f / l_run[r];
            act_t *dst = out + (((size_t)b * Tc + ql) * n_heads + h) * kHeadDim;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                uint32_t vh, vl;
                split_bf16x2(o[j][2 * r] * inv, o[j][2 * r + 1] * inv, vh, vl);
                *reinterpret_cast<uint32_t *>(dst + j * 8 + tig * 2) = vh;
                *reinterpret_cast<uint32_t *>(dst + lo_offset + j * 8 + tig * 2) = vl;
            }
        }
    }
}

// =====================================================================================================
// B2: merge split-KV partials -> o bf16 [B][H*64].  grid (B), block = H*8 threads... generic loop.
// =====================================================================================================
__global__ void __launch_bounds__(256) attn_combine_kernel(const float *part_o, const float2 *part_ml, act_t *out,
                                                           size_t lo_offset, const int *pos_ptr, int n_heads) {
    pdl_launch_dependents();
    pdl_wait();
    const int b = blockIdx.x;
    const int n_ctx = ld_act(pos_ptr) + 1;
    const int ns = attn_num_splits(n_ctx);
    for (int chunk = threadIdx.x; chunk < n_heads * 8; chunk += blockDim.x) {
        const int head = chunk >> 3, d0 = (chunk & 7) * 8;
        const size_t hb = (size_t)b * n_heads + head;
        const float2 *ml = part_ml + hb * kMaxSplits;
        // every (m, l) pair in one round trip, then the partial outputs four splits at a time (this kernel is a chain of L2
        // round trips: 8 CTAs, a few hundred bytes each)
        float2 mls[kMaxSplits];
#pragma unroll
        for (int s = 0; s < kMaxSplits; ++s) mls[s] = s < ns ? __ldcg(&ml[s]) : make_float2(-INFINITY, 0.f);
        float M = -INFINITY;
#pragma unroll
        for (int s = 0; s < kMaxSplits; ++s) M = fmaxf(M, mls[s].x);
        float acc[8] = {0, 0, 0, 0, 0, 0, 0, 0}, denom = 0.f;
#pragma unroll
        for (int s4 = 0; s4 < kMaxSplits; s4 += 4) {
            if (s4 < ns) {   // uniform over the CTA
                float4 a[4], c[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const float *po = part_o + (hb * kMaxSplits + s4 + u) * kHeadDim + d0;
                    const bool ok = s4 + u < ns;
                    a[u] = ok ? ld_act4(po) : make_float4(0.f, 0.f, 0.f, 0.f);
                    c[u] = ok ? ld_act4(po + 4) : make_float4(0.f, 0.f, 0.f, 0.f);
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    if (s4 + u < ns) {   // same order and arithmetic as one split after the other
                        const float w = __expf(mls[s4 + u].x - M);
                        denom += w * mls[s4 + u].y;
                        acc[0] += w * a[u].x; acc[1] += w * a[u].y; acc[2] += w * a[u].z; acc[3] += w * a[u].w;
                        acc[4] += w * c[u].x; acc[5] += w * c[u].y; acc[6] += w * c[u].z; acc[7] += w * c[u].w;
                    }
                }
            }
        }
        const float inv = 1.0f / denom;
        act_t *dst = out + hb * kHeadDim + d0;
#pragma unroll
        for (int i = 0; i < 8; i += 2) {
            uint32_t vh, vl;
            split_bf16x2(acc[i] * inv, acc[i + 1] * inv, vh, vl);
            *reinterpret_cast<uint32_t *>(dst + i) = vh;
            *reinterpret_cast<uint32_t *>(dst + lo_offset + i) = vl;
        }
    }
}

// =====================================================================================================
// greedy argmax per sequence over fp32 logits [B][V] (lowest index on ties) + step bookkeeping.
// grid (slices, B), block 256: per-slice winner -> packed 64-bit atomicMax per row; the last CTA of the launch writes
// the tokens, clears the winners and advances the shared position.
// =====================================================================================================
__global__ void __launch_bounds__(256) argmax_rows_kernel(const float *logits, int vocab, int batch, int *cur_tok,
                                                          int *tok_hist, int *pos, int pos_inc, unsigned int *counter,
                                                          unsigned long long *best_rows) {
    pdl_launch_dependents();
    pdl_wait();
    __shared__ unsigned long long red[8];
    __shared__ int last;
    const int b = blockIdx.y;
    const float *row = logits + (size_t)b * vocab;
    // slice of the row: float4 loads where the row start is 16-byte aligned, scalar otherwise
    const int per = ((vocab + (int)gridDim.x - 1) / (int)gridDim.x + 3) & ~3;
    const int i0 = blockIdx.x * per, i1 = min(vocab, i0 + per);
    unsigned long long best = 0ull;
    if ((vocab & 3) == 0) {
        for (int i = i0 + 4 * threadIdx.x; i + 3 < i1; i += 4 * blockDim.x) {
            const float4 v = ld_act4(row + i);
            unsigned long long k0 = pack_argmax(v.x, i), k1 = pack_argmax(v.y, i + 1), k2 = pack_argmax(v.z, i + 2), k3 = pack_argmax(v.w, i + 3);
            k0 = k0 > k1 ? k0 : k1;
            k2 = k2 > k3 ? k2 : k3;
            k0 = k0 > k2 ? k0 : k2;
            best = best > k0 ? best : k0;
        }
    } else {
        for (int i = i0 + threadIdx.x; i < i1; i += blockDim.x) {
            const unsigned long long k = pack_argmax(ld_act(row + i), i);
            best = best > k ? best : k;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(0xffffffffu, best, o);
        best = best > other ? best : other;
    }
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = best;
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int w = 1; w < 8; ++w) best = best > red[w] ? best : red[w];
        if (best) atomicMax(best_rows + b, best);   // packed (ordered logit, ~index): lowest index wins ties
        __threadfence();
        const unsigned int ticket = atomicAdd(counter, 1u);
        last = ticket == gridDim.x * gridDim.y - 1u;
    }
    __syncthreads();
    if (last) {   // the last CTA of the launch: every row's winner is final
        __threadfence();
        const int p = ld_act(pos);
        for (int r = threadIdx.x; r < batch; r += blockDim.x) {
            const int tok = unpack_argmax_idx(__ldcg(best_rows + r));
            cur_tok[r] = tok;
            tok_hist[(size_t)(p + pos_inc) * batch + r] = tok;
            best_rows[r] = 0ull;
        }
        if (threadIdx.x == 0) {
            *pos = p + pos_inc;
            *counter = 0u;
        }
    }
}

// =====================================================================================================
// Verbatim-relay verification: row j of logits [n_rows][vocab] is the LM head at the position that
// predicts answer token j (row n_answer = n_rows - 1: the token after the whole answer).  grid (slices, n_rows): per-slice
// winner -> packed atomicMax per row; the last CTA counts the leading rows whose greedy token equals the answer token,
// publishes the count, and leaves the step state as if envelope + accepted answer tokens had been fed: position,
// and as "last emitted token" the model's own choice at the first mismatch (streaming decode continues from there).
// =====================================================================================================
__global__ void __launch_bounds__(256) verify_rows_kernel(const float *logits, int vocab, int n_rows, const int *answer,
                                                          int n_envelope, int *cur_tok, int *tok_hist, int *pos,
                                                          unsigned int *counter, unsigned long long *best_rows,
                                                          int *n_accepted) {
    pdl_launch_dependents();
    pdl_wait();
    __shared__ unsigned long long red[8];
    __shared__ int last;
    const int b = blockIdx.y;
    const float *row = logits + (size_t)b * vocab;
    const int per = ((vocab + (int)gridDim.x - 1) / (int)gridDim.x + 3) & ~3;
    const int i0 = blockIdx.x * per, i1 = min(vocab, i0 + per);
    unsigned long long best = 0ull;
    for (int i = i0 + threadIdx.x; i < i1; i += blockDim.x) {
        const unsigned long long k = pack_argmax(ld_act(row + i), i);
        best = best > k ? best : k;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(0xffffffffu, best, o);
        best = best > other ? best : other;
    }
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = best;
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int w = 1; w < 8; ++w) best = best > red[w] ? best : red[w];
        if (best) atomicMax(best_rows + b, best);   // packed (ordered logit, ~index): lowest index wins ties
        __threadfence();
        const unsigned int ticket = atomicAdd(counter, 1u);
        last = ticket == gridDim.x * gridDim.y - 1u;
    }
    __syncthreads();
    if (last && threadIdx.x == 0) {   // every row's winner is final
        __threadfence();
        int j = 0;
        while (j < n_rows - 1 && unpack_argmax_idx(__ldcg(best_rows + j)) == ld_act(answer + j)) ++j;
        const int tok = unpack_argmax_idx(__ldcg(best_rows + j));
        const int p = ld_act(pos) + n_envelope + j;
        *n_accepted = j;
        *cur_tok = tok;
        tok_hist[p] = tok;
        *pos = p;
        for (int r = 0; r < n_rows; ++r) best_rows[r] = 0ull;
        *counter = 0u;
    }
}

// ---- launchers ------------------------------------------------------------------------------------------
template <typename... KArgs, typename... Args>
static cudaError_t launch_k(const LaunchCtx &c, void (*kernel)(KArgs...), dim3 grid, dim3 block, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.stream = c.stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = c.pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

cudaError_t launch_embed_rows(const LaunchCtx &c, const bf16 *emb, const int *tok, float *x, int hidden, int rows) {
    return launch_k(c, embed_rows_kernel, dim3(rows), dim3(256), emb, tok, x, hidden);
}
cudaError_t launch_rmsnorm_rows(const LaunchCtx &c, float *x, const float *delta, int n_parts, size_t part_stride, const bf16 *gain,
                                act_t *out, size_t lo_offset, int hidden, float eps, int rows, const int *row_index, int x_stride_rows,
                                float *zero, int zero_per_row) {
    if (zero && zero_per_row % 4 != 0) return cudaErrorInvalidValue;
    return launch_k(c, rmsnorm_rows_kernel, dim3(rows), dim3(256), x, delta, n_parts, part_stride, gain, out, lo_offset, hidden, eps,
                    row_index, x_stride_rows, zero, zero_per_row);
}
// x += delta, delta = 0 (parity capture needs the residual itself after every layer)
__global__ void __launch_bounds__(256) add_delta_rows_kernel(float *x, const float *delta, int n_parts, size_t part_stride, size_t n4) {
    pdl_launch_dependents();
    pdl_wait();
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
        float4 v = ld_act4(x + i * 4);
        for (int sp = 0; sp < n_parts; ++sp) {   // the split-K partials in fixed order
            const float4 dv = ld_act4(delta + (size_t)sp * part_stride + i * 4);
            v.x += dv.x; v.y += dv.y; v.z += dv.z; v.w += dv.w;
        }
        *reinterpret_cast<float4 *>(x + i * 4) = v;
    }
}
cudaError_t launch_add_delta_rows(const LaunchCtx &c, float *x, const float *delta, int n_parts, size_t part_stride, size_t n) {
    return launch_k(c, add_delta_rows_kernel, dim3(296), dim3(256), x, delta, n_parts, part_stride, n / 4);
}
cudaError_t launch_rope_append(const LaunchCtx &c, const float *qkv, int n_parts, size_t part_stride, __half *q16, float *q32, kv_t *kc,
                               kv_t *vc, const float2 *rope, const int *pos, int rows, int Tc, int n_heads, int n_kv_heads,
                               int max_seq) {
    return launch_k(c, rope_append_kernel, dim3(rows), dim3(256), qkv, n_parts, part_stride, q16, q32, kc, vc, rope, pos, Tc, n_heads,
                    n_kv_heads, max_seq);
}
cudaError_t launch_flash_prefill(const LaunchCtx &c, const __half *q16, const kv_t *kc, const kv_t *vc, act_t *out,
                                 size_t lo_offset, const int *pos, int batch, int Tc, int n_heads, int n_kv_heads,
                                 int max_seq) {
    return launch_k(c, flash_prefill_kernel, dim3((Tc + kFaTile - 1) / kFaTile, n_heads, batch), dim3(128), q16, kc, vc,
                    out, lo_offset, pos, Tc, n_heads, n_kv_heads, max_seq);
}
cudaError_t launch_attn_combine(const LaunchCtx &c, const float *part_o, const float2 *part_ml, act_t *out,
                                size_t lo_offset, const int *pos, int batch, int n_heads) {
    return launch_k(c, attn_combine_kernel, dim3(batch), dim3(256), part_o, part_ml, out, lo_offset, pos, n_heads);
}
cudaError_t launch_verify_rows(const LaunchCtx &c, const float *logits, int vocab, int n_rows, const int *answer, int n_envelope,
                               int *cur_tok, int *tok_hist, int *pos, unsigned int *counter, unsigned long long *best_rows,
                               int *n_accepted) {
    const int slices = vocab >= 32768 ? 16 : (vocab >= 4096 ? 4 : 1);
    return launch_k(c, verify_rows_kernel, dim3(slices, n_rows), dim3(256), logits, vocab, n_rows, answer, n_envelope, cur_tok,
                    tok_hist, pos, counter, best_rows, n_accepted);
}
cudaError_t launch_argmax_rows(const LaunchCtx &c, const float *logits, int vocab, int batch, int *cur_tok,
                               int *tok_hist, int *pos, int pos_inc, unsigned int *counter, unsigned long long *best_rows) {
    const int slices = vocab >= 32768 ? 32 : (vocab >= 4096 ? 4 : 1);
    return launch_k(c, argmax_rows_kernel, dim3(slices, batch), dim3(256), logits, vocab, batch, cur_tok, tok_hist, pos,
                    pos_inc, counter, best_rows);
}

}  // namespace hq
