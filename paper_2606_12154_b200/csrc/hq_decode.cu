// hq_decode.cu — batch-1 streaming decode kernels.
//
// One token per step is a chain of HBM-bound matrix-vector products (2.47 GB of bf16 weights per
// token), so every kernel here is built around one idea: keep 16-byte weight loads in flight.
//   * gemv_kernel (kernel-per-row path: QKV and O projections; the big streams are hq_stream.cu): a CTA of 256
//     threads owns a contiguous range of "units" (2 output rows each).  Thread t owns the same 8-element k-slices of
//     every row, so the (normalised) input vector lives in registers, a row is read by 512-byte coalesced warp
//     loads, and 2U*CH independent 16-byte loads per thread are double buffered.  Fused in: RMSNorm prologue (A2),
//     split-KV merge prologue (A5 combine), RoPE + KV append (A4), residual add (A6).
//   * Weight loads for the first batch are issued BEFORE griddepcontrol.wait (weights are
//     immutable), so under programmatic dependent launch they overlap the previous kernel's tail.
//   * attn_decode_kernel: GQA split-KV flash-decode; K/V tiles staged in shared memory with one
//     bulk async copy (TMA, cp.async.bulk) per tile, shared by the G query heads of the group.
#include "hq_common.cuh"
#include "hq_internal.h"
#include "hq_attn_tile.cuh"

namespace hq {

// =====================================================================================================
// A1: embedding gather  x[b] = float(E[tok[b]])
// =====================================================================================================
__global__ void __launch_bounds__(256) embed_kernel(const bf16 *__restrict__ emb, const int *tok,
                                                    float *__restrict__ x, int hidden) {
    pdl_launch_dependents();
    pdl_wait();
    const int b = blockIdx.x;
    const int t = ld_act(tok + b);
    const bf16 *row = emb + (size_t)t * hidden;
    for (int c = threadIdx.x; c < (hidden >> 3); c += blockDim.x) {
        uint4 w = ld_weight16(row + c * 8);
        float4 lo = make_float4(bf16lo(w.x), bf16hi(w.x), bf16lo(w.y), bf16hi(w.y));
        float4 hi = make_float4(bf16lo(w.z), bf16hi(w.z), bf16lo(w.w), bf16hi(w.w));
        float4 *dst = reinterpret_cast<float4 *>(x + (size_t)b * hidden + c * 8);
        dst[0] = lo;
        dst[1] = hi;
    }
}

__global__ void advance_kernel(int *pos, int inc) {
    pdl_launch_dependents();
    pdl_wait();
    if (threadIdx.x == 0) *pos = *pos + inc;
}

__global__ void set_state_kernel(int *pos, int pos_value, unsigned long long *best, unsigned int *counter,
                                 int batch, int *err) {
    if (threadIdx.x == 0) {
        *pos = pos_value;
        *counter = 0u;     // last-CTA ticket of the LM head
        *err = 0;
    }
    if ((int)threadIdx.x < batch) best[threadIdx.x] = 0ull;
}

__global__ void zero_tokens_kernel(int *cur_tok, int batch) {
    if ((int)threadIdx.x < batch) cur_tok[threadIdx.x] = 0;
}

// =====================================================================================================
// GEMV family
// =====================================================================================================
template <int MODE>
__device__ __forceinline__ void unit_rows(const GemvParams &p, int u, const bf16 *&ra, const bf16 *&rb) {
    if (MODE == GEMV_QKV) {
        // unit = (head hh, i in [0,32)): rows hh*64+i and hh*64+i+32 of wq | wk | wv (RoPE pair)
        const int hh = u >> 5, i = u & 31;
        const bf16 *base;
        int h;
        if (hh < p.n_heads) { base = p.w0; h = hh; }
        else if (hh < p.n_heads + p.n_kv_heads) { base = p.w1; h = hh - p.n_heads; }
        else { base = p.w2; h = hh - p.n_heads - p.n_kv_heads; }
        ra = base + (size_t)(h * kHeadDim + i) * p.K;
        rb = ra + (size_t)32 * p.K;
    } else {
        ra = p.w0 + (size_t)(2 * u) * p.K;
        rb = ra + p.K;
    }
}

template <int CH, int U, int MODE, int XIN>
__global__ void __launch_bounds__(kGemvThreads) gemv_kernel(const __grid_constant__ GemvParams p) {
    constexpr int R = 2 * U;
    constexpr int NW = kGemvThreads / 32;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int kchunks = p.K >> 3;

    // contiguous unit range of this CTA
    const int per = p.n_units / gridDim.x, rem = p.n_units % gridDim.x;
    const int u0 = blockIdx.x * per + min((int)blockIdx.x, rem);
    const int u1 = u0 + per + ((int)blockIdx.x < rem ? 1 : 0);

    __shared__ float red[2][NW][R];
    __shared__ float red_ss[NW];

    uint4 buf0[R][CH], buf1[R][CH];

    auto load_batch = [&](uint4(&buf)[R][CH], int ub) {
#pragma unroll
        for (int j = 0; j < U; ++j) {
            const int u = ub + j;
            const bf16 *ra, *rb;
            unit_rows<MODE>(p, u < u1 ? u : u0, ra, rb);
#pragma unroll
            for (int c = 0; c < CH; ++c) {
                const int chunk = tid + c * kGemvThreads;
                if (u < u1 && chunk < kchunks) {
                    buf[2 * j][c] = ld_weight16(ra + chunk * 8);
                    buf[2 * j + 1][c] = ld_weight16(rb + chunk * 8);
                } else {
                    buf[2 * j][c] = make_uint4(0, 0, 0, 0);
                    buf[2 * j + 1][c] = make_uint4(0, 0, 0, 0);
                }
            }
        }
    };

    // ---- prefetch the first batch of weights and the gains: legal before the dependency wait ----
    load_batch(buf0, u0);
    uint4 gain[CH];
    if (XIN == XIN_NORM) {
#pragma unroll
        for (int c = 0; c < CH; ++c) {
            const int chunk = tid + c * kGemvThreads;
            gain[c] = chunk < kchunks ? ld_weight16(p.gain + chunk * 8) : make_uint4(0, 0, 0, 0);
        }
    }
    pdl_launch_dependents();
    pdl_wait();

    // ---- input vector into registers -------------------------------------------------------------
    float xr[CH][8];
    if (XIN == XIN_ATTN) {
        // merge the split-KV partials of this thread's 8 output dims (A5 combine)
        const int n_ctx = ld_act(p.pos) + 1;
        const int ns = attn_num_splits(n_ctx);
#pragma unroll
        for (int c = 0; c < CH; ++c) {
            const int chunk = tid + c * kGemvThreads;
#pragma unroll
            for (int i = 0; i < 8; ++i) xr[c][i] = 0.f;
            if (chunk < kchunks) {
                const int head = chunk >> 3, d0 = (chunk & 7) * 8;
                const float2 *ml = p.part_ml + (size_t)head * kMaxSplits;
                float M = -INFINITY;
                for (int s = 0; s < ns; ++s) M = fmaxf(M, __ldcg(&ml[s]).x);
                float denom = 0.f;
                for (int s = 0; s < ns; ++s) {
                    const float2 v = __ldcg(&ml[s]);
                    const float w = __expf(v.x - M);
                    denom += w * v.y;
                    const float *po = p.xin + ((size_t)head * kMaxSplits + s) * kHeadDim + d0;
                    const float4 a = ld_act4(po), b = ld_act4(po + 4);
                    xr[c][0] += w * a.x; xr[c][1] += w * a.y; xr[c][2] += w * a.z; xr[c][3] += w * a.w;
                    xr[c][4] += w * b.x; xr[c][5] += w * b.y; xr[c][6] += w * b.z; xr[c][7] += w * b.w;
                }
                const float inv = 1.0f / denom;
#pragma unroll
                for (int i = 0; i < 8; ++i) xr[c][i] *= inv;
            }
        }
    } else {
        float ss = 0.f;
#pragma unroll
        for (int c = 0; c < CH; ++c) {
            const int chunk = tid + c * kGemvThreads;
            if (chunk < kchunks) {
                const float4 a = ld_act4(p.xin + chunk * 8), b = ld_act4(p.xin + chunk * 8 + 4);
                xr[c][0] = a.x; xr[c][1] = a.y; xr[c][2] = a.z; xr[c][3] = a.w;
                xr[c][4] = b.x; xr[c][5] = b.y; xr[c][6] = b.z; xr[c][7] = b.w;
            } else {
#pragma unroll
                for (int i = 0; i < 8; ++i) xr[c][i] = 0.f;
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) ss = fmaf(xr[c][i], xr[c][i], ss);
        }
        if (XIN == XIN_NORM) {
            // fused RMSNorm (A2): every CTA recomputes sum(x^2) of the 8 KB, L2-resident x
            ss = warp_sum(ss);
            if (lane == 0) red_ss[warp] = ss;
            __syncthreads();
            float tot = 0.f;
#pragma unroll
            for (int w = 0; w < NW; ++w) tot += red_ss[w];
            const float inv = 1.0f / sqrtf(tot / (float)p.K + p.eps);
#pragma unroll
            for (int c = 0; c < CH; ++c) {
                const uint32_t g[4] = {gain[c].x, gain[c].y, gain[c].z, gain[c].w};
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    xr[c][2 * i] *= inv * bf16lo(g[i]);
                    xr[c][2 * i + 1] *= inv * bf16hi(g[i]);
                }
            }
        }
    }

    // per-kernel constants for the epilogues
    int pos = 0;
    if (MODE == GEMV_QKV) pos = ld_act(p.pos);

    auto epilogue = [&](int u, float a, float b) {
        if (MODE == GEMV_QKV) {
            const int hh = u >> 5, i = u & 31;
            if (hh < p.n_heads) {
                const float2 cs = p.rope[(size_t)pos * 32 + i];
                p.out[hh * kHeadDim + i] = a * cs.x - b * cs.y;
                p.out[hh * kHeadDim + i + 32] = b * cs.x + a * cs.y;
            } else if (hh < p.n_heads + p.n_kv_heads) {
                const float2 cs = p.rope[(size_t)pos * 32 + i];
                kv_t *dst = p.kc + ((size_t)(hh - p.n_heads) * p.max_seq + pos) * kHeadDim;
                dst[i] = __float2half_rn(a * cs.x - b * cs.y);
                dst[i + 32] = __float2half_rn(b * cs.x + a * cs.y);
            } else {
                kv_t *dst = p.vc + ((size_t)(hh - p.n_heads - p.n_kv_heads) * p.max_seq + pos) * kHeadDim;
                dst[i] = __float2half_rn(a);
                dst[i + 32] = __float2half_rn(b);
            }
        } else {  // GEMV_RESID
            float2 *dst = reinterpret_cast<float2 *>(p.out + 2 * u);
            float2 v = __ldcg(dst);
            v.x += a;
            v.y += b;
            *dst = v;
        }
    };

    int it = 0;
    auto compute = [&](uint4(&buf)[R][CH], int ub) {
        float acc[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            acc[r] = 0.f;
#pragma unroll
            for (int c = 0; c < CH; ++c) acc[r] = dot8(buf[r][c], xr[c], acc[r]);
        }
        warp_reduce_rows<R>(acc, lane);
        if (warp_row_leader<R>(lane)) red[it & 1][warp][warp_row_of_lane<R>(lane)] = acc[0];
        __syncthreads();
        if (tid < U && ub + tid < u1) {
            float a = 0.f, b = 0.f;
#pragma unroll
            for (int w = 0; w < NW; ++w) {
                a += red[it & 1][w][2 * tid];
                b += red[it & 1][w][2 * tid + 1];
            }
            epilogue(ub + tid, a, b);
        }
        ++it;
    };

    for (int ub = u0; ub < u1; ub += 2 * U) {
        load_batch(buf1, ub + U);
        compute(buf0, ub);
        if (ub + U >= u1) break;
        load_batch(buf0, ub + 2 * U);
        compute(buf1, ub + U);
    }

}

// =====================================================================================================
// A5: GQA split-KV flash-decode.  grid = (kMaxSplits, n_kv_heads, batch), block = 32 * G threads:
// warp w is query head kv*G + w; the G heads share each K/V tile staged in shared memory.
// =====================================================================================================
constexpr int kAttnTile = 128;  // positions per staged tile (16 KB of K + 16 KB of V)

__global__ void __launch_bounds__(256) attn_decode_kernel(const __grid_constant__ AttnDecodeParams p) {
    __shared__ __align__(128) kv_t Ks[kAttnTile * kHeadDim];
    __shared__ __align__(128) kv_t Vs[kAttnTile * kHeadDim];
    __shared__ __align__(8) uint64_t bar;
    __shared__ __align__(16) float qs[8][kHeadDim];   // q of the (<= 8) heads of the group, pre-scaled: lanes read different chunks
    __shared__ __align__(16) float ps[8][32];         // per warp: the probabilities of a round (attn_tile)

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int G = p.n_heads / p.n_kv_heads;
    const int kvh = blockIdx.y, b = blockIdx.z;
    const int head = kvh * G + warp;

    if (threadIdx.x == 0) {
        mbar_init(&bar, 1);
        mbar_fence_init();
    }
    __syncthreads();
    pdl_launch_dependents();
    pdl_wait();

    // q pre-scaled by 1/sqrt(64) = 0.125 (exact); requested together with the position (one L2 round trip, not two)
    const float2 qv = __ldcg(reinterpret_cast<const float2 *>(p.q + ((size_t)b * p.n_heads + head) * kHeadDim) + lane);
    const int n_ctx = ld_act(p.pos) + 1;
    const int ns = attn_num_splits(n_ctx);
    const int split = blockIdx.x;
    if (split >= ns) return;
    const int len = attn_split_len(n_ctx, ns);
    const int s0 = split * len;
    const int s1 = min(n_ctx, s0 + len);

    const size_t seq_base = ((size_t)b * p.n_kv_heads + kvh) * p.max_seq * kHeadDim;
    const kv_t *kg = p.kc + seq_base, *vg = p.vc + seq_base;

    qs[warp][2 * lane] = qv.x * 0.125f;
    qs[warp][2 * lane + 1] = qv.y * 0.125f;
    __syncwarp();
    float qr[8][8];
    attn_load_q(qs[warp], lane, qr);

    float m = -INFINITY, l = 0.f, o0 = 0.f, o1 = 0.f;
    uint32_t parity = 0;
    for (int t0 = s0; t0 < s1; t0 += kAttnTile) {
        const int nt = min(kAttnTile, s1 - t0);
        if (threadIdx.x == 0) {
            const uint32_t bytes = (uint32_t)nt * kHeadDim * sizeof(kv_t);
            mbar_expect_tx(&bar, 2 * bytes);
            bulk_g2s(Ks, kg + (size_t)t0 * kHeadDim, bytes, &bar);
            bulk_g2s(Vs, vg + (size_t)t0 * kHeadDim, bytes, &bar);
        }
        mbar_wait(&bar, parity);
        parity ^= 1;
        attn_tile(Ks, Vs, nt, qr, ps[warp], lane, m, l, o0, o1, 0, 32);
        __syncthreads();  // everyone done with the tile before it is overwritten
    }
    const size_t pidx = ((size_t)b * p.n_heads + head) * kMaxSplits + split;
    reinterpret_cast<float2 *>(p.part_o + pidx * kHeadDim)[lane] = make_float2(o0, o1);
    if (lane == 0) p.part_ml[pidx] = make_float2(m, l);
}

// =====================================================================================================
// Batched decode, rows P4 + B2 of SURVEY.md 8(a) in ONE launch (was three: rope_append, attn_decode, attn_combine):
// RoPE of this step's q and k, KV append, split-KV attention, split merge.  Same grid and warp roles as
// attn_decode_kernel.  Per (sequence, KV head):
//   * every split CTA rotates the q of its G heads itself (64 values per head from the fp32 Q|K|V row);
//   * the split that holds the current position rotates k, rounds k and v to the cache type, appends the row to the
//     cache AND patches it into its staged tile (the bulk copy stops one row short: it must not race the append);
//   * the splits publish their states; the one that draws the last ticket (atomic counter per (sequence, KV head),
//     reset by that CTA for the next launch) merges them in split order and writes the attention vector as bf16 planes.
// Values and summation order are those of the three kernels it replaces.
// =====================================================================================================
__global__ void __launch_bounds__(256) attn_decode_fused_kernel(const __grid_constant__ AttnFusedParams p) {
    __shared__ __align__(128) kv_t Ks[kAttnTile * kHeadDim];
    __shared__ __align__(128) kv_t Vs[kAttnTile * kHeadDim];
    __shared__ __align__(8) uint64_t bar;
    __shared__ __align__(16) float qs[8][kHeadDim];
    __shared__ __align__(16) float ps[8][32];
    __shared__ __align__(16) kv_t new_k[kHeadDim], new_v[kHeadDim];
    __shared__ int is_last;

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int G = p.n_heads / p.n_kv_heads;
    const int kvh = blockIdx.y, b = blockIdx.z;
    const int head = kvh * G + warp;

    if (threadIdx.x == 0) {
        mbar_init(&bar, 1);
        mbar_fence_init();
    }
    __syncthreads();
    pdl_launch_dependents();
    pdl_wait();

    // the Q|K|V row of this sequence: RoPE pair (lane, lane + 32) of this warp's head, requested with the position
    const int nh = p.n_heads + 2 * p.n_kv_heads;
    const float *row = p.qkv + (size_t)b * nh * kHeadDim;
    const float qa = ld_act(row + head * kHeadDim + lane), qc = ld_act(row + head * kHeadDim + lane + 32);
    // warp 0 also requests this step's k and v now (needed only by the split that holds the current position, but the
    // loads do not depend on the position: one L2 round trip instead of a third one later)
    float ka = 0.f, kc2 = 0.f, va = 0.f, vc2 = 0.f;
    if (warp == 0) {
        const float *kr = row + (p.n_heads + kvh) * kHeadDim, *vr = row + (p.n_heads + p.n_kv_heads + kvh) * kHeadDim;
        ka = ld_act(kr + lane); kc2 = ld_act(kr + lane + 32); va = ld_act(vr + lane); vc2 = ld_act(vr + lane + 32);
    }
    const int pos = ld_act(p.pos);
    const int n_ctx = pos + 1;
    const int ns = attn_num_splits(n_ctx);
    const int split = blockIdx.x;
    if (split >= ns) return;
    const int len = attn_split_len(n_ctx, ns);
    const int s0 = split * len;
    const int s1 = min(n_ctx, s0 + len);
    const bool has_new = pos >= s0 && pos < s1;

    const size_t seq_base = ((size_t)b * p.n_kv_heads + kvh) * p.max_seq * kHeadDim;
    kv_t *kg = p.kc + seq_base, *vg = p.vc + seq_base;
    const float2 cs = p.rope[(size_t)pos * 32 + lane];
    // the cached rows of the first tile are requested before the RoPE arithmetic (they depend on the position only)
    const int nt_first = min(kAttnTile, s1 - s0);
    const int nc_first = (has_new && pos < s0 + nt_first) ? nt_first - 1 : nt_first;
    if (threadIdx.x == 0 && nc_first > 0) {
        const uint32_t bytes = (uint32_t)nc_first * kHeadDim * sizeof(kv_t);
        mbar_expect_tx(&bar, 2 * bytes);
        bulk_g2s(Ks, kg + (size_t)s0 * kHeadDim, bytes, &bar);
        bulk_g2s(Vs, vg + (size_t)s0 * kHeadDim, bytes, &bar);
    }
    qs[warp][lane] = (qa * cs.x - qc * cs.y) * 0.125f;        // pre-scaled by 1/sqrt(64) (exact)
    qs[warp][lane + 32] = (qc * cs.x + qa * cs.y) * 0.125f;
    if (has_new && warp == 0) {
        // this step's k (rotated) and v, rounded exactly as the cache row later steps will read
        const kv_t k0 = __float2half_rn(ka * cs.x - kc2 * cs.y), k1 = __float2half_rn(kc2 * cs.x + ka * cs.y);
        const kv_t v0 = __float2half_rn(va), v1 = __float2half_rn(vc2);
        new_k[lane] = k0; new_k[lane + 32] = k1; new_v[lane] = v0; new_v[lane + 32] = v1;
        kv_t *dk = kg + (size_t)pos * kHeadDim, *dv = vg + (size_t)pos * kHeadDim;
        dk[lane] = k0; dk[lane + 32] = k1; dv[lane] = v0; dv[lane + 32] = v1;
    }
    __syncthreads();
    float qr[8][8];
    attn_load_q(qs[warp], lane, qr);

    float m = -INFINITY, l = 0.f, o0 = 0.f, o1 = 0.f;
    uint32_t parity = 0;
    for (int t0 = s0; t0 < s1; t0 += kAttnTile) {
        const int nt = min(kAttnTile, s1 - t0);
        const bool patch = has_new && pos < t0 + nt;          // the current position is the last row of this tile
        const int n_cached = patch ? nt - 1 : nt;
        if (n_cached > 0) {
            if (threadIdx.x == 0 && t0 > s0) {   // (the first tile was requested above)
                const uint32_t bytes = (uint32_t)n_cached * kHeadDim * sizeof(kv_t);
                mbar_expect_tx(&bar, 2 * bytes);
                bulk_g2s(Ks, kg + (size_t)t0 * kHeadDim, bytes, &bar);
                bulk_g2s(Vs, vg + (size_t)t0 * kHeadDim, bytes, &bar);
            }
            mbar_wait(&bar, parity);
            parity ^= 1;
        }
        if (patch) {
            for (int i = threadIdx.x; i < kHeadDim; i += blockDim.x) {
                Ks[(nt - 1) * kHeadDim + i] = new_k[i];
                Vs[(nt - 1) * kHeadDim + i] = new_v[i];
            }
            __syncthreads();
        }
        attn_tile(Ks, Vs, nt, qr, ps[warp], lane, m, l, o0, o1, 0, 32);
        __syncthreads();  // everyone done with the tile before it is overwritten
    }
    const size_t hb = (size_t)b * p.n_heads + head;
    const size_t pidx = hb * kMaxSplits + split;
    reinterpret_cast<float2 *>(p.part_o + pidx * kHeadDim)[lane] = make_float2(o0, o1);
    if (lane == 0) p.part_ml[pidx] = make_float2(m, l);

    // ticket: the CTA that finds ns - 1 earlier arrivals merges (its own stores and the others' are fenced before the draw)
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned int *ticket = p.tickets + (size_t)b * p.n_kv_heads + kvh;
        const unsigned int old = atomicAdd(ticket, 1u);
        is_last = old == (unsigned int)(ns - 1);
        if (is_last) *ticket = 0u;       // for the next launch (kernel boundary orders it)
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    if (lane < 8) {
        // lanes 0-7 of warp w: 8 output dims each of head kvh * G + w; arithmetic and order of attn_combine_kernel
        const int d0 = lane * 8;
        const float2 *ml = p.part_ml + hb * kMaxSplits;
        float2 mls[kMaxSplits];
#pragma unroll
        for (int s = 0; s < kMaxSplits; ++s) mls[s] = s < ns ? __ldcg(&ml[s]) : make_float2(-INFINITY, 0.f);
        float M = -INFINITY;
#pragma unroll
        for (int s = 0; s < kMaxSplits; ++s) M = fmaxf(M, mls[s].x);
        float acc[8] = {0, 0, 0, 0, 0, 0, 0, 0}, denom = 0.f;
#pragma unroll
        for (int s4 = 0; s4 < kMaxSplits; s4 += 4) {
            if (s4 < ns) {
                float4 a[4], c[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const float *po = p.part_o + (hb * kMaxSplits + s4 + u) * kHeadDim + d0;
                    const bool ok = s4 + u < ns;
                    a[u] = ok ? ld_act4(po) : make_float4(0.f, 0.f, 0.f, 0.f);
                    c[u] = ok ? ld_act4(po + 4) : make_float4(0.f, 0.f, 0.f, 0.f);
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    if (s4 + u < ns) {
                        const float w = __expf(mls[s4 + u].x - M);
                        denom += w * mls[s4 + u].y;
                        acc[0] += w * a[u].x; acc[1] += w * a[u].y; acc[2] += w * a[u].z; acc[3] += w * a[u].w;
                        acc[4] += w * c[u].x; acc[5] += w * c[u].y; acc[6] += w * c[u].z; acc[7] += w * c[u].w;
                    }
                }
            }
        }
        const float inv = 1.0f / denom;
        act_t *dst = p.out + hb * kHeadDim + d0;
#pragma unroll
        for (int i = 0; i < 8; i += 2) {
            uint32_t vh, vl;
            split_bf16x2(acc[i] * inv, acc[i + 1] * inv, vh, vl);
            *reinterpret_cast<uint32_t *>(dst + i) = vh;
            *reinterpret_cast<uint32_t *>(dst + p.lo_offset + i) = vl;
        }
    }
}

// =====================================================================================================
// launchers
// =====================================================================================================
template <typename... KArgs, typename... Args>
static cudaError_t launch_k(const LaunchCtx &c, void (*kernel)(KArgs...), dim3 grid, dim3 block, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = 0;
    cfg.stream = c.stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = c.pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

cudaError_t launch_embed(const LaunchCtx &c, const bf16 *emb, const int *tok, float *x, int hidden, int batch) {
    return launch_k(c, embed_kernel, dim3(batch), dim3(256), emb, tok, x, hidden);
}

cudaError_t launch_advance(const LaunchCtx &c, int *pos, int inc) {
    return launch_k(c, advance_kernel, dim3(1), dim3(32), pos, inc);
}

cudaError_t launch_set_state(const LaunchCtx &c, int *pos, int pos_value, unsigned long long *best,
                             unsigned int *counter, int batch, int *err) {
    LaunchCtx nc = c;
    nc.pdl = false;
    return launch_k(nc, set_state_kernel, dim3(1), dim3(32), pos, pos_value, best, counter, batch, err);
}

cudaError_t launch_zero_tokens(const LaunchCtx &c, int *cur_tok, int batch) {
    LaunchCtx nc = c;
    nc.pdl = false;
    return launch_k(nc, zero_tokens_kernel, dim3(1), dim3(32), cur_tok, batch);
}

bool gemv_shape_supported(int K) { return K > 0 && (K % 8) == 0 && K <= 8 * 4 * kGemvThreads; }

constexpr int kGemvCtasPerSm = 2;   // 2 x 256 threads x (2 buffers of 8 x 16 B) = 128 KB of weight loads in flight per SM

template <int MODE, int XIN>
static cudaError_t launch_gemv_mx(const LaunchCtx &c, const GemvParams &p) {
    const int kchunks = p.K >> 3;
    const int max_ctas = c.n_sms * kGemvCtasPerSm;
    if (kchunks <= kGemvThreads) {
        const int grid = min(max_ctas, (p.n_units + 3) / 4);
        return launch_k(c, gemv_kernel<1, 4, MODE, XIN>, dim3(grid), dim3(kGemvThreads), p);
    } else if (kchunks <= 2 * kGemvThreads) {
        const int grid = min(max_ctas, (p.n_units + 1) / 2);
        return launch_k(c, gemv_kernel<2, 2, MODE, XIN>, dim3(grid), dim3(kGemvThreads), p);
    } else {
        const int grid = min(max_ctas, p.n_units);
        return launch_k(c, gemv_kernel<4, 1, MODE, XIN>, dim3(grid), dim3(kGemvThreads), p);
    }
}

cudaError_t launch_gemv(const LaunchCtx &c, GemvMode mode, GemvInput xin, const GemvParams &p) {
    if (mode == GEMV_QKV && xin == XIN_NORM) return launch_gemv_mx<GEMV_QKV, XIN_NORM>(c, p);
    if (mode == GEMV_RESID && xin == XIN_ATTN) return launch_gemv_mx<GEMV_RESID, XIN_ATTN>(c, p);
    return cudaErrorInvalidValue;
}

cudaError_t launch_attn_decode_fused(const LaunchCtx &c, const AttnFusedParams &p, int batch) {
    const int G = p.n_heads / p.n_kv_heads;
    return launch_k(c, attn_decode_fused_kernel, dim3(kMaxSplits, p.n_kv_heads, batch), dim3(32 * G), p);
}

cudaError_t launch_attn_decode(const LaunchCtx &c, const AttnDecodeParams &p, int batch) {
    const int G = p.n_heads / p.n_kv_heads;
    return launch_k(c, attn_decode_kernel, dim3(kMaxSplits, p.n_kv_heads, batch), dim3(32 * G), p);
}

}  // namespace hq
