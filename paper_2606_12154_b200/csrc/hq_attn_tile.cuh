// hq_attn_tile.cuh — the inner loop of decode attention of hq_decode.cu (batched decode and the kernel-per-row path).
// The batch-1 attention block (hq_attn.cu) keeps its own lane-group loop: with 8 warps alone on an SM it is latency-bound,
// and this loop's serial phases per round measured 4-16 % slower there (profiles/r02_sgemv_log.md).
#pragma once
#include "hq_common.cuh"
#include "hq_internal.h"

namespace hq {

// ---- decode attention over one staged K/V tile.  Tile rows are cached positions, 64 fp16 each, back to back.
// One staged tile of nt positions for one query head (one warp): online softmax over the tile, state (m, l, o0, o1) =
// running max, denominator and this lane's two output dims.
//   qr: the head's query, pre-scaled, in REGISTERS, chunk c of this lane = dims [8 ((c + lane) & 7), + 8) (attn_load_q): the
//       order in which the lane walks its K row, so that the 8 lanes of a quarter-warp hit 8 different bank groups;
//   ps: 32 floats of shared memory of this warp: the probabilities of a round, read back four at a time as broadcasts
//       (one LDS.128 per four positions instead of four shuffles).
__device__ __forceinline__ void attn_load_q(const float *q_smem, int lane, float (&qr)[8][8]) {
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const int cc = (c + lane) & 7;
        const float4 a = *reinterpret_cast<const float4 *>(q_smem + cc * 8), b = *reinterpret_cast<const float4 *>(q_smem + cc * 8 + 4);
        qr[c][0] = a.x; qr[c][1] = a.y; qr[c][2] = a.z; qr[c][3] = a.w; qr[c][4] = b.x; qr[c][5] = b.y; qr[c][6] = b.z; qr[c][7] = b.w;
    }
}
__device__ __forceinline__ void attn_tile(const kv_t *Ks, const kv_t *Vs, int nt, const float (&qr)[8][8], float *ps, int lane, float &m,
                                          float &l, float &o0, float &o1, int r_begin, int r_step) {
    // rounds of 32 positions r_begin, r_begin + r_step, ... (0, 32: the whole tile; sub-split s of n: 32 s, 32 n)
    for (int r0 = r_begin; r0 < nt; r0 += r_step) {
        const int nr = min(32, nt - r0);
        // scores of up to 32 positions: lane i computes the whole dot product of position r0 + i (one warp reduction per
        // position made this loop a chain of 5 dependent shuffles x 32: 2.6 us per 32 positions)
        float s_mine = -INFINITY;
        if (lane < nr) {
            const uint4 *krow = reinterpret_cast<const uint4 *>(Ks + (r0 + lane) * kHeadDim);
            float acc4[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                const uint4 kk = krow[(c + lane) & 7];
                const float2 k0 = __half22float2(*reinterpret_cast<const __half2 *>(&kk.x));
                const float2 k1 = __half22float2(*reinterpret_cast<const __half2 *>(&kk.y));
                const float2 k2 = __half22float2(*reinterpret_cast<const __half2 *>(&kk.z));
                const float2 k3 = __half22float2(*reinterpret_cast<const __half2 *>(&kk.w));
                acc4[0] = fmaf(qr[c][0], k0.x, fmaf(qr[c][1], k0.y, acc4[0]));
                acc4[1] = fmaf(qr[c][2], k1.x, fmaf(qr[c][3], k1.y, acc4[1]));
                acc4[2] = fmaf(qr[c][4], k2.x, fmaf(qr[c][5], k2.y, acc4[2]));
                acc4[3] = fmaf(qr[c][6], k3.x, fmaf(qr[c][7], k3.y, acc4[3]));
            }
            s_mine = (acc4[0] + acc4[1]) + (acc4[2] + acc4[3]);
        }
        const float m_new = fmaxf(m, warp_max(s_mine));
        const float corr = __expf(m - m_new);   // m = -inf first time -> 0
        const float pr = (lane < nr) ? __expf(s_mine - m_new) : 0.f;
        l = l * corr + warp_sum(pr);
        o0 *= corr;
        o1 *= corr;
        ps[lane] = pr;
        __syncwarp();
        for (int r = 0; r < nr; r += 4) {
            const float4 p4 = *reinterpret_cast<const float4 *>(ps + r);   // broadcast
            const float pb[4] = {p4.x, p4.y, p4.z, p4.w};
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                if (r + u < nr) {   // warp-uniform; rows past nr of the tile are not initialised
                    const float2 vv = __half22float2(*reinterpret_cast<const __half2 *>(Vs + (r0 + r + u) * kHeadDim + 2 * lane));
                    o0 = fmaf(pb[u], vv.x, o0);
                    o1 = fmaf(pb[u], vv.y, o1);
                }
            }
        }
        __syncwarp();   // ps is rewritten by the next round
        m = m_new;
    }
}

}  // namespace hq
