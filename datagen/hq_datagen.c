/*
 * hq_datagen — seeded synthetic inputs (weights, gains, tokens) for BOTH the CPU oracle and
 * the CUDA path.  This module holds NONE of the method's arithmetic: it only draws numbers.
 *
 * Recipe (SURVEY.md §8(c) readings 3, 4, 5, 16; BASELINE.json configs: "weights ~N(0,0.02)",
 * "uniform-random token ids"):
 *   key      = mix(seed ^ tensor_id * 0x9E3779B97F4A7C15)
 *   r_i      = mix(key + i)                                  (counter based, order independent)
 *   u1       = (hi32(r_i) + 1) / 2^32  in (0,1],  u2 = lo32(r_i) / 2^32  in [0,1)
 *   z_i      = sqrt(-2 ln u1) * cos(2 pi u2)                 (Box-Muller, double)
 *   normal   : value_i = (float)(mean + std * z_i)
 *   token    : r_i mod vocab
 * mix() is the SplitMix64 output function applied to (x + golden gamma); mix(0) is the
 * published first output of SplitMix64 seeded with 0, 0xE220A8397B1DCDAF (pinned in tests).
 * bf16 rounding is round-to-nearest-even on the fp32 bit pattern.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

static inline uint64_t mix64(uint64_t x) {
    uint64_t z = x + 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

uint64_t hqd_mix64(uint64_t x) { return mix64(x); }

uint64_t hqd_key(uint64_t seed, uint64_t tensor_id) {
    return mix64(seed ^ (tensor_id * 0x9E3779B97F4A7C15ULL));
}

/* out[i] = (float)(mean + std * z_i), i in [0, n) */
void hqd_normal_f32(uint64_t seed, uint64_t tensor_id, double mean, double std, float *out, size_t n) {
    const uint64_t key = hqd_key(seed, tensor_id);
    const double two_pi = 6.283185307179586476925286766559;
#pragma omp parallel for schedule(static)
    for (size_t i = 0; i < n; ++i) {
        uint64_t r = mix64(key + (uint64_t)i);
        double u1 = ((double)(uint32_t)(r >> 32) + 1.0) * (1.0 / 4294967296.0);
        double u2 = (double)(uint32_t)(r & 0xFFFFFFFFu) * (1.0 / 4294967296.0);
        double z = sqrt(-2.0 * log(u1)) * cos(two_pi * u2);
        out[i] = (float)(mean + std * z);
    }
}

/* out[i] = r_i mod vocab */
void hqd_tokens_i32(uint64_t seed, uint64_t tensor_id, int32_t vocab, int32_t *out, size_t n) {
    const uint64_t key = hqd_key(seed, tensor_id);
    for (size_t i = 0; i < n; ++i) out[i] = (int32_t)(mix64(key + (uint64_t)i) % (uint64_t)vocab);
}

/* fp32 -> bf16 bits, round to nearest even (inputs are finite by construction) */
void hqd_f32_to_bf16(const float *in, uint16_t *out, size_t n) {
#pragma omp parallel for schedule(static)
    for (size_t i = 0; i < n; ++i) {
        union { float f; uint32_t u; } v;
        v.f = in[i];
        uint32_t u = v.u;
        u += 0x7FFFu + ((u >> 16) & 1u);
        out[i] = (uint16_t)(u >> 16);
    }
}

/* bf16 bits -> fp32 (exact) */
void hqd_bf16_to_f32(const uint16_t *in, float *out, size_t n) {
#pragma omp parallel for schedule(static)
    for (size_t i = 0; i < n; ++i) {
        union { float f; uint32_t u; } v;
        v.u = ((uint32_t)in[i]) << 16;
        out[i] = v.f;
    }
}
