/*
 * hq_debug.h — measurement and diagnostic entry points of libhq, kept apart from the product ABI (hq.h).
 * bench.py's roofline leg, the ncu captures under profiles/ and the GEMM unit tests call these; an
 * application that speaks an answer needs none of them.
 */
#ifndef HQ_DEBUG_H_
#define HQ_DEBUG_H_

#include "hq.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Measurement hooks (bench.py roofline leg, ncu).  hq_kernel_count: kernels launched by this
 * model since create (graph replays count their kernel nodes).  hq_bench_kernel: enqueue `reps`
 * launches of one named kernel family of the decode step, cycling over layers so that the weights
 * streamed exceed L2: which = 0 gate/up+SwiGLU GEMV, 1 LM head+argmax, 2 QKV+RoPE, 3 O-proj,
 * 4 down-proj, 5 split-KV attention.  Needs a prefilled cache; results are discarded (the
 * residual stream is garbage afterwards: call hq_kv_reset + prefill again before decoding).
 * bytes_per_launch (HOST, may be NULL) receives the algorithmic HBM bytes of one launch. */
int64_t hq_kernel_count(const hq_model *m);
/* Which batch-1 decode path this model runs (decided at create from the shape, the flags and the device): static
 * string, "attention-block-cluster" (default) or "kernel-per-row" (HQ_FLAG_KERNEL_PER_ROW, unsupported shape, or clusters
 * not co-resident). */
const char *hq_decode_path(const hq_model *m);
int32_t hq_bench_kernel(hq_model *m, int32_t which, int32_t reps, int64_t *bytes_per_launch);

/* Diagnostics: the tcgen05 GEMM of the prefill / batched-decode path on its own (unit tests).
 * All pointers DEVICE.  w, w2: bf16 [n_rows][k]; x: bf16 [2][n_tokens][k], the activation as two planes
 * x = hi + lo (hi = bf16(x), lo = bf16(x - hi)); token_tile in {32,64,128,256}, or 8 / 16 (the batched-decode
 * tiles for <= 8 / <= 16 sequences; not in mode 2).
 *   mode 0: out fp32 [n_tokens][n_rows]  = x w^T   (splits > 1: out must be zeroed, partials add atomically)
 *   mode 1: out fp32 [n_tokens][n_rows] += x w^T   (residual epilogue)
 *   mode 2: out bf16 [2][n_tokens][n_rows] = hi/lo planes of silu(x w^T) * (x w2^T)   (SwiGLU epilogue)
 *   mode 3: the result of mode 2 computed from 64-row weight tiles (the batched-decode form; n_rows % 64 == 0)
 * Asynchronous on cuda_stream. */
int32_t hq_debug_gemm(void *cuda_stream, int32_t mode, const void *w_dev, const void *w2_dev, const void *x_dev,
                      void *out_dev, int32_t n_rows, int32_t k, int32_t n_tokens, int32_t token_tile, int32_t splits);

/* Measurement: hq_debug_gemm with a timeline (profiles/r02_launches.md).  trace_dev: DEVICE uint64
 * [CTAs along the weight rows][8] (ceil(n_rows / 128) CTAs, n_rows / 64 for mode 3, rounded up to even for CTA pairs);
 * every CTA of the first token tile and K split writes GPU globaltimer values (ns): [0] barriers and tensor memory set up,
 * [1] first stage of operands landed, [2] last stage landed, [3] accumulator complete (all MMAs retired),
 * [4] epilogue of the stamping warp issued.  Same arguments, result and asynchrony as hq_debug_gemm. */
int32_t hq_debug_gemm_timeline(void *cuda_stream, int32_t mode, const void *w_dev, const void *w2_dev, const void *x_dev,
                               void *out_dev, int32_t n_rows, int32_t k, int32_t n_tokens, int32_t token_tile,
                               int32_t splits, uint64_t *trace_dev);

/* Measurement: read-only streaming probe: one launch sums the 32-bit words of src_dev[0, bytes) into
 * *sum_dev (atomicAdd, wraps; DEVICE uint32, caller-zeroed).  Time it with CUDA events on cuda_stream over a buffer much
 * larger than L2: bytes / time is what a kernel that only reads HBM reaches on this box.  Asynchronous. */
int32_t hq_debug_read_probe(void *cuda_stream, const void *src_dev, size_t bytes, uint32_t *sum_dev);

/* Measurement: what an SM pulls from HBM through cp.async.bulk as a function of the size of the individual copy.  One
 * launch: n_ctas CTAs (one per SM) each stream their share of src_dev[0, bytes) through a ring of 3 x 64 KB shared-memory
 * stages, a stage being 64 KB / copy_bytes bulk copies; nothing is computed.  bytes_streamed = n_ctas * floor(bytes /
 * 65536 / n_ctas) * 65536.  copy_bytes: power of two in [16, 65536].  Time it with CUDA events.  Asynchronous. */
int32_t hq_debug_copy_probe(void *cuda_stream, const void *src_dev, size_t bytes, int32_t copy_bytes, int32_t n_ctas);

/* Parity: one cached position read back.  which = 0 (K, rotated) or 1 (V); row_dev: DEVICE fp16 [n_kv_heads][64] <-
 * the cache row of `layer`, sequence `seq`, position `pos` (the cache itself is [L][B][Hkv][max_seq][64] fp16).
 * Asynchronous device-to-device copy on the model's stream. */
int32_t hq_debug_kv_row(hq_model *m, int32_t which, int32_t layer, int32_t seq, int32_t pos, void *row_dev);

/* Diagnostics: timeline of one batch-1 decode step.  trace_dev: DEVICE uint64 [n_slots][4] with n_slots >= 2 + 3 *
 * n_layers, or NULL to switch off.  While set, every directly launched decode kernel (HQ_FLAG_NO_GRAPH; a captured graph
 * keeps the setting it was captured with) updates its slot — 1 + 3 l attention block, 2 + 3 l gate/up, 3 + 3 l down of
 * layer l, 1 + 3 n_layers the LM head — with global-timer stamps (ns): [0] min over CTAs of the CTA start, [1] min of the
 * end of the dependency wait, [2] max of the CTA end, [3] max of the CTA start.  The caller initialises [0], [1] to
 * UINT64_MAX and [2], [3] to 0 before the step.  The buffer is BORROWED until tracing is switched off. */
int32_t hq_debug_step_trace(hq_model *m, uint64_t *trace_dev, int32_t n_slots);

/* Diagnostics: timeline of the attention block.  trace_dev: DEVICE uint64 [n_ctas][cap] (n_ctas = 8 * n_kv_heads), or
 * NULL to switch tracing off.  While set, thread 0 of every CTA of an attention-block launch stores the GPU global timer
 * (ns) at fixed points of the launch (see ab_trace in csrc/hq_attn.cu), restarting at index 0 each launch; stamps beyond
 * cap are dropped.  The buffer is BORROWED until tracing is switched off.  Takes effect for direct launches
 * (hq_bench_kernel, HQ_FLAG_NO_GRAPH); a captured graph keeps the setting it was captured with. */
int32_t hq_debug_trace(hq_model *m, uint64_t *trace_dev, int32_t cap);

#ifdef __cplusplus
}
#endif
#endif /* HQ_DEBUG_H_ */
