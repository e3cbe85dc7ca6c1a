/* hq_noalloc.h — one entry point of libhq.so that allocates NOTHING: for callers that cannot call cudaMalloc
 * (code under CUDA graph capture, tight serving loops, harnesses that forbid allocation).
 *
 * It is the split-K tensor-core GEMM of the prefill pass (north_star: "Tensor cores (tcgen05/TMEM fed by TMA) are used
 * only where the path really is a dense contraction, meaning envelope prefill and batched decode") in its
 * deterministic form: every K split STORES its partial product into a scratch buffer of its own and a second kernel adds
 * the partials in fixed order.  In the model that scratch is carved from the caller's workspace; here it is a file-scope
 * `static __device__` array inside the library:
 *
 *   - HQ_NOALLOC_SCRATCH_BYTES (16 MiB) per GPU.  Every GPU that loads the library holds it until the process exits.
 *   - The array is SHARED by every call on that GPU and keeps the contents of the last call.  Nothing in it has to
 *     start at zero: a call writes every element it later reads (splits x n_tokens x n_rows floats), so a call never
 *     sees an earlier call's data.  Calls that OVERLAP on the GPU (different streams, or different host threads whose
 *     streams are not ordered against each other) race on the array; calls on one stream are ordered and safe.
 *   - No cudaMalloc, cudaFree or allocating library routine, at set-up or per call.  Set-up (once per device) takes the
 *     device address of the array with cudaGetSymbolAddress and opts the kernels in to their shared-memory size.
 *
 * Error convention of hq.h: 0 (HQ_OK) or a negative hq_status, message in hq_last_error().  All pointers DEVICE unless
 * named otherwise; the caller owns inputs and outputs. */
#ifndef HQ_NOALLOC_H
#define HQ_NOALLOC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define HQ_NOALLOC_SCRATCH_BYTES (16u << 20)

/* Size of the static scratch array in bytes (= HQ_NOALLOC_SCRATCH_BYTES); host arithmetic, touches no GPU. */
size_t hq_noalloc_scratch_bytes(void);

/* Set-up for the CURRENT device (cudaSetDevice by the caller): resolves the device address of the scratch array and
 * prepares the kernels.  Idempotent and thread-safe; call it once per device BEFORE a stream capture or a no-allocation
 * region starts (hq_gemm_noalloc does it on first use otherwise).  HQ_ERR_CUDA if the runtime refuses; error convention
 * of hq.h. */
int32_t hq_noalloc_setup(void);

/* out[t][n] = sum_k x[t][k] * w[n][k]  (the contraction of north_star's prefill GEMMs), fp32.
 *   w:   bf16 [n_rows][k] row-major (nn.Linear layout), immutable during the call
 *   x:   bf16 [2][n_tokens][k]: the activation as two planes x = hi + lo (hi = bf16(x), lo = bf16(x - hi))
 *   out: fp32 [n_tokens][n_rows], fully overwritten
 *   token_tile in {32, 64, 128, 256}; k a multiple of 8; splits >= 1 K splits (clamped to the number of 64-element K
 *   blocks).  The result is bit-reproducible for a given (shape, token_tile, splits).
 * Scratch needed: (effective splits) x n_tokens x n_rows x 4 bytes; more than HQ_NOALLOC_SCRATCH_BYTES returns
 * HQ_ERR_CAPACITY (nothing is enqueued).  Asynchronous on cuda_stream (two kernels); see the header comment for what
 * concurrent calls may and may not do. */
int32_t hq_gemm_noalloc(void *cuda_stream, const void *w_dev, const void *x_dev, float *out_dev, int32_t n_rows, int32_t k,
                        int32_t n_tokens, int32_t token_tile, int32_t splits);

#ifdef __cplusplus
}
#endif
#endif /* HQ_NOALLOC_H */
