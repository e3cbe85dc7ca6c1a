/*
 * hq.h — C ABI of libhq: B200 (sm_100a) prefill + streaming decode of the 1B-class dense "mouth"
 * transformer that speaks a stored entry in arxiv/paper_2606_12154.
 *
 * What the calls compute is the runtime job the paper states (§4 "Runtime phase":
 * "A 1B-class model ... then streams the answer to the user"; §6.2: "one prompt
 * evaluation" = prefill, "decode rate" = streaming generation, "TTFT" = time to first token).  The
 * paper gives no equations; the forward is the Llama-style decoder of
 * BASELINE.json `configs`, written out step by step in SURVEY.md §8(c) and DESIGN.md §2.
 *
 * Conventions
 *  - Every pointer is tagged HOST or DEVICE.  The library never allocates device memory for
 *    tensors: weights and the workspace are caller-owned (e.g. torch.empty) and BORROWED for the
 *    life of the model.  Host structs (hq_config, hq_weights and the pointer arrays inside it) are
 *    copied at create time and may be freed afterwards.
 *  - All GPU work is enqueued on the one CUDA stream given at create time, in call order.  Calls
 *    that hand a result to a HOST pointer synchronise that stream before returning; all others
 *    are asynchronous.  Asynchronous CUDA faults surface at the next synchronising call.
 *  - Every call returns HQ_OK (0) or a negative hq_status and hq_last_error() describes the failure.
 *    HQ_ERR_INVALID_ARG / CAPACITY / STATE / UNSUPPORTED are detected before any work is enqueued: the
 *    model state (KV cache length, last token) is unchanged.  After HQ_ERR_CUDA (a runtime call or a
 *    kernel failed, possibly midway through a multi-launch call) the device-side position may be ahead of
 *    the host's: call hq_kv_reset (or destroy the model) before using it again.  No exceptions, no
 *    abort().  There is NO CPU fallback: without a CUDA device the calls return HQ_ERR_CUDA.
 *  - Weight matrices are bf16, nn.Linear layout [out_features, in_features], row-major, rows
 *    16-byte aligned.  Norm gains are bf16 [hidden].  Activations inside the library: fp32
 *    residual stream, fp32 accumulators/softmax/norm statistics, fp16 KV cache (2 bytes per element,
 *    32,768 B per cached token for the 1B shape; K/V magnitudes beyond 65,504 would overflow it).  Every
 *    matrix product runs on the tensor cores with bf16 weight operands x activation operands split into two
 *    bf16 planes hi + lo (16 mantissa bits, bf16 range): mma.sync in the batch-1 decode kernels, tcgen05 in
 *    prefill / batched decode; the vectors between kernels (SwiGLU output, normalised hidden state, attention
 *    output) are stored as those two planes or as fp32.  Prefill attention computes in fp16 mma.sync.
 *  - Sequences of a batch advance in lock step (equal lengths), as in every BASELINE.json config.
 */
#ifndef HQ_H_
#define HQ_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    HQ_OK = 0,
    HQ_ERR_INVALID_ARG = -1, /* NULL where forbidden, batch/n_tokens <= 0, token id outside [0, vocab) */
    HQ_ERR_CAPACITY = -2,    /* seq_len + n_tokens > max_seq, batch > max_batch, workspace too small */
    HQ_ERR_STATE = -3,       /* e.g. decode before any prefill, hidden capture not enabled */
    HQ_ERR_CUDA = -4,        /* a CUDA runtime/driver call failed (message has the CUDA error) */
    HQ_ERR_UNSUPPORTED = -5  /* shape outside what the kernels implement (see hq_model_create) */
} hq_status;

enum { HQ_BF16 = 0, HQ_Q4 = 1 /* bf16 model whose FFN and LM-head matrices are additionally given in the 4-bit hq4 format (hq_model_create_q4) */ };
enum {
    HQ_FLAG_CAPTURE_HIDDEN = 1u, /* keep the residual stream after every layer (parity tests) */
    HQ_FLAG_NO_GRAPH = 2u,       /* launch decode kernels directly instead of replaying a CUDA graph */
    HQ_FLAG_NO_PDL = 4u,         /* no programmatic dependent launch edges between kernels */
    HQ_FLAG_VERIFY = 16u,        /* reserve workspace for hq_verify_relay: fp32 logits of 256 positions (vocab * 1 KiB) */
    HQ_FLAG_KERNEL_PER_ROW = 8u  /* batch-1 decode with one kernel per row of SURVEY.md 8(a) (QKV, attention, O as three
                                    launches) instead of the cluster attention block; also what a device that cannot keep
                                    all the block's clusters resident falls back to */
};

typedef struct hq_model hq_model; /* opaque, library-owned (host memory) */

/* Shape of the decoder (BASELINE.json configs).  HOST struct, copied. */
typedef struct {
    int32_t n_layers, hidden, n_heads, n_kv_heads, head_dim, ffn, vocab;
    float rms_eps;      /* inside the sqrt */
    float rope_theta;   /* rotate-half pairing (i, i + head_dim/2), angle pos * theta^(-2i/head_dim) */
    int32_t max_batch;  /* KV capacity: sequences */
    int32_t max_seq;    /* KV capacity: positions per sequence */
    int32_t weight_dtype; /* HQ_BF16, or HQ_Q4 with hq_model_create_q4 */
    uint32_t flags;       /* HQ_FLAG_* */
} hq_config;

/* DEVICE pointers to the weights; the arrays of per-layer pointers are HOST arrays of n_layers
 * DEVICE pointers.  lm_head may alias tok_embedding (tied head, counted once in the byte model). */
typedef struct {
    const void *tok_embedding;   /* [vocab, hidden] */
    const void *const *attn_norm; /* [hidden] */
    const void *const *wq;        /* [n_heads*head_dim, hidden] */
    const void *const *wk;        /* [n_kv_heads*head_dim, hidden] */
    const void *const *wv;        /* [n_kv_heads*head_dim, hidden] */
    const void *const *wo;        /* [hidden, n_heads*head_dim] */
    const void *const *ffn_norm;  /* [hidden] */
    const void *const *w_gate;    /* [ffn, hidden] */
    const void *const *w_up;      /* [ffn, hidden] */
    const void *const *w_down;    /* [hidden, ffn] */
    const void *final_norm;       /* [hidden] */
    const void *lm_head;          /* [vocab, hidden] */
} hq_weights;

/* Bytes of DEVICE workspace hq_model_create needs for this config (KV cache + activations +
 * RoPE table + scratch); 0 if the config is invalid.  Pure host arithmetic, needs no GPU.
 * Defined by: north_star "PyTorch used only for device memory" (the caller allocates); the KV share is the paper's
 * "context length is free" accounting (section 6.6): 2 * n_kv_heads * 64 * 2 B * n_layers per cached token. */
size_t hq_workspace_bytes(const hq_config *cfg);

/* Build a model over borrowed DEVICE weights and a borrowed DEVICE workspace (256-byte aligned,
 * >= hq_workspace_bytes).  cuda_stream is a cudaStream_t (NULL = legacy default stream).
 * Supported shapes: head_dim == 64, n_heads % n_kv_heads == 0 with group size <= 8, hidden and
 * ffn multiples of 8 and <= 8192, max_batch <= 32; anything else returns HQ_ERR_UNSUPPORTED.
 * batch 1 decodes with one CUDA graph per token: per layer one "attention block" launch (thread-block clusters, one per
 * KV head: RMSNorm, QKV, RoPE + KV append, split-KV attention, O projection, residual; shapes with hidden and
 * n_heads*head_dim <= 2048) and two fused GEMV kernels (gate/up + SwiGLU, down + residual), then the LM-head GEMV with
 * fused argmax.  The clusters of one attention-block launch wait for one another, so create proves with
 * cudaOccupancyMaxActiveClusters that all of them are resident at once ON AN OTHERWISE IDLE DEVICE and takes the
 * kernel-per-row path otherwise (as does HQ_FLAG_KERNEL_PER_ROW).  The proof does not cover a co-tenant: a model that
 * decodes with the attention block needs the device to itself (no second decoding model on another stream, no MPS
 * neighbour holding shared memory); a lost arrival traps after 2^24 polls and surfaces as HQ_ERR_CUDA at the next
 * synchronising call.  batch > 1 and prompts of >= 8 tokens run on the tcgen05 GEMM path.  The library reads no
 * environment variable.  Requires compute capability 10.x.
 * Defined by: BASELINE.json north_star ("hq_model_create from a shape config and device weight pointers"). */
int32_t hq_model_create(const hq_config *cfg, const hq_weights *weights, void *workspace_dev,
                        size_t workspace_bytes, void *cuda_stream, hq_model **out);

/* 4-bit weight-only decode.  The paper's mouth model runs at 4-bit quantisation ("A
 * 1B-class model (MiniCPM5-1B, 4-bit) then streams the answer"; section 5); its runtime's format is not
 * described and not used.  "hq4" is this library's own format: a weight row of K elements (K % 32 == 0) is cut into
 * groups of 32 consecutive elements; group exponent e = the smallest integer with max|w| <= 7 * 2^e (-126 for an all-zero
 * group, at most 120), stored as the byte e + 127; code q = round-half-to-even(w / 2^e) in [-8, 7], stored as the nibble
 * q + 8, element 2j of a row in the low nibble of byte j and element 2j + 1 in the high nibble.  The weight computed with
 * is w' = q * 2^e, exactly representable in bf16.
 *   codes: DEVICE uint8 [n_rows][K / 2];  exponent bytes: DEVICE uint8 [n_rows][K / 32]
 * hq_quantize_q4 / hq_dequantize_q4: bf16 [n_rows][k] -> hq4 -> bf16 (w'), asynchronous on cuda_stream, all DEVICE.
 * hq_model_create_q4: like hq_model_create with weight_dtype = HQ_Q4.  `weights` must hold the DEQUANTISED bf16 matrices
 * w' for w_gate, w_up, w_down of every layer and for tok_embedding / lm_head (the tensor-core paths — prefill, batched
 * decode, hq_verify_relay — compute with them), `q4` the hq4 tensors of the same matrices: batch-1 decode streams those
 * (4.25 bits per weight instead of 16) through the streaming GEMV.  Attention weights and norm gains stay bf16.  Keeping
 * the two copies consistent is the caller's business (quantise, then dequantise).  Extra shape limits: hidden a multiple of
 * 64 and <= 2048, ffn a multiple of 32 (of 1024 above 2048), vocab a multiple of 16. */
typedef struct {
    const void *const *w_gate_codes, *const *w_gate_exps; /* HOST arrays of n_layers DEVICE pointers */
    const void *const *w_up_codes, *const *w_up_exps;
    const void *const *w_down_codes, *const *w_down_exps;
    const void *lm_head_codes, *lm_head_exps;
} hq_weights_q4;
int32_t hq_quantize_q4(void *cuda_stream, const void *w_dev, int64_t n_rows, int32_t k, void *codes_dev, void *exps_dev);
/* Inverse of hq_quantize_q4 (same passage: PAPER.md:L70, L82): w' = q * 2^e as bf16, exact. */
int32_t hq_dequantize_q4(void *cuda_stream, const void *codes_dev, const void *exps_dev, int64_t n_rows, int32_t k, void *w_dev);
/* See the hq4 comment above. */
int32_t hq_model_create_q4(const hq_config *cfg, const hq_weights *weights, const hq_weights_q4 *q4, void *workspace_dev,
                           size_t workspace_bytes, void *cuda_stream, hq_model **out);

/* Frees graphs/events/handles; never the borrowed memory.  NULL is a no-op.  (Counterpart of hq_model_create.) */
void hq_model_destroy(hq_model *m);

/* Envelope prefill ("a single prompt evaluation"): feed n_tokens tokens per
 * sequence at positions seq_len .. seq_len+n_tokens-1 (appends when the cache is non-empty =
 * chunked prefill), fill the KV cache, and evaluate the LM head at the LAST position only.
 *   tokens_host      HOST  int32 [batch][n_tokens]
 *   logits_dev       DEVICE fp32 [batch][vocab], or NULL: the time-to-first-token logits
 *   first_token_host HOST  int32 [batch], or NULL: greedy argmax (lowest index on ties); when
 *                    non-NULL the call synchronises (this is the TTFT point)
 * The first call fixes the active batch (1 <= batch <= max_batch) until hq_kv_reset. */
int32_t hq_prefill(hq_model *m, const int32_t *tokens_host, int32_t batch, int32_t n_tokens,
                   float *logits_dev, int32_t *first_token_host);

/* One streaming decode step for every active sequence ("streams the answer"): feed
 * one token per sequence at position seq_len, append its K/V, emit the greedy next token.
 *   tokens_in_host  HOST int32 [batch], or NULL = feed the token emitted by the previous
 *                   prefill/step (device-resident, no host round trip); non-NULL = teacher forcing
 *   tokens_out_host HOST int32 [batch], or NULL = stay asynchronous (no sync, no copy) */
int32_t hq_decode_step(hq_model *m, const int32_t *tokens_in_host, int32_t *tokens_out_host);

/* n_steps free-running greedy decode steps enqueued back to back (no host round trip between
 * them): the "decode rate" of PAPER.md:L109-111 (section 6.2) is this call's tokens per second.
 * tokens_out_host: HOST int32 [n_steps][batch] or NULL (asynchronous). */
int32_t hq_decode_run(hq_model *m, int32_t n_steps, int32_t *tokens_out_host);

/* Verbatim-relay verification in one dense pass.  The paper's renderer LOCKS the answer line before
 * the mouth speaks it ("the factual content is locked by the renderer, and the small model's job is
 * delivery") and its section 6.4 measures whether the mouth then repeats the line verbatim.  Since
 * the expected tokens are known in advance, one prefill-style pass over envelope + answer scores every answer position at
 * once (tensor-core GEMMs, weights read once) instead of one decode step per token; speculative decoding is the related
 * work the paper cites.  The call is not in the paper.
 *   tokens_host      HOST int32 [n_envelope + n_answer]: the rendered envelope, then the answer line; ONE sequence,
 *                    appended at seq_len; n_answer <= 255, n_envelope + n_answer <= 2,048
 *   n_accepted_host  HOST int32: how many leading answer tokens the greedy argmax reproduces (0 .. n_answer); synchronises
 * On return the cache holds envelope + accepted tokens (seq_len += n_envelope + n_accepted) and the device-resident
 * "last emitted token" is the model's own greedy choice at the first mismatch (after the whole answer when everything
 * matched), so hq_decode_step(m, NULL, ...) streams on from there and hq_decode_logits returns the logits that chose it.
 * Needs HQ_FLAG_VERIFY (HQ_ERR_STATE otherwise). */
int32_t hq_verify_relay(hq_model *m, const int32_t *tokens_host, int32_t n_envelope, int32_t n_answer,
                        int32_t *n_accepted_host);

/* Parity (north_star: "relative L2 <= 1e-2 per-layer hidden state, <= 2e-2 on logits" against the oracle).
 * logits_dev: DEVICE fp32 [batch][vocab] <- logits of the last prefill/step.
 * hidden_dev: DEVICE fp32 [batch][hidden] <- residual stream after `layer` at the last position
 * of the last prefill/step (needs HQ_FLAG_CAPTURE_HIDDEN).  Asynchronous device-to-device copies. */
int32_t hq_decode_logits(hq_model *m, float *logits_dev);
/* Same passage as hq_decode_logits (north_star parity tolerances): the per-layer hidden state. */
int32_t hq_get_hidden(hq_model *m, int32_t layer, float *hidden_dev);

/* Block until everything enqueued so far has finished (the point at which PAPER.md:L109 "end-to-end wall" stops). */
int32_t hq_sync(hq_model *m);

/* Cached positions per sequence (host mirror; exact because lengths advance in lock step): the context the paper's
 * section 6.6 sweeps. */
int32_t hq_seq_len(const hq_model *m, int32_t *out);

/* seq_len <- 0, active batch cleared; the cache memory is not scrubbed.  north_star "hq_kv_reset": every query of the
 * paper's runtime is independent (route, render, speak), so the cache restarts per query. */
int32_t hq_kv_reset(hq_model *m);

/* Thread-local message of the last failing call on this thread; static storage, never NULL (error convention above). */
const char *hq_last_error(void);

/* Library version string, e.g. "hq 0.2 sm_100a" (north_star: "built for sm_100a"; the tests check the suffix). */
const char *hq_version(void);

#ifdef __cplusplus
}
#endif
#endif /* HQ_H_ */
