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
 *  - Every call returns HQ_OK (0) or a negative hq_status; on error the model state (KV cache
 *    length, last token) is unchanged and hq_last_error() describes the failure.  No exceptions,
 *    no abort().  There is NO CPU fallback: without a CUDA device the calls return HQ_ERR_CUDA.
 *  - Weight matrices are bf16, nn.Linear layout [out_features, in_features], row-major, rows
 *    16-byte aligned.  Norm gains are bf16 [hidden].  Activations inside the library: fp32
 *    residual stream, fp32 accumulators/softmax/norm statistics, fp16 KV cache (2 bytes per element,
 *    32,768 B per cached token for the 1B shape), on the tensor cores (prefill / batched decode only) bf16
 *    weight operands x activation operands split into two bf16 planes hi + lo (16 mantissa bits).
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

enum { HQ_BF16 = 0 };
enum {
    HQ_FLAG_CAPTURE_HIDDEN = 1u, /* keep the residual stream after every layer (parity tests) */
    HQ_FLAG_NO_GRAPH = 2u,       /* launch decode kernels directly instead of replaying a CUDA graph */
    HQ_FLAG_NO_PDL = 4u,         /* no programmatic dependent launch edges between kernels */
    HQ_FLAG_NO_MEGA = 8u,        /* never use the persistent decode kernel (wins over HQ_FLAG_MEGA and the HQ_MEGA environment variable) */
    HQ_FLAG_MEGA = 16u           /* batch-1 decode in ONE persistent kernel per call instead of one kernel per step of the path */
};

typedef struct hq_model hq_model; /* opaque, library-owned (host memory) */

/* Shape of the decoder (BASELINE.json configs).  HOST struct, copied. */
typedef struct {
    int32_t n_layers, hidden, n_heads, n_kv_heads, head_dim, ffn, vocab;
    float rms_eps;      /* inside the sqrt */
    float rope_theta;   /* rotate-half pairing (i, i + head_dim/2), angle pos * theta^(-2i/head_dim) */
    int32_t max_batch;  /* KV capacity: sequences */
    int32_t max_seq;    /* KV capacity: positions per sequence */
    int32_t weight_dtype; /* HQ_BF16 */
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
 * RoPE table + scratch); 0 if the config is invalid.  Pure host arithmetic, needs no GPU. */
size_t hq_workspace_bytes(const hq_config *cfg);

/* Build a model over borrowed DEVICE weights and a borrowed DEVICE workspace (256-byte aligned,
 * >= hq_workspace_bytes).  cuda_stream is a cudaStream_t (NULL = legacy default stream).
 * Supported shapes: head_dim == 64, n_heads % n_kv_heads == 0 with group size <= 8, hidden and
 * ffn multiples of 8 and <= 8192, max_batch <= 32; anything else returns HQ_ERR_UNSUPPORTED.
 * batch 1 decodes, by default, with one CUDA graph per token: per layer one "attention block" launch (RMSNorm, QKV,
 * RoPE + KV append, split-KV attention, O projection, residual; shapes with hidden and n_heads*head_dim <= 2048) and two
 * fused GEMV kernels (gate/up + SwiGLU, down + residual), then the LM-head GEMV with fused argmax.  HQ_FLAG_MEGA runs the
 * whole of hq_decode_run in ONE persistent kernel (TMA-fed weight ring, tagged-word exchange between the SMs, no grid
 * barrier); HQ_FLAG_NO_MEGA uses one kernel per step of the path.  batch > 1 and prompts of >= 8 tokens run on the tcgen05
 * GEMM path.
 * Requires compute capability 10.x. */
int32_t hq_model_create(const hq_config *cfg, const hq_weights *weights, void *workspace_dev,
                        size_t workspace_bytes, void *cuda_stream, hq_model **out);

/* Frees graphs/events/handles; never the borrowed memory.  NULL is a no-op. */
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
 * them).  tokens_out_host: HOST int32 [n_steps][batch] or NULL (asynchronous). */
int32_t hq_decode_run(hq_model *m, int32_t n_steps, int32_t *tokens_out_host);

/* Parity/diagnostics.  logits_dev: DEVICE fp32 [batch][vocab] <- logits of the last prefill/step.
 * hidden_dev: DEVICE fp32 [batch][hidden] <- residual stream after `layer` at the last position
 * of the last prefill/step (needs HQ_FLAG_CAPTURE_HIDDEN).  Asynchronous device-to-device copies. */
int32_t hq_decode_logits(hq_model *m, float *logits_dev);
int32_t hq_get_hidden(hq_model *m, int32_t layer, float *hidden_dev);

/* Block until everything enqueued so far has finished. */
int32_t hq_sync(hq_model *m);

/* Cached positions per sequence (host mirror; exact because lengths advance in lock step). */
int32_t hq_seq_len(const hq_model *m, int32_t *out);

/* seq_len <- 0, active batch cleared; the cache memory is not scrubbed. */
int32_t hq_kv_reset(hq_model *m);

/* Measurement hooks (bench.py roofline leg, ncu).  hq_kernel_count: kernels launched by this
 * model since create (graph replays count their kernel nodes).  hq_bench_kernel: enqueue `reps`
 * launches of one named kernel family of the decode step, cycling over layers so that the weights
 * streamed exceed L2: which = 0 gate/up+SwiGLU GEMV, 1 LM head+argmax, 2 QKV+RoPE, 3 O-proj,
 * 4 down-proj, 5 split-KV attention.  Needs a prefilled cache; results are discarded (the
 * residual stream is garbage afterwards: call hq_kv_reset + prefill again before decoding).
 * bytes_per_launch (HOST, may be NULL) receives the algorithmic HBM bytes of one launch. */
int64_t hq_kernel_count(const hq_model *m);
/* Which batch-1 decode path this model runs (decided at create from the shape, the flags and the device): static
 * string, "attention-block-cluster" (default), "kernel-per-row" (HQ_FLAG_NO_MEGA or unsupported shape / clusters not
 * co-resident) or "persistent" (HQ_FLAG_MEGA). */
const char *hq_decode_path(const hq_model *m);
int32_t hq_bench_kernel(hq_model *m, int32_t which, int32_t reps, int64_t *bytes_per_launch);

/* Diagnostics: the tcgen05 GEMM of the prefill / batched-decode path on its own (unit tests).
 * All pointers DEVICE.  w, w2: bf16 [n_rows][k]; x: bf16 [2][n_tokens][k], the activation as two planes
 * x = hi + lo (hi = bf16(x), lo = bf16(x - hi)); token_tile in {32,64,128,256}.
 *   mode 0: out fp32 [n_tokens][n_rows]  = x w^T   (splits > 1: out must be zeroed, partials add atomically)
 *   mode 1: out fp32 [n_tokens][n_rows] += x w^T   (residual epilogue)
 *   mode 2: out bf16 [2][n_tokens][n_rows] = hi/lo planes of silu(x w^T) * (x w2^T)   (SwiGLU epilogue)
 * Asynchronous on cuda_stream. */
int32_t hq_debug_gemm(void *cuda_stream, int32_t mode, const void *w_dev, const void *w2_dev, const void *x_dev,
                      void *out_dev, int32_t n_rows, int32_t k, int32_t n_tokens, int32_t token_tile, int32_t splits);

/* Diagnostics: timeline of the persistent batch-1 decode kernel.  trace_dev: DEVICE uint64 [n_ctas][cap] (n_ctas =
 * number of SMs), or NULL to switch tracing off.  While set, thread 0 of every CTA stores the GPU global timer (ns)
 * at the start of the launch and then, in program order, three times per phase — weight phases (QKV, O, gate/up, down,
 * LM head): input staged / first ring stage landed / phase consumed; attention (after QKV): query polled / computed /
 * published — plus once when the next token is known, for every step of every later launch, restarting at index 0 each
 * launch; stamps beyond cap are dropped.  The buffer is BORROWED until tracing is switched off.  Takes effect for direct
 * launches (hq_decode_run with HQ_FLAG_MEGA, the attention block of hq_bench_kernel); a captured graph keeps the setting it
 * was captured with. */
int32_t hq_debug_trace(hq_model *m, uint64_t *trace_dev, int32_t cap);

/* Thread-local message of the last failing call on this thread; static storage, never NULL. */
const char *hq_last_error(void);

/* Library version string, e.g. "hq 0.1 sm_100a". */
const char *hq_version(void);

#ifdef __cplusplus
}
#endif
#endif /* HQ_H_ */
