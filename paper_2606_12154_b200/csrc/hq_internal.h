// hq_internal.h — host-side model object and launcher prototypes shared by the libhq TUs.
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/hq_debug.h"
#include "../../include/hq_noalloc.h"

namespace hq {

typedef __nv_bfloat16 bf16;
// KV cache element type.  fp16, not bf16: same 2 bytes, 3 more mantissa bits.  With bf16 the
// cache rounding alone costs 0.008 of the 0.01 per-layer hidden-state tolerance on the 1B
// random-weight model; K/V magnitudes here are O(1..10), far from
// the fp16 range limit.
typedef __half kv_t;
// Activation operands of the tensor-core GEMMs are bf16 like the weights (tcgen05 kind::f16 rejects
// mixed fp16 x bf16 operands: illegal instruction on sm_100a), but a single bf16 rounding of the
// activations drifts the per-layer hidden state of the 1B model past the 1e-2 tolerance by layer 5
// (measured 1.04e-2).  So every activation operand is stored as TWO bf16 planes, x = hi + lo with
// hi = bf16(x), lo = bf16(x - hi) (16 mantissa bits), and every K step issues two MMAs into the same
// accumulator.  Plane layout: [2][rows][K], lo plane `rows` rows below the hi plane.
typedef __nv_bfloat16 act_t;

constexpr int kHeadDim = 64;        // only head_dim the kernels implement
constexpr int kMaxSplits = 16;      // split-KV partials per head (decode attention)
constexpr int kMinSplitLen = 64;    // do not split contexts shorter than this per split
constexpr int kGemvThreads = 256;
constexpr int kPrefillSplits = 4;   // split-K partial buffers of a prefill pass (qkv, delta): each split stores its own, consumers add in order
constexpr int kVerifyRows = 256;    // answer tokens + 1 of one hq_verify_relay call (the paper's rule: answer lines of at most ~230 tokens)
struct alignas(64) TensorMap { uint64_t opaque[16]; };   // mirrors CUtensorMap (driver type, 128 bytes)

struct LayerW {
    const bf16 *attn_norm, *wq, *wk, *wv, *wo, *ffn_norm, *w_gate, *w_up, *w_down;
};
// hq4 copies of the streamed matrices of a layer (HQ_Q4 models): codes and exponent bytes
struct LayerQ4 {
    const uint8_t *gate_q, *gate_e, *up_q, *up_e, *down_q, *down_e;
};

// Device buffers carved from the caller's workspace (see hq_api.cu carve()).
struct Buffers {
    kv_t *kcache = nullptr, *vcache = nullptr;  // [L][B][Hkv][Tmax][64] fp16
    float2 *rope = nullptr;                     // [Tmax][32] (cos, sin), built on the host in double
    // decode state / activations (fp32)
    int *pos = nullptr;                         // cached positions (device resident, graph safe)
    int *cur_tok = nullptr;                     // [B] token to feed next
    int *tok_hist = nullptr;                    // [Tmax+1][B] emitted tokens, index = pos at emission
    unsigned long long *best = nullptr;         // [B] packed argmax
    unsigned int *counter = nullptr;            // last-CTA ticket
    unsigned int *attn_tickets = nullptr;       // [B][Hkv] last-split tickets of attn_decode_fused_kernel (zero between launches)
    float *x = nullptr;                         // [B][d] residual stream
    float *q = nullptr;                         // [B][H*64]
    float *part_o = nullptr;                    // [B][H][kMaxSplits][64]
    float2 *part_ml = nullptr;                  // [B][H][kMaxSplits] (m, l)
    float *act = nullptr;                       // [B][F]
    float *logits = nullptr;                    // [B][V]
    float *hidden = nullptr;                    // [L][B][d] (capture flag)
    int *prompt = nullptr;                      // [B][Tmax] staged prompt tokens
    // row-batched (tensor-core) path: rows m = b * Tc + t of one pass, at most pf_rows of them
    int *pf_tok = nullptr;                      // [pf_rows]
    int *last_idx = nullptr;                    // [B] row of the last position of every sequence
    float *xs = nullptr;                        // [pf_rows][d] residual stream
    float *delta = nullptr;                     // [pf_rows][d] deferred output of the O / down projection (prefill passes)
    act_t *hn = nullptr;                        // [2][pf_rows][d] normalised hidden (GEMM operand, hi/lo)
    float *qkv = nullptr;                       // [pf_rows][(H+2Hkv)*64]
    __half *q16 = nullptr;                      // [pf_rows][H*64] rotated queries
    act_t *ao = nullptr;                        // [2][pf_rows][H*64] attention output (GEMM operand, hi/lo)
    act_t *actb = nullptr;                      // [2][pf_rows][F] SwiGLU output (GEMM operand, hi/lo)
    act_t *hn_last = nullptr;                   // [2][32][d] normalised last rows (LM-head operand, hi/lo)
    // verbatim-relay verification (HQ_FLAG_VERIFY)
    float *verify_logits = nullptr;             // [kVerifyRows][V]
    unsigned long long *verify_best = nullptr;  // [kVerifyRows] packed argmax per row
    int *verify_out = nullptr;                  // accepted answer tokens
    int *err = nullptr;                         // device error flag (a lost cluster arrival / tagged word traps instead of hanging)
    unsigned long long *ab_ll = nullptr;        // attention block: tagged words of the attention vector [H * 64] (zeroed at create)
    unsigned int *ab_epoch = nullptr;           // attention block: tag of the next launch (starts at 1, never reset)
};

constexpr int kTokenTiles[6] = {32, 64, 128, 256, 8, 16};   // indices 4, 5: batched decode steps of <= 8 / <= 16 sequences
struct LayerMaps { TensorMap wq, wk, wv, wo, w_gate, w_up, w_down, w_gate64, w_up64; };   // *64: 64-row boxes (EPI_SWIGLU64)

struct hq_model_impl {
    hq_config cfg;
    std::vector<LayerW> layers;
    bool q4 = false;                            // HQ_Q4: batch-1 decode streams gate/up/down/LM head as hq4
    std::vector<LayerQ4> layers_q4;
    const uint8_t *lm_head_q = nullptr, *lm_head_e = nullptr;
    const bf16 *emb = nullptr, *final_norm = nullptr, *lm_head = nullptr;
    cudaStream_t stream = nullptr;
    int device = 0;                             // CUDA device the model was created on (made current by every entry point)
    Buffers b;
    int n_sms = 148;
    int batch = 0;      // active batch (0 = none)
    int seq_len = 0;    // host mirror of *b.pos
    bool have_token = false;
    cudaGraphExec_t step_graph = nullptr;
    long long kernel_count = 0;
    int kernels_per_step = 0;
    bool use_pdl = true;
    // tensor-core path
    int pf_rows = 0;                            // row capacity of one pass
    std::vector<LayerMaps> maps;
    TensorMap map_lm_head;
    TensorMap map_hn[6], map_ao[6], map_actb[6], map_hn_last[6];   // activation maps per token tile (map_hn_last: tiles <= 32 only)
    cudaGraphExec_t batch_graph = nullptr;      // batched decode step (captured for batch_graph_b)
    int batch_graph_b = 0, batch_graph_kernels = 0, batch_eager_b = 0;
    int delta_pending = 0;                      // split-K partials of the last O / down projection of a pass not yet added to xs
    bool use_attn_block = false;                // per-step path: QKV + attention + O of a layer in one cluster launch (hq_attn.cu)
    unsigned long long *trace = nullptr;        // hq_debug_trace: device buffer [n_sms][trace_cap] or NULL
    unsigned long long *step_trace = nullptr;   // hq_debug_step_trace: device buffer [slots][4] or NULL
    int step_trace_slots = 0;
    int trace_cap = 0;
};

// ---- parameter blocks --------------------------------------------------------------------------------
enum GemvMode { GEMV_QKV = 0, GEMV_RESID = 2 };
enum GemvInput { XIN_NORM = 0, XIN_ATTN = 2 };

struct GemvParams {
    // weights: QKV uses w0=wq, w1=wk, w2=wv; RESID w0
    const bf16 *w0, *w1, *w2;
    const bf16 *gain;        // XIN_NORM
    const float *xin;        // XIN_NORM: residual x [K]; XIN_ATTN: part_o
    const float2 *part_ml;   // XIN_ATTN
    int K;                   // input features
    int n_units;             // work units (2 output rows each)
    float eps;
    // outputs
    float *out;              // QKV: q [H*64]; RESID: x (read-modify-write)
    kv_t *kc, *vc;           // QKV: this layer's cache base for sequence 0
    const float2 *rope;
    const int *pos;          // device-resident position
    int n_heads, n_kv_heads, max_seq;
};

// ---- streaming GEMV (hq_stream.cu): gate/up + SwiGLU, down + residual, LM head + argmax of batch-1 decode -------------
enum SgemvMode { SGEMV_GATEUP = 0, SGEMV_RESID = 1, SGEMV_LMHEAD = 2 };
enum SgemvInput { SGEMV_XIN_NORM = 0, SGEMV_XIN_PLANES = 1 };
struct SgemvParams {
    const bf16 *w0, *w1;     // GATEUP: gate, up [n_rows][K] each; RESID / LMHEAD: w0 [n_rows][K]
    const uint8_t *q0, *q1;  // hq4 weights instead (hq_stream_q4.cu): codes [n_rows][K / 2] ...
    const uint8_t *e0, *e1;  // ... and exponent bytes [n_rows][K / 32]; q0 == NULL: bf16 weights
    const bf16 *gain;        // XIN_NORM: RMSNorm gains [K]
    const float *xin;        // XIN_NORM: fp32 residual stream [K]; XIN_PLANES: bf16 hi plane [K] then lo plane [K]
    int K, n_rows;
    int mode, xin_mode;
    float eps;
    float *out;              // RESID: x [n_rows], += ; LMHEAD: logits [n_rows]
    bf16 *out_planes;        // GATEUP: SwiGLU vector as bf16 hi plane [n_rows] then lo plane [n_rows]
    // LMHEAD: fused argmax + step bookkeeping
    const int *pos;
    unsigned long long *best;
    unsigned int *counter;
    int *cur_tok, *tok_hist, *pos_rw;
    int pos_inc;
    int max_ctas;            // > 0: launch at most this many CTAs (leave the other SMs to the kernel that follows)
    int n_early;             // CTAs expected to start (and pre-fill their rings) while the previous kernel holds the other SMs
    float late_deficit;      // ... and how many stages more than the others each of them takes
    unsigned long long *trace;   // NULL or step timeline [slots][4] (hq_debug_step_trace)
    int trace_slot;
};
struct AttnDecodeParams {
    const float *q;          // [H*64]
    const kv_t *kc, *vc;     // layer base
    float *part_o;
    float2 *part_ml;
    const int *pos;
    int n_heads, n_kv_heads, max_seq;
};

// batched decode: RoPE + KV append + split-KV attention + split merge in one launch (attn_decode_fused_kernel)
struct AttnFusedParams {
    const float *qkv;        // fp32 [batch][(H + 2 Hkv) * 64]: this step's projections, complete (not rotated)
    kv_t *kc, *vc;           // layer base; row pos of every sequence is appended
    const float2 *rope;      // [max_seq][32] (cos, sin)
    float *part_o;
    float2 *part_ml;
    unsigned int *tickets;   // [batch][Hkv], zero between launches
    act_t *out;              // attention vector as bf16 planes: hi [batch][H * 64], lo at + lo_offset
    size_t lo_offset;
    const int *pos;
    int n_heads, n_kv_heads, max_seq;
};

// split policy shared by the attention kernel and the O-proj prologue (host + device)
__host__ __device__ inline int attn_num_splits(int n_ctx) {
    int s = (n_ctx + kMinSplitLen - 1) / kMinSplitLen;
    return s < 1 ? 1 : (s > kMaxSplits ? kMaxSplits : s);
}
__host__ __device__ inline int attn_split_len(int n_ctx, int n_splits) {
    int c = (n_ctx + n_splits - 1) / n_splits;
    return (c + 15) & ~15;  // 16-position granules
}

// records the message hq_last_error() returns and hands the code back (for entry points outside hq_api.cu)
int32_t set_error(int32_t code, const char *fmt, ...);

struct LaunchCtx {
    cudaStream_t stream;
    bool pdl;
    int n_sms;
};

bool sgemv_shape_supported(int K);
cudaError_t sgemv_prepare();
cudaError_t launch_sgemv(const LaunchCtx &c, const SgemvParams &p);   // dispatches to the hq4 kernel when p.q0 is set
bool sgemv_q4_shape_supported(int K);
cudaError_t sgemv_q4_prepare();
cudaError_t launch_sgemv_q4(const LaunchCtx &c, const SgemvParams &p);
cudaError_t launch_q4_quantize(cudaStream_t stream, const bf16 *w, size_t n_rows, int K, uint8_t *codes, uint8_t *exps);
cudaError_t launch_q4_dequantize(cudaStream_t stream, const uint8_t *codes, const uint8_t *exps, size_t n_rows, int K, bf16 *w);

// ---- attention block: A2-A6 of a layer in one cluster launch (hq_attn.cu) -----------------------------------
constexpr int kAbCluster = 8;        // CTAs per cluster = per KV head (portable cluster size)
struct AttnBlockParams {
    const bf16 *wq, *wk, *wv, *wo, *gain;   // this layer's projections and attn_norm gains
    float *x;                        // [hidden] residual stream, in and out
    kv_t *kc, *vc;                   // this layer's cache of sequence 0: [n_kv_heads][max_seq][64]
    const float2 *rope;              // [max_seq][32]
    const int *pos;                  // device-resident position
    unsigned long long *ll_attn;     // [n_heads * 64] tagged words (fp32 value | epoch tag): the attention vector
    unsigned int *epoch;             // launches so far + 1: the tag of this launch (advanced by the kernel, never reset)
    int *err;                        // device error flag (a lost arrival traps instead of hanging)
    int hidden, n_heads, n_kv_heads, max_seq;
    float eps;
    unsigned long long *trace;       // NULL or [grid][trace_cap] global-timer stamps (hq_debug_trace)
    int trace_cap;
    unsigned long long *step_trace;  // NULL or the step timeline [slots][4] (hq_debug_step_trace); this launch fills step_slot
    int step_slot;
};
size_t attn_block_smem_bytes();
bool attn_block_shape_supported(const hq_config &c);
cudaError_t attn_block_prepare(int n_kv_heads, bool *co_resident);
cudaError_t launch_attn_block(const LaunchCtx &c, const AttnBlockParams &p);

// ---- tensor-core GEMM (hq_gemm.cu) -------------------------------------------------------------------
constexpr int kGemmTraceLen = 8;   // stamps per CTA: 0 set up, 1 first stage landed, 2 last stage landed, 3 accumulator complete, 4 epilogue issued
enum GemmEpilogue { EPI_STORE = 0, EPI_RESID = 1, EPI_SWIGLU = 2, EPI_SWIGLU64 = 3 };   // 3: SwiGLU from 64-row tiles (tensor maps with 64-row boxes)
struct GemmParams {
    int K, n_rows, T, NT, k_blocks, k_blocks_per_split, stages;
    float *out_f32;
    act_t *out_act;     // hi plane; lo plane at out_act + out_lo_offset
    size_t out_lo_offset;
    int ld_out;
    int atomic;
    int x_lo_row;       // row offset of the lo plane inside the activation tensor map
    size_t split_stride;      // > 0: K split z stores its partial at out_f32 + z * split_stride (no atomics; the consumer adds them in order)
    unsigned long long *trace;   // NULL, or [CTAs along the weight rows][kGemmTraceLen] globaltimer stamps (hq_debug_gemm_timeline)
    int tiles_w1, tiles_w2;   // EPI_STORE over three stacked weight matrices: 128-row tiles of the first and second (0 = one matrix)
};
bool make_tensor_map_16b(TensorMap *out, const void *base, uint64_t rows, uint64_t cols, uint32_t box_rows);
cudaError_t gemm_prepare();   // shared-memory opt-in on the current device
cudaError_t launch_gemm(const LaunchCtx &c, GemmEpilogue mode, const TensorMap &w, const TensorMap *w2,
                        const TensorMap &x, int x_lo_row, int n_rows, int K, int T, int NT, int splits, float *out_f32,
                        act_t *out_act, size_t out_lo_offset, int ld_out, size_t split_stride = 0, unsigned long long *trace = nullptr);

cudaError_t launch_gemm_qkv(const LaunchCtx &c, const TensorMap &wq, const TensorMap &wk, const TensorMap &wv, const TensorMap &x,
                            int x_lo_row, int n1, int n2, int n3, int K, int T, int NT, int splits, float *out_f32, int ld_out,
                            size_t split_stride = 0);

// ---- row-batched kernels (hq_prefill.cu) -------------------------------------------------------------
cudaError_t launch_embed_rows(const LaunchCtx &c, const bf16 *emb, const int *tok, float *x, int hidden, int rows);
cudaError_t launch_rmsnorm_rows(const LaunchCtx &c, float *x, const float *delta, int n_parts, size_t part_stride, const bf16 *gain,
                                act_t *out, size_t lo_offset, int hidden, float eps, int rows, const int *row_index, int x_stride_rows,
                                float *zero = nullptr, int zero_per_row = 0);
cudaError_t launch_add_delta_rows(const LaunchCtx &c, float *x, const float *delta, int n_parts, size_t part_stride, size_t n);
cudaError_t launch_rope_append(const LaunchCtx &c, const float *qkv, int n_parts, size_t part_stride, __half *q16, float *q32, kv_t *kc,
                               kv_t *vc, const float2 *rope, const int *pos, int rows, int Tc, int n_heads, int n_kv_heads,
                               int max_seq);
cudaError_t launch_flash_prefill(const LaunchCtx &c, const __half *q16, const kv_t *kc, const kv_t *vc, act_t *out,
                                 size_t lo_offset, const int *pos, int batch, int Tc, int n_heads, int n_kv_heads, int max_seq);
cudaError_t launch_attn_combine(const LaunchCtx &c, const float *part_o, const float2 *part_ml, act_t *out,
                                size_t lo_offset, const int *pos, int batch, int n_heads);
cudaError_t launch_verify_rows(const LaunchCtx &c, const float *logits, int vocab, int n_rows, const int *answer, int n_envelope,
                               int *cur_tok, int *tok_hist, int *pos, unsigned int *counter, unsigned long long *best_rows,
                               int *n_accepted);
cudaError_t launch_argmax_rows(const LaunchCtx &c, const float *logits, int vocab, int batch, int *cur_tok,
                               int *tok_hist, int *pos, int pos_inc, unsigned int *counter, unsigned long long *best_rows);

// ---- read-only streaming probe (hq_probe.cu) --------------------------------------------------------
cudaError_t launch_read_probe(cudaStream_t stream, const void *src, size_t bytes, unsigned int *out, int n_sms);
cudaError_t launch_copy_probe(cudaStream_t stream, const void *src, size_t bytes, int copy_bytes, int n_ctas);

// ---- launchers (hq_decode.cu) ------------------------------------------------------------------------
cudaError_t launch_embed(const LaunchCtx &c, const bf16 *emb, const int *tok, float *x, int hidden, int batch);
cudaError_t launch_gemv(const LaunchCtx &c, GemvMode mode, GemvInput xin, const GemvParams &p);
cudaError_t launch_attn_decode(const LaunchCtx &c, const AttnDecodeParams &p, int batch);
cudaError_t launch_attn_decode_fused(const LaunchCtx &c, const AttnFusedParams &p, int batch);
cudaError_t launch_advance(const LaunchCtx &c, int *pos, int inc);
cudaError_t launch_set_state(const LaunchCtx &c, int *pos, int pos_value, unsigned long long *best,
                             unsigned int *counter, int batch, int *err);
cudaError_t launch_zero_tokens(const LaunchCtx &c, int *cur_tok, int batch);
bool gemv_shape_supported(int K);

}  // namespace hq
