// hq_api.cu — the C ABI of include/hq.h: argument checking, workspace carve-up, step scheduling,
// CUDA-graph capture.  Every step of the path runs in the kernels of hq_decode.cu / hq_prefill.cu;
// there is no CPU fallback anywhere in this file.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "hq_internal.h"

using namespace hq;

struct hq_model : public hq_model_impl {};

static thread_local char g_err[512] = "";

static int32_t fail(int32_t code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define HQ_CUDA(call)                                                                                  \
    do {                                                                                               \
        cudaError_t e__ = (call);                                                                      \
        if (e__ != cudaSuccess)                                                                        \
            return fail(HQ_ERR_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e__), __FILE__, \
                        __LINE__);                                                                     \
    } while (0)

extern "C" const char *hq_last_error(void) { return g_err; }

// the same message buffer for entry points that live in other files (hq_noalloc.cu)
namespace hq {
int32_t set_error(int32_t code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}
}  // namespace hq

// Every entry point that touches the GPU makes the model's device current first (a caller may have switched devices
// between calls; kernel attributes and launches are per device).
#define HQ_ON_DEVICE(m) HQ_CUDA(cudaSetDevice((m)->device))
extern "C" const char *hq_version(void) { return "hq 0.2 sm_100a"; }

// ---- workspace layout ---------------------------------------------------------------------------------
static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

static bool config_ok(const hq_config *c, const char **why) {
#define BAD(msg) do { *why = msg; return false; } while (0)
    if (!c) BAD("cfg is NULL");
    if (c->n_layers <= 0 || c->hidden <= 0 || c->n_heads <= 0 || c->n_kv_heads <= 0 || c->ffn <= 0 ||
        c->vocab <= 0 || c->max_batch <= 0 || c->max_seq <= 0)
        BAD("non-positive dimension");
    if (c->weight_dtype != HQ_BF16 && c->weight_dtype != HQ_Q4) BAD("weight_dtype must be HQ_BF16 or HQ_Q4");
    return true;
#undef BAD
}

static bool config_supported(const hq_config *c, const char **why) {
#define BAD(msg) do { *why = msg; return false; } while (0)
    if (c->head_dim != kHeadDim) BAD("head_dim must be 64");
    if (c->n_heads % c->n_kv_heads != 0) BAD("n_heads must be a multiple of n_kv_heads");
    if (c->n_heads / c->n_kv_heads > 8) BAD("GQA group size must be <= 8");
    if (!gemv_shape_supported(c->hidden) || !gemv_shape_supported(c->ffn) ||
        !gemv_shape_supported(c->n_heads * c->head_dim) || !sgemv_shape_supported(c->hidden) || !sgemv_shape_supported(c->ffn))
        BAD("hidden, ffn and n_heads*head_dim must be multiples of 8 (of 16 above 2048) and <= 8192");
    if (c->vocab % 2 != 0 || c->hidden % 2 != 0) BAD("vocab and hidden must be even");
    if (c->max_batch > 32) BAD("max_batch must be <= 32");
    if (c->n_kv_heads > 56) BAD("n_kv_heads must be <= 56");
    return true;
#undef BAD
}

// Row capacity of one row-batched pass (tokens of all sequences together), a multiple of 256.
static size_t pass_rows(const hq_config *c) {
    size_t r = (size_t)c->max_batch * c->max_seq;
    if (r > 2048) r = 2048;
    if (r < (size_t)c->max_batch) r = c->max_batch;
    return (r + 255) / 256 * 256;
}

// Walks the layout; when base != NULL also assigns the pointers.
static size_t carve(const hq_config *c, char *base, Buffers *b) {
    size_t off = 0;
    auto take = [&](size_t bytes) -> char * {
        char *p = base ? base + off : nullptr;
        off = align_up(off + bytes, 256);
        return p;
    };
    const size_t B = c->max_batch, L = c->n_layers, T = c->max_seq, d = c->hidden;
    const size_t H = c->n_heads, Hkv = c->n_kv_heads, F = c->ffn, V = c->vocab;
    const size_t kv_elems = L * B * Hkv * T * kHeadDim;
    Buffers tmp;
    Buffers &o = b ? *b : tmp;
    o.kcache = (kv_t *)take(kv_elems * sizeof(kv_t));
    o.vcache = (kv_t *)take(kv_elems * sizeof(kv_t));
    o.rope = (float2 *)take(T * 32 * sizeof(float2));
    o.pos = (int *)take(sizeof(int));
    o.cur_tok = (int *)take(B * sizeof(int));
    o.tok_hist = (int *)take((T + 1) * B * sizeof(int));
    o.best = (unsigned long long *)take(B * sizeof(unsigned long long));
    o.counter = (unsigned int *)take(sizeof(unsigned int));
    o.attn_tickets = (unsigned int *)take(B * Hkv * sizeof(unsigned int));
    o.x = (float *)take(B * d * sizeof(float));
    o.q = (float *)take(B * H * kHeadDim * sizeof(float));
    o.part_o = (float *)take(B * H * kMaxSplits * kHeadDim * sizeof(float));
    o.part_ml = (float2 *)take(B * H * kMaxSplits * sizeof(float2));
    o.act = (float *)take(B * F * sizeof(float));
    o.logits = (float *)take(B * V * sizeof(float));
    o.hidden = (float *)take((c->flags & HQ_FLAG_CAPTURE_HIDDEN) ? L * B * d * sizeof(float) : 0);
    o.prompt = (int *)take(B * T * sizeof(int));
    const size_t R = pass_rows(c), qdim = H * kHeadDim, qkvd = (H + 2 * Hkv) * kHeadDim;
    o.pf_tok = (int *)take(R * sizeof(int));
    o.last_idx = (int *)take(B * sizeof(int));
    o.xs = (float *)take(R * d * sizeof(float));
    o.delta = (float *)take(kPrefillSplits * R * d * sizeof(float));
    o.hn = (act_t *)take(2 * R * d * sizeof(act_t));
    o.qkv = (float *)take(kPrefillSplits * R * qkvd * sizeof(float));
    o.q16 = (__half *)take(R * qdim * sizeof(__half));
    o.ao = (act_t *)take(2 * R * qdim * sizeof(act_t));
    o.actb = (act_t *)take(2 * R * F * sizeof(act_t));
    o.hn_last = (act_t *)take(2 * 32 * d * sizeof(act_t));
    o.err = (int *)take(sizeof(int));
    const bool verify = (c->flags & HQ_FLAG_VERIFY) != 0;
    o.verify_logits = (float *)take(verify ? (size_t)kVerifyRows * V * sizeof(float) : 0);
    o.verify_best = (unsigned long long *)take(verify ? kVerifyRows * sizeof(unsigned long long) : 0);
    o.verify_out = (int *)take(sizeof(int));
    o.ab_ll = (unsigned long long *)take((size_t)H * kHeadDim * sizeof(unsigned long long));
    o.ab_epoch = (unsigned int *)take(sizeof(unsigned int));
    return off;
}

extern "C" size_t hq_workspace_bytes(const hq_config *cfg) {
    const char *why = "";
    if (!config_ok(cfg, &why)) {
        fail(HQ_ERR_INVALID_ARG, "hq_workspace_bytes: %s", why);
        return 0;
    }
    return carve(cfg, nullptr, nullptr);
}

// ---- one decode step: A1..A9 ------------------------------------------------------------------------
// tok_src: device pointer to the token fed at this step.  with_head = false skips A9 and advances
// the position with a one-thread kernel instead (used while walking a prompt token by token).
static AttnBlockParams attn_block_params(const hq_model *m, int l) {
    const hq_config &c = m->cfg;
    const Buffers &b = m->b;
    const LayerW &w = m->layers[l];
    const size_t layer_kv = (size_t)c.max_batch * c.n_kv_heads * c.max_seq * kHeadDim;
    AttnBlockParams a = {};
    a.wq = w.wq; a.wk = w.wk; a.wv = w.wv; a.wo = w.wo; a.gain = w.attn_norm;
    a.x = b.x; a.kc = b.kcache + l * layer_kv; a.vc = b.vcache + l * layer_kv; a.rope = b.rope; a.pos = b.pos;
    a.ll_attn = b.ab_ll; a.epoch = b.ab_epoch; a.err = b.err;
    a.hidden = c.hidden; a.n_heads = c.n_heads; a.n_kv_heads = c.n_kv_heads; a.max_seq = c.max_seq; a.eps = c.rms_eps;
    a.trace = m->trace; a.trace_cap = m->trace_cap;
    a.step_trace = m->step_trace; a.step_slot = 1 + 3 * l;
    return a;
}

// Stages (64 KB) by which a gate/up CTA that was resident during the attention block is ahead of one that starts on an SM
// the block has just left: two of its three ring stages (measured optimum 2-4, flat; 0 costs 1.5 % of the step).
constexpr float kLateDeficit = 2.0f;

static SgemvParams sgemv_gateup(const hq_model *m, int l) {
    const hq_config &c = m->cfg;
    const LayerW &w = m->layers[l];
    SgemvParams p = {};
    p.w0 = w.w_gate; p.w1 = w.w_up; p.gain = w.ffn_norm; p.xin = m->b.x; p.K = c.hidden; p.n_rows = c.ffn;
    p.mode = SGEMV_GATEUP; p.xin_mode = SGEMV_XIN_NORM; p.eps = c.rms_eps;
    p.trace = m->step_trace; p.trace_slot = 2 + 3 * l;
    if (m->use_attn_block) { p.n_early = m->n_sms - kAbCluster * c.n_kv_heads; p.late_deficit = kLateDeficit; }
    p.out_planes = reinterpret_cast<bf16 *>(m->b.act);
    if (m->q4) { p.q0 = m->layers_q4[l].gate_q; p.e0 = m->layers_q4[l].gate_e; p.q1 = m->layers_q4[l].up_q; p.e1 = m->layers_q4[l].up_e; }
    return p;
}
static SgemvParams sgemv_down(const hq_model *m, int l) {
    const hq_config &c = m->cfg;
    SgemvParams p = {};
    p.w0 = m->layers[l].w_down; p.xin = m->b.act; p.K = c.ffn; p.n_rows = c.hidden;
    p.trace = m->step_trace; p.trace_slot = 3 + 3 * l;
    p.mode = SGEMV_RESID; p.xin_mode = SGEMV_XIN_PLANES; p.out = m->b.x;
    if (m->q4) { p.q0 = m->layers_q4[l].down_q; p.e0 = m->layers_q4[l].down_e; }
    // Three quarters of the SMs stream the down projection as fast as all of them (HBM is the limit from ~64 streaming SMs
    // on, profiles/r02_copy_size.md); the others are free for the clusters of the next layer's attention block, which become
    // resident — barriers, cluster sync, first weight stages — under this kernel instead of after it (measured: 104-124 CTAs
    // all -2 % of the step, 84 and 128-148 none)
    // (bf16 only: the hq4 kernel is bound by expanding nibbles, not by HBM, and wants every SM: 0.431 -> 0.424 ms per token)
    if (m->use_attn_block && !m->q4) p.max_ctas = (m->n_sms * 3) / 4;
    return p;
}
// final norm + LM head + argmax over the residual row x; the position advances by pos_inc
static SgemvParams sgemv_lm_head(const hq_model *m, const float *x, int pos_inc) {
    const hq_config &c = m->cfg;
    const Buffers &b = m->b;
    SgemvParams p = {};
    p.w0 = m->lm_head; p.gain = m->final_norm; p.xin = x; p.K = c.hidden; p.n_rows = c.vocab;
    p.mode = SGEMV_LMHEAD; p.xin_mode = SGEMV_XIN_NORM; p.eps = c.rms_eps; p.out = b.logits;
    p.pos = b.pos; p.best = b.best; p.counter = b.counter; p.cur_tok = b.cur_tok; p.tok_hist = b.tok_hist;
    p.trace = m->step_trace; p.trace_slot = 1 + 3 * c.n_layers;
    p.pos_rw = b.pos; p.pos_inc = pos_inc;
    if (m->q4) { p.q0 = m->lm_head_q; p.e0 = m->lm_head_e; }
    return p;
}

static cudaError_t enqueue_step(hq_model *m, const int *tok_src, bool with_head, int *n_launched) {
    const hq_config &c = m->cfg;
    const LaunchCtx lc{m->stream, m->use_pdl, m->n_sms};
    const Buffers &b = m->b;
    const int qdim = c.n_heads * kHeadDim;
    const size_t layer_kv = (size_t)c.max_batch * c.n_kv_heads * c.max_seq * kHeadDim;
    cudaError_t e;
    int n = 0;
#define STEP(call) do { e = (call); if (e != cudaSuccess) return e; ++n; } while (0)
    STEP(launch_embed(lc, m->emb, tok_src, b.x, c.hidden, 1));
    for (int l = 0; l < c.n_layers; ++l) {
        const LayerW &w = m->layers[l];
        GemvParams p = {};
        if (m->use_attn_block) {
            // A2-A6 of the layer in ONE cluster launch (hq_attn.cu)
            STEP(launch_attn_block(lc, attn_block_params(m, l)));
        } else {
        // A2+A3+A4: RMSNorm -> QKV GEMV -> RoPE + KV append
        p.w0 = w.wq; p.w1 = w.wk; p.w2 = w.wv; p.gain = w.attn_norm; p.xin = b.x; p.K = c.hidden;
        p.n_units = (c.n_heads + 2 * c.n_kv_heads) * 32; p.eps = c.rms_eps; p.out = b.q;
        p.kc = b.kcache + l * layer_kv; p.vc = b.vcache + l * layer_kv; p.rope = b.rope; p.pos = b.pos;
        p.n_heads = c.n_heads; p.n_kv_heads = c.n_kv_heads; p.max_seq = c.max_seq;
        STEP(launch_gemv(lc, GEMV_QKV, XIN_NORM, p));
        // A5: split-KV flash-decode
        AttnDecodeParams a = {b.q, p.kc, p.vc, b.part_o, b.part_ml, b.pos, c.n_heads, c.n_kv_heads, c.max_seq};
        STEP(launch_attn_decode(lc, a, 1));
        // A6: merge splits -> O GEMV -> residual
        GemvParams po = {};
        po.w0 = w.wo; po.xin = b.part_o; po.part_ml = b.part_ml; po.K = qdim; po.n_units = c.hidden / 2;
        po.out = b.x; po.pos = b.pos;
        STEP(launch_gemv(lc, GEMV_RESID, XIN_ATTN, po));
        }
        // A2+A7: RMSNorm -> gate/up GEMV -> SwiGLU (bf16 hi/lo planes of the vector); A8: down GEMV -> residual
        STEP(launch_sgemv(lc, sgemv_gateup(m, l)));
        STEP(launch_sgemv(lc, sgemv_down(m, l)));
        if (c.flags & HQ_FLAG_CAPTURE_HIDDEN) {
            e = cudaMemcpyAsync(b.hidden + (size_t)l * c.max_batch * c.hidden, b.x, c.hidden * sizeof(float),
                                cudaMemcpyDeviceToDevice, m->stream);
            if (e != cudaSuccess) return e;
        }
    }
    if (with_head) {
        // A9: final norm -> LM head GEMV -> logits + argmax + step bookkeeping
        STEP(launch_sgemv(lc, sgemv_lm_head(m, b.x, 1)));
    } else {
        STEP(launch_advance(lc, b.pos, 1));
    }
#undef STEP
    if (n_launched) *n_launched = n;
    return cudaSuccess;
}

static cudaError_t capture_step_graph(hq_model *m) {
    cudaError_t e = cudaStreamBeginCapture(m->stream, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) return e;
    int n = 0;
    cudaError_t e_step = enqueue_step(m, m->b.cur_tok, true, &n);
    cudaGraph_t g = nullptr;
    e = cudaStreamEndCapture(m->stream, &g);
    if (e_step != cudaSuccess) { if (g) cudaGraphDestroy(g); return e_step; }
    if (e != cudaSuccess) return e;
    e = cudaGraphInstantiate(&m->step_graph, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) { m->step_graph = nullptr; return e; }
    m->kernels_per_step = n;
    return cudaSuccess;
}

// ---- row-batched (tensor-core) path: envelope prefill passes and batched decode steps ---------------
static int tile_index(int rows) { return rows <= 32 ? 0 : rows <= 64 ? 1 : rows <= 128 ? 2 : 3; }

// Tile plan of one GEMM of a pass: token tile (index into kTokenTiles) and split-K factor.
// Fill the SMs with (weight tile x token tile) CTAs first: a token tile of 64 still feeds the tensor core at full
// rate (the 128-row weight tile is re-read from shared memory every 32 cycles), the weight tile's second reader hits
// L2, and no atomics are needed.  Split K (fp32 atomics into the output) only when the grid is still under half the
// SMs — 9-way split-K cost more in atomics than it gained (profiles/r01_launches_v2.md).  Prefill passes stay bit-
// reproducible: at most 2 splits into a zeroed buffer (0 + a + b is order-independent), none into the residual
// (x + a + b is not).  Batched decode steps (few rows, weight-stream bound) split as far as the SMs go.
struct TilePlan { int ti, NT, splits; };
static TilePlan plan_gemm(const hq_model *m, int n_rows, int rows, int K, int max_splits) {
    const int n_tiles = (n_rows + 127) / 128;
    if (rows > 32 && max_splits > 1) {
        // Prefill pass with split-K partial buffers (no atomics).  Pick the (token tile, splits) with the least modelled time:
        // the slower of a per-CTA tile stream (times the number of waves) and a chip-wide one.  A heuristic fitted to
        // measured launches: the main loops themselves run at the tensor-core rate (profiles/r02_launches.md), what the
        // model really ranks is CTA count (waves) against K blocks per CTA and partial buffers to write.
        const int kb = (K + 63) / 64;
        TilePlan best{1, 64, 1};
        double best_t = 1e30;
        for (int ti = 1; ti <= 3; ++ti) {
            const int NT = kTokenTiles[ti];
            if (ti > 1 && NT > ((rows + 63) / 64) * 64) continue;   // no tile wider than the pass (rounded to 64)
            const int t_tiles = (rows + NT - 1) / NT;
            for (int sp = 1; sp <= max_splits; sp *= 2) {
                if (sp > 1 && kb / sp < 8) break;
                const double ctas = (double)n_tiles * t_tiles * sp, waves = ceil(ctas / m->n_sms);
                // tile bytes per K block: the weight tile + the token tile's planes (CTA pairs, token tile <= 128: one plane each)
                const double per_cta = (double)((kb + sp - 1) / sp) * (16384.0 + (NT <= 128 ? 1.0 : 2.0) * NT * 128.0);
                const double t = fmax(waves * per_cta / (NT == 256 ? 40e9 : 65e9), ctas * per_cta / 8.5e12) + 2e-6 * (sp - 1) / 4;
                if (t < best_t) { best_t = t; best = TilePlan{ti, NT, sp}; }
            }
        }
        return best;
    }
    const int ti_max = tile_index(rows);
    int ti = ti_max;
    while (ti > 1 && n_tiles * ((rows + kTokenTiles[ti] - 1) / kTokenTiles[ti]) < (m->n_sms * 3) / 4) --ti;
    TilePlan p{ti, kTokenTiles[ti], 1};
    if (max_splits > 1) {
        const int tiles = n_tiles * ((rows + p.NT - 1) / p.NT);
        const int kb = (K + 63) / 64;
        int s = m->n_sms / (tiles > 0 ? tiles : 1);
        // few token rows (batched decode): the weight stream is the bound, the atomics are few -> as many CTAs as SMs;
        // many rows (prefill): at least 16 K blocks per split and at most 4 splits
        const int min_kb = rows <= 32 ? 4 : 16;
        if (s > kb / min_kb) s = kb / min_kb;
        if (s > max_splits) s = max_splits;
        p.splits = s < 1 ? 1 : s;
    }
    return p;
}

// Batched decode steps of <= 16 sequences: token tiles of 8 / 16 rows instead of 32.  The main loop of these GEMMs pays
// for every shared-memory byte (profiles/r02_batched_decode.md, item 10): a 32-row tile that is 3/4 padding is 8 KB of TMA
// writes and 8 KB of operand reads per 16 KB of weights, an 8-row tile 2 KB of each.
static void small_token_tile(TilePlan &p, int rows) {
    if (rows <= 8) { p.ti = 4; p.NT = 8; }
    else if (rows <= 16) { p.ti = 5; p.NT = 16; }
}

// All layers for `rows` = batch * Tc token rows already embedded in b.xs; positions start at *b.pos.
// decode = true: Tc == 1, attention over the cache with the split-KV decode kernel.
static cudaError_t enqueue_rows_layers(hq_model *m, int batch, int Tc, bool decode, bool capture_hidden, int *n_launched) {
    const hq_config &c = m->cfg;
    const LaunchCtx lc{m->stream, m->use_pdl, m->n_sms};
    const Buffers &b = m->b;
    const int rows = batch * Tc;
    const int d = c.hidden, qdim = c.n_heads * kHeadDim, kvdim = c.n_kv_heads * kHeadDim, qkvd = qdim + 2 * kvdim;
    const size_t layer_kv = (size_t)c.max_batch * c.n_kv_heads * c.max_seq * kHeadDim;
    const int R = m->pf_rows;                                  // lo plane sits R rows below the hi plane
    const size_t lo_d = (size_t)R * d, lo_q = (size_t)R * qdim, lo_f = (size_t)R * c.ffn;
    cudaError_t e;
    int n = 0;
#define STEP(call) do { e = (call); if (e != cudaSuccess) return e; ++n; } while (0)
    // Prefill passes defer the residual adds of the O and down projections (bit-reproducible split-K, see
    // rmsnorm_rows_kernel); decode steps add atomically into the residual.
    const bool defer = !decode;
    // split-K partials of the O / down projection not yet added to xs (prefill passes): buffers R * d floats apart
    const size_t d_stride = (size_t)R * d, q_stride = (size_t)R * qkvd;
    int pending = 0;
    for (int l = 0; l < c.n_layers; ++l) {
        const LayerW &w = m->layers[l];
        const LayerMaps &mp = m->maps[l];
        kv_t *kc = b.kcache + l * layer_kv, *vc = b.vcache + l * layer_kv;
        // P1: Q, K, V projections (three weight pointers, no repack) into one fp32 [rows][qkvd] buffer
        const bool stacked = qdim % 128 == 0 && kvdim % 128 == 0;
        const int split_store = decode ? 16 : kPrefillSplits, split_resid = decode ? 16 : kPrefillSplits;
        TilePlan pq = plan_gemm(m, stacked ? qkvd : qdim, rows, d, split_store);
        if (decode) small_token_tile(pq, rows);
        const size_t qs = defer ? q_stride : 0;   // prefill: one partial buffer per split; batched decode: atomics into a zeroed buffer
        // batched decode: the norm kernel clears the rows the split-K projections add into (no memset node between the two)
        const bool zero_qkv = pq.splits > 1 && !defer;
        if (zero_qkv && qkvd % 4 != 0) {
            e = cudaMemsetAsync(b.qkv, 0, (size_t)rows * qkvd * sizeof(float), m->stream);
            if (e != cudaSuccess) return e;
        }
        STEP(launch_rmsnorm_rows(lc, b.xs, b.delta, pending, d_stride, w.attn_norm, b.hn, lo_d, d, c.rms_eps, rows, nullptr, d,
                                 zero_qkv && qkvd % 4 == 0 ? b.qkv : nullptr, qkvd));
        pending = 0;
        if (stacked) {
            STEP(launch_gemm_qkv(lc, mp.wq, mp.wk, mp.wv, m->map_hn[pq.ti], R, qdim, kvdim, kvdim, d, rows, pq.NT, pq.splits, b.qkv, qkvd, qs));
        } else {
            STEP(launch_gemm(lc, EPI_STORE, mp.wq, nullptr, m->map_hn[pq.ti], R, qdim, d, rows, pq.NT, pq.splits, b.qkv, nullptr, 0, qkvd, qs));
            STEP(launch_gemm(lc, EPI_STORE, mp.wk, nullptr, m->map_hn[pq.ti], R, kvdim, d, rows, pq.NT, pq.splits, b.qkv + qdim, nullptr, 0, qkvd, qs));
            STEP(launch_gemm(lc, EPI_STORE, mp.wv, nullptr, m->map_hn[pq.ti], R, kvdim, d, rows, pq.NT, pq.splits, b.qkv + qdim + kvdim, nullptr, 0, qkvd, qs));
        }
        if (decode) {
            // P4 + B2 in one launch: RoPE, KV append, split-KV decode attention per sequence, split merge
            AttnFusedParams a = {b.qkv, kc, vc, b.rope, b.part_o, b.part_ml, b.attn_tickets, b.ao, lo_q, b.pos, c.n_heads, c.n_kv_heads, c.max_seq};
            STEP(launch_attn_decode_fused(lc, a, batch));
        } else {
            // P4: RoPE + KV append (adds the split-K partials of the projection in order)
            STEP(launch_rope_append(lc, b.qkv, pq.splits, q_stride, b.q16, nullptr, kc, vc, b.rope, b.pos, rows, Tc,
                                    c.n_heads, c.n_kv_heads, c.max_seq));
            // P2: causal flash attention
            STEP(launch_flash_prefill(lc, b.q16, kc, vc, b.ao, lo_q, b.pos, batch, Tc, c.n_heads, c.n_kv_heads, c.max_seq));
        }
        TilePlan po = plan_gemm(m, d, rows, qdim, split_resid);
        if (decode) small_token_tile(po, rows);
        STEP(launch_gemm(lc, defer ? EPI_STORE : EPI_RESID, mp.wo, nullptr, m->map_ao[po.ti], R, d, qdim, rows, po.NT, po.splits,
                         defer ? b.delta : b.xs, nullptr, 0, d, defer ? d_stride : 0));
        if (defer) pending = po.splits;
        STEP(launch_rmsnorm_rows(lc, b.xs, b.delta, pending, d_stride, w.ffn_norm, b.hn, lo_d, d, c.rms_eps, rows, nullptr, d));
        pending = 0;
        TilePlan pg = plan_gemm(m, c.ffn, rows, d, 1);
        // batched decode (one token tile): 64-row weight tiles, so that ffn / 64 CTAs stream gate/up instead of ffn / 128
        const bool half_tiles = decode && c.ffn % 64 == 0 && (c.ffn / 128) * ((rows + pg.NT - 1) / pg.NT) < m->n_sms;
        if (half_tiles) small_token_tile(pg, rows);   // (the two-accumulator form keeps 32-row tiles)
        STEP(launch_gemm(lc, half_tiles ? EPI_SWIGLU64 : EPI_SWIGLU, half_tiles ? mp.w_gate64 : mp.w_gate, half_tiles ? &mp.w_up64 : &mp.w_up,
                         m->map_hn[pg.ti], R, c.ffn, d, rows, pg.NT, 1, nullptr, b.actb, lo_f, c.ffn));
        TilePlan pd = plan_gemm(m, d, rows, c.ffn, split_resid);
        if (decode) small_token_tile(pd, rows);
        STEP(launch_gemm(lc, defer ? EPI_STORE : EPI_RESID, mp.w_down, nullptr, m->map_actb[pd.ti], R, d, c.ffn, rows, pd.NT, pd.splits,
                         defer ? b.delta : b.xs, nullptr, 0, d, defer ? d_stride : 0));
        if (defer) pending = pd.splits;
        if (defer && capture_hidden) {
            STEP(launch_add_delta_rows(lc, b.xs, b.delta, pending, d_stride, (size_t)rows * d));
            pending = 0;
        }
        if (capture_hidden) {
            // residual of the last position of every sequence -> hidden[l][b]
            e = cudaMemcpy2DAsync(b.hidden + (size_t)l * c.max_batch * d, d * sizeof(float),
                                  b.xs + (size_t)(Tc - 1) * d, (size_t)Tc * d * sizeof(float), d * sizeof(float), batch,
                                  cudaMemcpyDeviceToDevice, m->stream);
            if (e != cudaSuccess) return e;
        }
    }
#undef STEP
    m->delta_pending = pending;   // consumed by the head / verification pass that follows
    if (n_launched) *n_launched += n;
    return cudaSuccess;
}

// LM head for the last row of every sequence: final norm -> GEMM (weights read once for all
// sequences) -> fp32 logits [batch][vocab] -> argmax + step bookkeeping (pos += pos_inc).
static cudaError_t enqueue_rows_head(hq_model *m, int batch, int Tc, int pos_inc, bool deferred, int *n_launched) {
    const hq_config &c = m->cfg;
    const LaunchCtx lc{m->stream, m->use_pdl, m->n_sms};
    const Buffers &b = m->b;
    cudaError_t e;
    int n = 0;
#define STEP(call) do { e = (call); if (e != cudaSuccess) return e; ++n; } while (0)
    if (batch == 1) {
        // one sequence: the batch-1 LM-head GEMV (A9: final norm, 6.4 TB/s weight stream, fused argmax and bookkeeping) on the
        // last row of the pass instead of norm + 32-token-tile GEMM + argmax (116 + 10 us -> 85 us)
        float *xl = b.xs + (size_t)(Tc - 1) * c.hidden;
        if (deferred && m->delta_pending) STEP(launch_add_delta_rows(lc, xl, b.delta + (size_t)(Tc - 1) * c.hidden, m->delta_pending, (size_t)m->pf_rows * c.hidden, (size_t)c.hidden));
        STEP(launch_sgemv(lc, sgemv_lm_head(m, xl, pos_inc)));
        if (n_launched) *n_launched += n;
        return cudaSuccess;
    }
    // rows (Tc-1), (2Tc-1), ... : stride Tc rows starting at row Tc-1
    STEP(launch_rmsnorm_rows(lc, b.xs + (size_t)(Tc - 1) * c.hidden, b.delta + (size_t)(Tc - 1) * c.hidden, deferred ? m->delta_pending : 0,
                             (size_t)m->pf_rows * c.hidden, m->final_norm, b.hn_last, (size_t)32 * c.hidden, c.hidden, c.rms_eps, batch, nullptr,
                             Tc * c.hidden));
    TilePlan ph{0, 32, 1};
    small_token_tile(ph, batch);
    STEP(launch_gemm(lc, EPI_STORE, m->map_lm_head, nullptr, m->map_hn_last[ph.ti], 32, c.vocab, c.hidden, batch, ph.NT, 1, b.logits,
                     nullptr, 0, c.vocab));
    STEP(launch_argmax_rows(lc, b.logits, c.vocab, batch, b.cur_tok, b.tok_hist, b.pos, pos_inc, b.counter, b.best));
#undef STEP
    if (n_launched) *n_launched += n;
    return cudaSuccess;
}

// one batched decode step (B1 + B2): embed -> layers -> head
static cudaError_t enqueue_batch_step(hq_model *m, int batch, int *n_launched) {
    const LaunchCtx lc{m->stream, m->use_pdl, m->n_sms};
    int n = 0;
    cudaError_t e = launch_embed_rows(lc, m->emb, m->b.cur_tok, m->b.xs, m->cfg.hidden, batch);
    if (e != cudaSuccess) return e;
    ++n;
    e = enqueue_rows_layers(m, batch, 1, true, (m->cfg.flags & HQ_FLAG_CAPTURE_HIDDEN) != 0, &n);
    if (e != cudaSuccess) return e;
    e = enqueue_rows_head(m, batch, 1, 1, false, &n);
    if (e != cudaSuccess) return e;
    if (n_launched) *n_launched = n;
    return cudaSuccess;
}

static cudaError_t capture_batch_graph(hq_model *m, int batch) {
    if (m->batch_graph) { cudaGraphExecDestroy(m->batch_graph); m->batch_graph = nullptr; m->batch_graph_b = 0; }
    cudaError_t e = cudaStreamBeginCapture(m->stream, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) return e;
    int n = 0;
    cudaError_t e_step = enqueue_batch_step(m, batch, &n);
    cudaGraph_t g = nullptr;
    e = cudaStreamEndCapture(m->stream, &g);
    if (e_step != cudaSuccess) { if (g) cudaGraphDestroy(g); return e_step; }
    if (e != cudaSuccess) return e;
    e = cudaGraphInstantiate(&m->batch_graph, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) { m->batch_graph = nullptr; return e; }
    m->batch_graph_b = batch;
    m->batch_graph_kernels = n;
    return cudaSuccess;
}

static bool build_tensor_maps(hq_model *m) {
    const hq_config &c = m->cfg;
    const Buffers &b = m->b;
    const uint64_t d = c.hidden, qdim = (uint64_t)c.n_heads * kHeadDim, kvdim = (uint64_t)c.n_kv_heads * kHeadDim, F = c.ffn;
    m->maps.resize(c.n_layers);
    bool ok = true;
    for (int l = 0; l < c.n_layers; ++l) {
        const LayerW &w = m->layers[l];
        LayerMaps &mp = m->maps[l];
        ok = ok && make_tensor_map_16b(&mp.wq, w.wq, qdim, d, 128) && make_tensor_map_16b(&mp.wk, w.wk, kvdim, d, 128) &&
             make_tensor_map_16b(&mp.wv, w.wv, kvdim, d, 128) && make_tensor_map_16b(&mp.wo, w.wo, d, qdim, 128) &&
             make_tensor_map_16b(&mp.w_gate, w.w_gate, F, d, 128) && make_tensor_map_16b(&mp.w_up, w.w_up, F, d, 128) &&
             make_tensor_map_16b(&mp.w_down, w.w_down, d, F, 128) && make_tensor_map_16b(&mp.w_gate64, w.w_gate, F, d, 64) &&
             make_tensor_map_16b(&mp.w_up64, w.w_up, F, d, 64);
    }
    ok = ok && make_tensor_map_16b(&m->map_lm_head, m->lm_head, c.vocab, d, 128);
    for (int i = 0; i < 6; ++i) {
        const uint32_t nt = kTokenTiles[i];
        ok = ok && make_tensor_map_16b(&m->map_hn[i], b.hn, 2 * (uint64_t)m->pf_rows, d, nt) &&
             make_tensor_map_16b(&m->map_ao[i], b.ao, 2 * (uint64_t)m->pf_rows, qdim, nt) &&
             make_tensor_map_16b(&m->map_actb[i], b.actb, 2 * (uint64_t)m->pf_rows, F, nt);
    }
    for (int i : {0, 4, 5}) ok = ok && make_tensor_map_16b(&m->map_hn_last[i], b.hn_last, 64, d, kTokenTiles[i]);
    return ok;
}

// ---- create / destroy ---------------------------------------------------------------------------------
static int32_t model_create(const hq_config *cfg, const hq_weights *w, const hq_weights_q4 *q, void *workspace, size_t ws_bytes,
                            void *cuda_stream, hq_model **out);

extern "C" int32_t hq_model_create(const hq_config *cfg, const hq_weights *w, void *workspace, size_t ws_bytes,
                                   void *cuda_stream, hq_model **out) {
    if (cfg && cfg->weight_dtype == HQ_Q4) return fail(HQ_ERR_INVALID_ARG, "hq_model_create: HQ_Q4 models are created with hq_model_create_q4");
    return model_create(cfg, w, nullptr, workspace, ws_bytes, cuda_stream, out);
}

extern "C" int32_t hq_model_create_q4(const hq_config *cfg, const hq_weights *w, const hq_weights_q4 *q, void *workspace,
                                      size_t ws_bytes, void *cuda_stream, hq_model **out) {
    if (!cfg || cfg->weight_dtype != HQ_Q4 || !q) return fail(HQ_ERR_INVALID_ARG, "hq_model_create_q4: needs weight_dtype HQ_Q4 and the hq4 tensors");
    if (!q->w_gate_codes || !q->w_gate_exps || !q->w_up_codes || !q->w_up_exps || !q->w_down_codes || !q->w_down_exps ||
        !q->lm_head_codes || !q->lm_head_exps)
        return fail(HQ_ERR_INVALID_ARG, "hq_model_create_q4: an hq4 pointer is NULL");
    for (int l = 0; l < cfg->n_layers; ++l)
        if (!q->w_gate_codes[l] || !q->w_gate_exps[l] || !q->w_up_codes[l] || !q->w_up_exps[l] || !q->w_down_codes[l] || !q->w_down_exps[l])
            return fail(HQ_ERR_INVALID_ARG, "hq_model_create_q4: an hq4 pointer of layer %d is NULL", l);
    if (!sgemv_q4_shape_supported(cfg->hidden) || !sgemv_q4_shape_supported(cfg->ffn) || cfg->hidden % 64 != 0 || cfg->ffn % 16 != 0 ||
        cfg->hidden % 16 != 0 || cfg->vocab % 16 != 0 || cfg->hidden > 2048)
        return fail(HQ_ERR_UNSUPPORTED, "hq_model_create_q4: hq4 needs hidden a multiple of 64 and <= 2048, ffn a multiple of 32 (of 1024 above 2048), "
                                        "vocab a multiple of 16");
    return model_create(cfg, w, q, workspace, ws_bytes, cuda_stream, out);
}

extern "C" int32_t hq_quantize_q4(void *cuda_stream, const void *w_dev, int64_t n_rows, int32_t k, void *codes_dev, void *exps_dev) {
    if (!w_dev || !codes_dev || !exps_dev || n_rows <= 0 || k <= 0 || k % 32 != 0) return fail(HQ_ERR_INVALID_ARG, "hq_quantize_q4: bad argument (k must be a multiple of 32)");
    HQ_CUDA(launch_q4_quantize((cudaStream_t)cuda_stream, (const bf16 *)w_dev, (size_t)n_rows, k, (uint8_t *)codes_dev, (uint8_t *)exps_dev));
    return HQ_OK;
}

extern "C" int32_t hq_dequantize_q4(void *cuda_stream, const void *codes_dev, const void *exps_dev, int64_t n_rows, int32_t k, void *w_dev) {
    if (!w_dev || !codes_dev || !exps_dev || n_rows <= 0 || k <= 0 || k % 32 != 0) return fail(HQ_ERR_INVALID_ARG, "hq_dequantize_q4: bad argument (k must be a multiple of 32)");
    HQ_CUDA(launch_q4_dequantize((cudaStream_t)cuda_stream, (const uint8_t *)codes_dev, (const uint8_t *)exps_dev, (size_t)n_rows, k, (bf16 *)w_dev));
    return HQ_OK;
}

static int32_t model_create(const hq_config *cfg, const hq_weights *w, const hq_weights_q4 *q, void *workspace, size_t ws_bytes,
                            void *cuda_stream, hq_model **out) {
    const char *why = "";
    if (!out) return fail(HQ_ERR_INVALID_ARG, "hq_model_create: out is NULL");
    *out = nullptr;
    if (!config_ok(cfg, &why)) return fail(HQ_ERR_INVALID_ARG, "hq_model_create: %s", why);
    if (!config_supported(cfg, &why)) return fail(HQ_ERR_UNSUPPORTED, "hq_model_create: %s", why);
    if (!w || !workspace) return fail(HQ_ERR_INVALID_ARG, "hq_model_create: weights or workspace is NULL");
    if (!w->tok_embedding || !w->final_norm || !w->lm_head || !w->attn_norm || !w->wq || !w->wk || !w->wv ||
        !w->wo || !w->ffn_norm || !w->w_gate || !w->w_up || !w->w_down)
        return fail(HQ_ERR_INVALID_ARG, "hq_model_create: a weight pointer is NULL");
    for (int l = 0; l < cfg->n_layers; ++l)
        if (!w->attn_norm[l] || !w->wq[l] || !w->wk[l] || !w->wv[l] || !w->wo[l] || !w->ffn_norm[l] ||
            !w->w_gate[l] || !w->w_up[l] || !w->w_down[l])
            return fail(HQ_ERR_INVALID_ARG, "hq_model_create: a weight pointer of layer %d is NULL", l);
    if (((uintptr_t)workspace & 255) != 0) return fail(HQ_ERR_INVALID_ARG, "hq_model_create: workspace not 256-byte aligned");
    const size_t need = carve(cfg, nullptr, nullptr);
    if (ws_bytes < need)
        return fail(HQ_ERR_CAPACITY, "hq_model_create: workspace %zu bytes < %zu needed", ws_bytes, need);

    int dev = 0;
    HQ_CUDA(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    HQ_CUDA(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10)
        return fail(HQ_ERR_UNSUPPORTED, "hq_model_create: needs compute capability 10.x (sm_100a), found %d.%d",
                    prop.major, prop.minor);

    HQ_CUDA(gemm_prepare());
    HQ_CUDA(sgemv_prepare());
    HQ_CUDA(sgemv_q4_prepare());
    hq_model *m = new (std::nothrow) hq_model();
    if (!m) return fail(HQ_ERR_INVALID_ARG, "hq_model_create: out of host memory");
    m->cfg = *cfg;
    m->device = dev;
    m->stream = (cudaStream_t)cuda_stream;
    m->n_sms = prop.multiProcessorCount;
    m->emb = (const bf16 *)w->tok_embedding;
    m->final_norm = (const bf16 *)w->final_norm;
    m->lm_head = (const bf16 *)w->lm_head;
    m->layers.resize(cfg->n_layers);
    for (int l = 0; l < cfg->n_layers; ++l) {
        LayerW &lw = m->layers[l];
        lw.attn_norm = (const bf16 *)w->attn_norm[l]; lw.wq = (const bf16 *)w->wq[l];
        lw.wk = (const bf16 *)w->wk[l]; lw.wv = (const bf16 *)w->wv[l]; lw.wo = (const bf16 *)w->wo[l];
        lw.ffn_norm = (const bf16 *)w->ffn_norm[l]; lw.w_gate = (const bf16 *)w->w_gate[l];
        lw.w_up = (const bf16 *)w->w_up[l]; lw.w_down = (const bf16 *)w->w_down[l];
    }
    if (q) {
        m->q4 = true;
        m->layers_q4.resize(cfg->n_layers);
        for (int l = 0; l < cfg->n_layers; ++l)
            m->layers_q4[l] = LayerQ4{(const uint8_t *)q->w_gate_codes[l], (const uint8_t *)q->w_gate_exps[l], (const uint8_t *)q->w_up_codes[l],
                                      (const uint8_t *)q->w_up_exps[l], (const uint8_t *)q->w_down_codes[l], (const uint8_t *)q->w_down_exps[l]};
        m->lm_head_q = (const uint8_t *)q->lm_head_codes;
        m->lm_head_e = (const uint8_t *)q->lm_head_exps;
    }
    carve(cfg, (char *)workspace, &m->b);
    m->pf_rows = (int)pass_rows(cfg);
    if (!build_tensor_maps(m)) {
        delete m;
        return fail(HQ_ERR_CUDA, "hq_model_create: cuTensorMapEncodeTiled failed (driver entry point or bad alignment)");
    }
    m->use_pdl = !(cfg->flags & HQ_FLAG_NO_PDL);
    m->use_attn_block = !(cfg->flags & HQ_FLAG_KERNEL_PER_ROW) && attn_block_shape_supported(*cfg);
    if (m->use_attn_block) {
        // the clusters of one launch wait for one another's attention vector: all of them must be resident at once
        // (cudaOccupancyMaxActiveClusters); otherwise batch-1 decode takes the kernel-per-row path
        bool co_resident = false;
        cudaError_t e = attn_block_prepare(cfg->n_kv_heads, &co_resident);
        if (e != cudaSuccess) { cudaGetLastError(); co_resident = false; }
        m->use_attn_block = co_resident;
    }
    {
        // tagged exchange words start with tag 0 (never a valid epoch); the epoch counter only ever grows
        const unsigned int one = 1u;
        cudaError_t e = cudaMemsetAsync(m->b.ab_ll, 0, (size_t)cfg->n_heads * kHeadDim * sizeof(unsigned long long), m->stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(m->b.ab_epoch, &one, sizeof(one), cudaMemcpyHostToDevice, m->stream);
        if (e == cudaSuccess && (cfg->flags & HQ_FLAG_VERIFY))
            e = cudaMemsetAsync(m->b.verify_best, 0, kVerifyRows * sizeof(unsigned long long), m->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(m->stream);
        if (e != cudaSuccess) {
            delete m;
            return fail(HQ_ERR_CUDA, "hq_model_create: exchange buffer init failed: %s", cudaGetErrorString(e));
        }
    }

    // RoPE table in double on the host (reading 7): angle = pos * theta^(-2i/64)
    {
        std::vector<float2> tab((size_t)cfg->max_seq * 32);
        for (int p = 0; p < cfg->max_seq; ++p)
            for (int i = 0; i < 32; ++i) {
                const double phi = (double)p * pow((double)cfg->rope_theta, -2.0 * i / (double)kHeadDim);
                tab[(size_t)p * 32 + i] = make_float2((float)cos(phi), (float)sin(phi));
            }
        cudaError_t e = cudaMemcpyAsync(m->b.rope, tab.data(), tab.size() * sizeof(float2), cudaMemcpyHostToDevice, m->stream);
        if (e == cudaSuccess) e = launch_set_state(LaunchCtx{m->stream, false, m->n_sms}, m->b.pos, 0, m->b.best,
                                                   m->b.counter, cfg->max_batch, m->b.err);
        if (e == cudaSuccess) e = launch_zero_tokens(LaunchCtx{m->stream, false, m->n_sms}, m->b.cur_tok, cfg->max_batch);
        if (e == cudaSuccess) e = cudaMemsetAsync(m->b.attn_tickets, 0, (size_t)cfg->max_batch * cfg->n_kv_heads * sizeof(unsigned int), m->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(m->stream);
        if (e != cudaSuccess) {
            delete m;
            return fail(HQ_ERR_CUDA, "hq_model_create: state init failed: %s", cudaGetErrorString(e));
        }
    }

    // A stream capture cannot start on the legacy default stream: without a real stream the decode
    // step is launched kernel by kernel.
    if (!(cfg->flags & HQ_FLAG_NO_GRAPH) && m->stream != nullptr) {
        // One eager step first so that every kernel is loaded before the capture (lazy module
        // loading is not allowed while capturing); its side effects are reset right after.
        cudaError_t e = enqueue_step(m, m->b.cur_tok, true, nullptr);
        if (e == cudaSuccess) e = launch_set_state(LaunchCtx{m->stream, false, m->n_sms}, m->b.pos, 0, m->b.best,
                                                   m->b.counter, cfg->max_batch, m->b.err);
        if (e == cudaSuccess) e = cudaStreamSynchronize(m->stream);
        if (e == cudaSuccess) e = capture_step_graph(m);
        if (e != cudaSuccess && m->use_pdl) {  // retry without programmatic edges
            cudaGetLastError();
            m->use_pdl = false;
            e = capture_step_graph(m);
        }
        if (e != cudaSuccess) {
            cudaGetLastError();
            delete m;
            return fail(HQ_ERR_CUDA, "hq_model_create: graph capture failed: %s", cudaGetErrorString(e));
        }
    }
    *out = m;
    return HQ_OK;
}

extern "C" void hq_model_destroy(hq_model *m) {
    if (!m) return;
    if (m->step_graph) cudaGraphExecDestroy(m->step_graph);
    if (m->batch_graph) cudaGraphExecDestroy(m->batch_graph);
    delete m;
}

// ---- state --------------------------------------------------------------------------------------------
extern "C" int32_t hq_sync(hq_model *m) {
    if (!m) return fail(HQ_ERR_INVALID_ARG, "hq_sync: model is NULL");
    HQ_ON_DEVICE(m);
    cudaError_t e = cudaStreamSynchronize(m->stream);
    if (e != cudaSuccess)
        return fail(HQ_ERR_CUDA, "hq_sync: %s (a trapped attention-block launch means a cluster arrival or a tagged word never came: "
                    "the device was not exclusive to this model, see hq_model_create)", cudaGetErrorString(e));
    return HQ_OK;
}

extern "C" int32_t hq_seq_len(const hq_model *m, int32_t *out) {
    if (!m || !out) return fail(HQ_ERR_INVALID_ARG, "hq_seq_len: NULL argument");
    *out = m->seq_len;
    return HQ_OK;
}

extern "C" int32_t hq_kv_reset(hq_model *m) {
    if (!m) return fail(HQ_ERR_INVALID_ARG, "hq_kv_reset: model is NULL");
    HQ_ON_DEVICE(m);
    HQ_CUDA(launch_set_state(LaunchCtx{m->stream, false, m->n_sms}, m->b.pos, 0, m->b.best, m->b.counter,
                             m->cfg.max_batch, m->b.err));
    // the split tickets of the batched decode attention are zero between launches unless a launch was cut short (HQ_ERR_CUDA)
    HQ_CUDA(cudaMemsetAsync(m->b.attn_tickets, 0, (size_t)m->cfg.max_batch * m->cfg.n_kv_heads * sizeof(unsigned int), m->stream));
    m->kernel_count += 1;
    m->seq_len = 0;
    m->batch = 0;
    m->have_token = false;
    return HQ_OK;
}

extern "C" int64_t hq_kernel_count(const hq_model *m) { return m ? m->kernel_count : 0; }

extern "C" const char *hq_decode_path(const hq_model *m) {
    if (!m) return "";
    if (m->use_attn_block) return "attention-block-cluster";
    return "kernel-per-row";
}

// ---- prefill -----------------------------------------------------------------------------------------
extern "C" int32_t hq_prefill(hq_model *m, const int32_t *tokens_host, int32_t batch, int32_t n_tokens,
                              float *logits_dev, int32_t *first_token_host) {
    if (!m || !tokens_host) return fail(HQ_ERR_INVALID_ARG, "hq_prefill: NULL argument");
    HQ_ON_DEVICE(m);
    if (batch <= 0 || n_tokens <= 0) return fail(HQ_ERR_INVALID_ARG, "hq_prefill: batch and n_tokens must be > 0");
    const hq_config &c = m->cfg;
    if (batch > c.max_batch) return fail(HQ_ERR_CAPACITY, "hq_prefill: batch %d > max_batch %d", batch, c.max_batch);
    if (m->batch != 0 && batch != m->batch)
        return fail(HQ_ERR_STATE, "hq_prefill: active batch is %d, got %d (hq_kv_reset first)", m->batch, batch);
    if ((long long)m->seq_len + n_tokens > c.max_seq)
        return fail(HQ_ERR_CAPACITY, "hq_prefill: seq_len %d + %d tokens > max_seq %d", m->seq_len, n_tokens, c.max_seq);
    for (long long i = 0; i < (long long)batch * n_tokens; ++i)
        if (tokens_host[i] < 0 || tokens_host[i] >= c.vocab)
            return fail(HQ_ERR_INVALID_ARG, "hq_prefill: token %d at index %lld outside [0, %d)", tokens_host[i], i, c.vocab);
    const LaunchCtx lc{m->stream, m->use_pdl, m->n_sms};
    const bool capture = (c.flags & HQ_FLAG_CAPTURE_HIDDEN) != 0;
    if (batch == 1 && n_tokens < 8) {
        // very short appends: walk the tokens with the batch-1 decode kernels
        HQ_CUDA(cudaMemcpyAsync(m->b.prompt, tokens_host, (size_t)n_tokens * sizeof(int), cudaMemcpyHostToDevice, m->stream));
        for (int t = 0; t < n_tokens; ++t) {
            int n = 0;
            HQ_CUDA(enqueue_step(m, m->b.prompt + t, t == n_tokens - 1, &n));
            m->kernel_count += n;
        }
    } else {
        // tensor-core passes of at most pf_rows token rows (all sequences together)
        const int tc_max = m->pf_rows / batch;
        for (int t0 = 0; t0 < n_tokens; t0 += tc_max) {
            const int Tc = n_tokens - t0 < tc_max ? n_tokens - t0 : tc_max;
            const bool last = t0 + Tc == n_tokens;
            // rows m = b * Tc + t  <-  tokens_host[b][t0 + t]
            HQ_CUDA(cudaMemcpy2DAsync(m->b.pf_tok, (size_t)Tc * sizeof(int), tokens_host + t0, (size_t)n_tokens * sizeof(int),
                                      (size_t)Tc * sizeof(int), batch, cudaMemcpyHostToDevice, m->stream));
            int n = 0;
            HQ_CUDA(launch_embed_rows(lc, m->emb, m->b.pf_tok, m->b.xs, c.hidden, batch * Tc));
            ++n;
            HQ_CUDA(enqueue_rows_layers(m, batch, Tc, false, capture && last, &n));
            HQ_CUDA(launch_advance(lc, m->b.pos, Tc));
            ++n;
            if (last) HQ_CUDA(enqueue_rows_head(m, batch, Tc, 0, true, &n));
            m->kernel_count += n;
        }
    }
    m->batch = batch;
    m->seq_len += n_tokens;
    m->have_token = true;
    if (logits_dev)
        HQ_CUDA(cudaMemcpyAsync(logits_dev, m->b.logits, (size_t)batch * c.vocab * sizeof(float),
                                cudaMemcpyDeviceToDevice, m->stream));
    if (first_token_host) {
        HQ_CUDA(cudaMemcpyAsync(first_token_host, m->b.cur_tok, batch * sizeof(int), cudaMemcpyDeviceToHost, m->stream));
        HQ_CUDA(cudaStreamSynchronize(m->stream));
    }
    return HQ_OK;
}

// ---- verbatim-relay verification in one dense pass -------------------------------------------
extern "C" int32_t hq_verify_relay(hq_model *m, const int32_t *tokens_host, int32_t n_envelope, int32_t n_answer,
                                   int32_t *n_accepted_host) {
    if (!m || !tokens_host || !n_accepted_host) return fail(HQ_ERR_INVALID_ARG, "hq_verify_relay: NULL argument");
    HQ_ON_DEVICE(m);
    const hq_config &c = m->cfg;
    if (!(c.flags & HQ_FLAG_VERIFY)) return fail(HQ_ERR_STATE, "hq_verify_relay: model created without HQ_FLAG_VERIFY");
    if (n_envelope <= 0 || n_answer <= 0) return fail(HQ_ERR_INVALID_ARG, "hq_verify_relay: n_envelope and n_answer must be > 0");
    if (m->batch > 1) return fail(HQ_ERR_STATE, "hq_verify_relay: one sequence only (active batch is %d)", m->batch);
    const int T = n_envelope + n_answer, nv = n_answer + 1;
    if (nv > kVerifyRows) return fail(HQ_ERR_CAPACITY, "hq_verify_relay: n_answer %d > %d", n_answer, kVerifyRows - 1);
    if (T > m->pf_rows) return fail(HQ_ERR_CAPACITY, "hq_verify_relay: %d tokens > %d rows of one pass", T, m->pf_rows);
    if ((long long)m->seq_len + T > c.max_seq)
        return fail(HQ_ERR_CAPACITY, "hq_verify_relay: seq_len %d + %d tokens > max_seq %d", m->seq_len, T, c.max_seq);
    for (int i = 0; i < T; ++i)
        if (tokens_host[i] < 0 || tokens_host[i] >= c.vocab)
            return fail(HQ_ERR_INVALID_ARG, "hq_verify_relay: token %d at index %d outside [0, %d)", tokens_host[i], i, c.vocab);
    const LaunchCtx lc{m->stream, m->use_pdl, m->n_sms};
    const Buffers &b = m->b;
    const int d = c.hidden;
    // one tensor-core pass over envelope + answer (the cache rows of the answer are written speculatively: rows beyond the
    // accepted prefix are simply never read, the position decides what is cached)
    HQ_CUDA(cudaMemcpyAsync(b.pf_tok, tokens_host, (size_t)T * sizeof(int), cudaMemcpyHostToDevice, m->stream));
    int n = 0;
    HQ_CUDA(launch_embed_rows(lc, m->emb, b.pf_tok, b.xs, d, T));
    ++n;
    HQ_CUDA(enqueue_rows_layers(m, 1, T, false, false, &n));
    // LM head at the n_answer + 1 positions n_envelope - 1 .. T - 1: final norm (folds the deferred residual of the last
    // layer in) -> one GEMM over the vocabulary (weights read once per 256-token tile) -> per-row argmax against the answer
    const int r0 = n_envelope - 1;
    HQ_CUDA(launch_rmsnorm_rows(lc, b.xs + (size_t)r0 * d, b.delta + (size_t)r0 * d, m->delta_pending, (size_t)m->pf_rows * d, m->final_norm, b.hn,
                                (size_t)m->pf_rows * d, d, c.rms_eps, nv, nullptr, d));
    const TilePlan pv = plan_gemm(m, c.vocab, nv, d, 1);
    HQ_CUDA(launch_gemm(lc, EPI_STORE, m->map_lm_head, nullptr, m->map_hn[pv.ti], m->pf_rows, c.vocab, d, nv, pv.NT, 1,
                        b.verify_logits, nullptr, 0, c.vocab));
    HQ_CUDA(launch_verify_rows(lc, b.verify_logits, c.vocab, nv, b.pf_tok + n_envelope, n_envelope, b.cur_tok, b.tok_hist, b.pos,
                               b.counter, b.verify_best, b.verify_out));
    m->kernel_count += n + 3;
    int accepted = 0;
    HQ_CUDA(cudaMemcpyAsync(&accepted, b.verify_out, sizeof(int), cudaMemcpyDeviceToHost, m->stream));
    HQ_CUDA(cudaStreamSynchronize(m->stream));
    // hq_decode_logits: the logits that chose the token now waiting to be fed
    HQ_CUDA(cudaMemcpyAsync(b.logits, b.verify_logits + (size_t)accepted * c.vocab, (size_t)c.vocab * sizeof(float),
                            cudaMemcpyDeviceToDevice, m->stream));
    m->batch = 1;
    m->seq_len += n_envelope + accepted;
    m->have_token = true;
    *n_accepted_host = accepted;
    return HQ_OK;
}

// ---- decode ------------------------------------------------------------------------------------------
static int32_t decode_precheck(hq_model *m, const char *who, int n_steps) {
    if (!m) return fail(HQ_ERR_INVALID_ARG, "%s: model is NULL", who);
    HQ_ON_DEVICE(m);
    if (m->batch == 0) return fail(HQ_ERR_STATE, "%s: no active sequence (call hq_prefill first)", who);
    if ((long long)m->seq_len + n_steps > m->cfg.max_seq)
        return fail(HQ_ERR_CAPACITY, "%s: seq_len %d + %d > max_seq %d", who, m->seq_len, n_steps, m->cfg.max_seq);
    return HQ_OK;
}

static int32_t launch_one_step(hq_model *m) {
    if (m->batch > 1) {
        // batched decode (B1/B2): tensor-core GEMMs, weights read once per step for all sequences.
        // The first step of a batch size runs eagerly (loads every kernel), the second captures a graph.
        const bool want_graph = !(m->cfg.flags & HQ_FLAG_NO_GRAPH) && m->stream != nullptr;
        if (want_graph && m->batch_graph_b != m->batch && m->batch_eager_b == m->batch) {
            cudaError_t e = capture_batch_graph(m, m->batch);
            if (e != cudaSuccess) { cudaGetLastError(); m->batch_eager_b = -1; }   // stay eager
        }
        if (m->batch_graph && m->batch_graph_b == m->batch) {
            HQ_CUDA(cudaGraphLaunch(m->batch_graph, m->stream));
            m->kernel_count += m->batch_graph_kernels;
        } else {
            int n = 0;
            HQ_CUDA(enqueue_batch_step(m, m->batch, &n));
            m->kernel_count += n;
            if (m->batch_eager_b != -1) m->batch_eager_b = m->batch;
        }
    } else if (m->step_graph) {
        HQ_CUDA(cudaGraphLaunch(m->step_graph, m->stream));
        m->kernel_count += m->kernels_per_step;
    } else {
        int n = 0;
        HQ_CUDA(enqueue_step(m, m->b.cur_tok, true, &n));
        m->kernel_count += n;
    }
    m->seq_len += 1;
    return HQ_OK;
}

extern "C" int32_t hq_decode_step(hq_model *m, const int32_t *tokens_in_host, int32_t *tokens_out_host) {
    int32_t rc = decode_precheck(m, "hq_decode_step", 1);
    if (rc != HQ_OK) return rc;
    if (tokens_in_host) {
        for (int b = 0; b < m->batch; ++b)
            if (tokens_in_host[b] < 0 || tokens_in_host[b] >= m->cfg.vocab)
                return fail(HQ_ERR_INVALID_ARG, "hq_decode_step: token %d outside [0, %d)", tokens_in_host[b], m->cfg.vocab);
        HQ_CUDA(cudaMemcpyAsync(m->b.cur_tok, tokens_in_host, m->batch * sizeof(int), cudaMemcpyHostToDevice, m->stream));
    } else if (!m->have_token) {
        return fail(HQ_ERR_STATE, "hq_decode_step: no device-resident token to feed");
    }
    rc = launch_one_step(m);
    if (rc != HQ_OK) return rc;
    m->have_token = true;
    if (tokens_out_host) {
        HQ_CUDA(cudaMemcpyAsync(tokens_out_host, m->b.cur_tok, m->batch * sizeof(int), cudaMemcpyDeviceToHost, m->stream));
        HQ_CUDA(cudaStreamSynchronize(m->stream));
    }
    return HQ_OK;
}

extern "C" int32_t hq_decode_run(hq_model *m, int32_t n_steps, int32_t *tokens_out_host) {
    if (n_steps <= 0) return fail(HQ_ERR_INVALID_ARG, "hq_decode_run: n_steps must be > 0");
    int32_t rc = decode_precheck(m, "hq_decode_run", n_steps);
    if (rc != HQ_OK) return rc;
    if (!m->have_token) return fail(HQ_ERR_STATE, "hq_decode_run: no device-resident token to feed");
    const int first = m->seq_len + 1;
    for (int i = 0; i < n_steps; ++i) {
        rc = launch_one_step(m);
        if (rc != HQ_OK) return rc;
    }
    if (tokens_out_host) {
        HQ_CUDA(cudaMemcpyAsync(tokens_out_host, m->b.tok_hist + (size_t)first * m->batch,
                                (size_t)n_steps * m->batch * sizeof(int), cudaMemcpyDeviceToHost, m->stream));
        HQ_CUDA(cudaStreamSynchronize(m->stream));
    }
    return HQ_OK;
}

extern "C" int32_t hq_decode_logits(hq_model *m, float *logits_dev) {
    if (!m || !logits_dev) return fail(HQ_ERR_INVALID_ARG, "hq_decode_logits: NULL argument");
    HQ_ON_DEVICE(m);
    if (m->batch == 0) return fail(HQ_ERR_STATE, "hq_decode_logits: nothing has been evaluated yet");
    HQ_CUDA(cudaMemcpyAsync(logits_dev, m->b.logits, (size_t)m->batch * m->cfg.vocab * sizeof(float),
                            cudaMemcpyDeviceToDevice, m->stream));
    return HQ_OK;
}

extern "C" int32_t hq_get_hidden(hq_model *m, int32_t layer, float *hidden_dev) {
    if (!m || !hidden_dev) return fail(HQ_ERR_INVALID_ARG, "hq_get_hidden: NULL argument");
    HQ_ON_DEVICE(m);
    if (!(m->cfg.flags & HQ_FLAG_CAPTURE_HIDDEN)) return fail(HQ_ERR_STATE, "hq_get_hidden: model created without HQ_FLAG_CAPTURE_HIDDEN");
    if (layer < 0 || layer >= m->cfg.n_layers) return fail(HQ_ERR_INVALID_ARG, "hq_get_hidden: layer %d outside [0, %d)", layer, m->cfg.n_layers);
    if (m->batch == 0) return fail(HQ_ERR_STATE, "hq_get_hidden: nothing has been evaluated yet");
    HQ_CUDA(cudaMemcpyAsync(hidden_dev, m->b.hidden + (size_t)layer * m->cfg.max_batch * m->cfg.hidden,
                            (size_t)m->batch * m->cfg.hidden * sizeof(float), cudaMemcpyDeviceToDevice, m->stream));
    return HQ_OK;
}

// ---- measurement hook ---------------------------------------------------------------------------------
extern "C" int32_t hq_bench_kernel(hq_model *m, int32_t which, int32_t reps, int64_t *bytes_per_launch) {
    if (!m || reps <= 0) return fail(HQ_ERR_INVALID_ARG, "hq_bench_kernel: bad argument");
    HQ_ON_DEVICE(m);
    if (m->batch == 0 || m->seq_len == 0) return fail(HQ_ERR_STATE, "hq_bench_kernel: needs a prefilled cache");
    if (m->seq_len >= m->cfg.max_seq) return fail(HQ_ERR_CAPACITY, "hq_bench_kernel: cache is full");
    const hq_config &c = m->cfg;
    const LaunchCtx lc{m->stream, m->use_pdl, m->n_sms};
    const Buffers &b = m->b;
    const size_t layer_kv = (size_t)c.max_batch * c.n_kv_heads * c.max_seq * kHeadDim;
    const int qdim = c.n_heads * kHeadDim;
    int64_t bytes = 0;
    for (int r = 0; r < reps; ++r) {
        const int l = r % c.n_layers;
        const LayerW &w = m->layers[l];
        GemvParams p = {};
        switch (which) {
            case 0: {
                SgemvParams pg = sgemv_gateup(m, l);
                pg.n_early = 0;   // timed alone there is no attention block in front of it: even split
                HQ_CUDA(launch_sgemv(lc, pg));
                bytes = m->q4 ? 2ll * c.ffn * (c.hidden / 2 + c.hidden / 32) : 2ll * 2 * c.ffn * c.hidden;
                break;
            }
            case 1: {
                // LM head without state side effects: pos_inc = 0 (token / history writes repeat the current slot)
                HQ_CUDA(launch_sgemv(lc, sgemv_lm_head(m, b.x, 0)));
                bytes = m->q4 ? 1ll * c.vocab * (c.hidden / 2 + c.hidden / 32) : 2ll * c.vocab * c.hidden;
                break;
            }
            case 2:
                // QKV: rewrites the K/V row at the current position with garbage from the scratch x
                p.w0 = w.wq; p.w1 = w.wk; p.w2 = w.wv; p.gain = w.attn_norm; p.xin = b.x; p.K = c.hidden;
                p.n_units = (c.n_heads + 2 * c.n_kv_heads) * 32; p.eps = c.rms_eps; p.out = b.q;
                p.kc = b.kcache + l * layer_kv; p.vc = b.vcache + l * layer_kv; p.rope = b.rope; p.pos = b.pos;
                p.n_heads = c.n_heads; p.n_kv_heads = c.n_kv_heads; p.max_seq = c.max_seq;
                HQ_CUDA(launch_gemv(lc, GEMV_QKV, XIN_NORM, p));
                bytes = 2ll * (c.n_heads + 2 * c.n_kv_heads) * kHeadDim * c.hidden;
                break;
            case 3:
                p.w0 = w.wo; p.xin = b.part_o; p.part_ml = b.part_ml; p.K = qdim; p.n_units = c.hidden / 2;
                p.out = b.x; p.pos = b.pos;
                HQ_CUDA(launch_gemv(lc, GEMV_RESID, XIN_ATTN, p));
                bytes = 2ll * c.hidden * qdim;
                break;
            case 4:
                HQ_CUDA(launch_sgemv(lc, sgemv_down(m, l)));
                bytes = m->q4 ? 1ll * c.hidden * (c.ffn / 2 + c.ffn / 32) : 2ll * c.hidden * c.ffn;
                break;
            case 5: {
                AttnDecodeParams a = {b.q, b.kcache + l * layer_kv, b.vcache + l * layer_kv, b.part_o, b.part_ml,
                                      b.pos, c.n_heads, c.n_kv_heads, c.max_seq};
                HQ_CUDA(launch_attn_decode(lc, a, 1));
                bytes = 2ll * 2 * c.n_kv_heads * kHeadDim * (m->seq_len + 1);
                break;
            }
            case 6: {
                // attention block: QKV + attention + O of layer l in one launch (rewrites the K/V row at the current position)
                if (!m->use_attn_block) return fail(HQ_ERR_UNSUPPORTED, "hq_bench_kernel: this model does not run the attention block");
                HQ_CUDA(launch_attn_block(lc, attn_block_params(m, l)));
                bytes = 2ll * ((c.n_heads + 2 * c.n_kv_heads) * kHeadDim + c.hidden) * c.hidden +
                        2ll * 2 * c.n_kv_heads * kHeadDim * (m->seq_len + 1);
                break;
            }
            default:
                return fail(HQ_ERR_INVALID_ARG, "hq_bench_kernel: unknown kernel %d", which);
        }
        m->kernel_count += 1;
    }
    if (bytes_per_launch) *bytes_per_launch = bytes;
    return HQ_OK;
}

extern "C" int32_t hq_debug_read_probe(void *cuda_stream, const void *src_dev, size_t bytes, uint32_t *sum_dev) {
    if (!src_dev || !sum_dev || bytes < 16 || ((uintptr_t)src_dev & 15) != 0)
        return fail(HQ_ERR_INVALID_ARG, "hq_debug_read_probe: needs a 16-byte aligned buffer of >= 16 bytes and a result word");
    int dev = 0, n_sms = 0;
    HQ_CUDA(cudaGetDevice(&dev));
    HQ_CUDA(cudaDeviceGetAttribute(&n_sms, cudaDevAttrMultiProcessorCount, dev));
    HQ_CUDA(launch_read_probe((cudaStream_t)cuda_stream, src_dev, bytes, sum_dev, n_sms));
    return HQ_OK;
}

extern "C" int32_t hq_debug_copy_probe(void *cuda_stream, const void *src_dev, size_t bytes, int32_t copy_bytes, int32_t n_ctas) {
    if (!src_dev || ((uintptr_t)src_dev & 127) != 0 || n_ctas <= 0 || copy_bytes < 16 || copy_bytes > 65536 || (copy_bytes & (copy_bytes - 1)) != 0 ||
        bytes / 65536 / (size_t)n_ctas == 0)
        return fail(HQ_ERR_INVALID_ARG, "hq_debug_copy_probe: needs a 128-byte aligned buffer of >= 64 KB per CTA and a power-of-two copy size in [16, 65536]");
    HQ_CUDA(launch_copy_probe((cudaStream_t)cuda_stream, src_dev, bytes, copy_bytes, n_ctas));
    return HQ_OK;
}

extern "C" int32_t hq_debug_kv_row(hq_model *m, int32_t which, int32_t layer, int32_t seq, int32_t pos, void *row_dev) {
    if (!m || !row_dev) return fail(HQ_ERR_INVALID_ARG, "hq_debug_kv_row: NULL argument");
    HQ_ON_DEVICE(m);
    const hq_config &c = m->cfg;
    if ((which != 0 && which != 1) || layer < 0 || layer >= c.n_layers || seq < 0 || seq >= c.max_batch || pos < 0 || pos >= c.max_seq)
        return fail(HQ_ERR_INVALID_ARG, "hq_debug_kv_row: index out of range");
    const kv_t *base = (which == 0 ? m->b.kcache : m->b.vcache) +
                       (((size_t)layer * c.max_batch + seq) * c.n_kv_heads * c.max_seq + pos) * kHeadDim;
    // [n_kv_heads] rows of 64 elements, max_seq * 64 elements apart -> contiguous [n_kv_heads][64]
    HQ_CUDA(cudaMemcpy2DAsync(row_dev, kHeadDim * sizeof(kv_t), base, (size_t)c.max_seq * kHeadDim * sizeof(kv_t),
                              kHeadDim * sizeof(kv_t), c.n_kv_heads, cudaMemcpyDeviceToDevice, m->stream));
    return HQ_OK;
}

extern "C" int32_t hq_debug_step_trace(hq_model *m, uint64_t *trace_dev, int32_t n_slots) {
    if (!m) return fail(HQ_ERR_INVALID_ARG, "hq_debug_step_trace: model is NULL");
    if (trace_dev && n_slots < 2 + 3 * m->cfg.n_layers)
        return fail(HQ_ERR_INVALID_ARG, "hq_debug_step_trace: needs %d slots", 2 + 3 * m->cfg.n_layers);
    m->step_trace = (unsigned long long *)trace_dev;
    m->step_trace_slots = trace_dev ? n_slots : 0;
    return HQ_OK;
}

extern "C" int32_t hq_debug_trace(hq_model *m, uint64_t *trace_dev, int32_t cap) {
    if (!m || cap < 0 || (trace_dev && cap == 0)) return fail(HQ_ERR_INVALID_ARG, "hq_debug_trace: bad argument");
    m->trace = (unsigned long long *)trace_dev;
    m->trace_cap = trace_dev ? cap : 0;
    return HQ_OK;
}

// ---- diagnostics: the tensor-core GEMM on its own ------------------------------------------------------
static int32_t debug_gemm_impl(void *cuda_stream, int32_t mode, const void *w_dev, const void *w2_dev, const void *x_dev, void *out_dev,
                               int32_t n_rows, int32_t k, int32_t n_tokens, int32_t token_tile, int32_t splits, uint64_t *trace_dev) {
    if (!w_dev || !x_dev || !out_dev || n_rows <= 0 || k <= 0 || n_tokens <= 0)
        return fail(HQ_ERR_INVALID_ARG, "hq_debug_gemm: bad argument");
    if (mode < 0 || mode > 3 || (mode >= 2 && !w2_dev)) return fail(HQ_ERR_INVALID_ARG, "hq_debug_gemm: bad mode");
    if (mode == 3 && n_rows % 64 != 0) return fail(HQ_ERR_UNSUPPORTED, "hq_debug_gemm: mode 3 needs n_rows % 64 == 0");
    if (token_tile != 32 && token_tile != 64 && token_tile != 128 && token_tile != 256 && !((token_tile == 8 || token_tile == 16) && mode != 2))
        return fail(HQ_ERR_INVALID_ARG, "hq_debug_gemm: token_tile must be 32, 64, 128 or 256 (8 or 16 too, except in mode 2)");
    if (k % 8 != 0) return fail(HQ_ERR_UNSUPPORTED, "hq_debug_gemm: k must be a multiple of 8");
    TensorMap mw, mw2, mx;
    // x_dev holds the hi plane [n_tokens][k] followed by the lo plane [n_tokens][k]
    const uint32_t wbox = mode == 3 ? 64 : 128;
    if (!make_tensor_map_16b(&mw, w_dev, n_rows, k, wbox) || !make_tensor_map_16b(&mx, x_dev, 2 * (uint64_t)n_tokens, k, token_tile) ||
        (mode >= 2 && !make_tensor_map_16b(&mw2, w2_dev, n_rows, k, wbox)))
        return fail(HQ_ERR_CUDA, "hq_debug_gemm: cuTensorMapEncodeTiled failed");
    const LaunchCtx lc{(cudaStream_t)cuda_stream, false, 148};
    HQ_CUDA(gemm_prepare());
    HQ_CUDA(launch_gemm(lc, (GemmEpilogue)mode, mw, mode >= 2 ? &mw2 : nullptr, mx, n_tokens, n_rows, k, n_tokens, token_tile,
                        mode >= 2 ? 1 : splits, mode >= 2 ? nullptr : (float *)out_dev, mode >= 2 ? (act_t *)out_dev : nullptr,
                        (size_t)n_tokens * n_rows, n_rows, 0, (unsigned long long *)trace_dev));
    return HQ_OK;
}

extern "C" int32_t hq_debug_gemm(void *cuda_stream, int32_t mode, const void *w_dev, const void *w2_dev, const void *x_dev, void *out_dev,
                                 int32_t n_rows, int32_t k, int32_t n_tokens, int32_t token_tile, int32_t splits) {
    return debug_gemm_impl(cuda_stream, mode, w_dev, w2_dev, x_dev, out_dev, n_rows, k, n_tokens, token_tile, splits, nullptr);
}

extern "C" int32_t hq_debug_gemm_timeline(void *cuda_stream, int32_t mode, const void *w_dev, const void *w2_dev, const void *x_dev,
                                          void *out_dev, int32_t n_rows, int32_t k, int32_t n_tokens, int32_t token_tile, int32_t splits,
                                          uint64_t *trace_dev) {
    if (!trace_dev) return fail(HQ_ERR_INVALID_ARG, "hq_debug_gemm_timeline: trace_dev is NULL");
    return debug_gemm_impl(cuda_stream, mode, w_dev, w2_dev, x_dev, out_dev, n_rows, k, n_tokens, token_tile, splits, trace_dev);
}
