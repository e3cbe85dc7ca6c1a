/*
 * hq_oracle — TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, obviously-correct CPU forward of the Llama-style decoder whose prefill + streaming
 * decode is the hot path of arxiv/paper_2606_12154 ("A 1B-class model ... then
 * streams the answer"; "one prompt evaluation", "decode rate", "TTFT").
 * The paper discloses no equations, so the computation is the plain
 * definition fixed by BASELINE.json `configs` and written out in SURVEY.md §8(c); every function
 * below cites the step of that algorithm it implements.  DESIGN.md "Readings" lists every point
 * on which the paper is silent and the reading taken.
 *
 * Precision: weights are fp32 values (the exact values of the bf16-rounded tensors the GPU sees,
 * or the raw fp32 draw for self-checks); EVERYTHING else — activations, residual, norms, RoPE
 * angles, softmax, KV cache, accumulators — is double (BASELINE.json north_star "plain, slow fp32
 * CPU transformer forward"; this is stricter).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this file.  It shares no code with paper_2606_12154_b200/csrc.  OpenMP is used only to
 * spread independent output elements over cores; there is no blocking, fusion or reordering.
 *
 * Pins (tests/test_oracle_pins.py): RoPE closed forms, softmax rows sum to 1, context-1 attention,
 * brute-force attention, GQA == MHA on repeated K/V, RMSNorm closed forms, SiLU values,
 * incremental == full-sequence forward, causality, W_o = W_d = 0 special case, FFN/head
 * permutation symmetry, and an independent float64 torch re-expression of configs[0].
 * Parity against numbers printed by the paper: UNPINNED — the paper prints no value this path
 * must reproduce (weights and data undisclosed); see DESIGN.md.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t n_layers, hidden, n_heads, n_kv_heads, head_dim, ffn, vocab;
    int32_t max_seq;
    double rms_eps, rope_theta;
} hqo_config;

typedef struct {
    const float *tok_embedding;              /* [vocab, hidden]                          */
    const float *const *attn_norm;           /* n_layers x [hidden]                      */
    const float *const *wq, *const *wk, *const *wv, *const *wo; /* [out, in] row-major    */
    const float *const *ffn_norm;
    const float *const *w_gate, *const *w_up, *const *w_down;
    const float *final_norm;                 /* [hidden]                                 */
    const float *lm_head;                    /* [vocab, hidden]; == tok_embedding if tied */
} hqo_weights;

typedef struct {
    hqo_config c;
    hqo_weights w;
    const float **ptrs;  /* owned copy of the 9 per-layer pointer arrays */
    double *kcache;      /* [n_layers][max_seq][n_kv_heads*head_dim], unrounded (reading 18) */
    double *vcache;
    int32_t seq_len;
} hqo_model;

int hqo_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- step 2a / 2g / 3: RMSNorm, eps inside the sqrt (reading 10) -------------------------- */
void hqo_rmsnorm(const double *x, const float *g, int32_t d, double eps, double *out) {
    double ss = 0.0;
    for (int32_t i = 0; i < d; ++i) ss += x[i] * x[i];
    double inv = 1.0 / sqrt(ss / (double)d + eps);
    for (int32_t i = 0; i < d; ++i) out[i] = x[i] * inv * (double)g[i];
}

/* ---- step 2b / 2f / 2g / 3: y = W x, W is [n_out, n_in] row-major, no bias ------------------ */
static inline double dot_fd(const float *w, const double *x, int32_t n) {
    double acc = 0.0;
#pragma omp simd reduction(+ : acc)
    for (int32_t k = 0; k < n; ++k) acc += (double)w[k] * x[k];
    return acc;
}

/* Y[t][o] = <W[o], X[t]> for t < T */
void hqo_matmul(const float *W, const double *X, int32_t T, int32_t n_out, int32_t n_in, double *Y) {
#pragma omp parallel for schedule(static)
    for (int32_t o = 0; o < n_out; ++o) {
        const float *wrow = W + (size_t)o * n_in;
        for (int32_t t = 0; t < T; ++t)
            Y[(size_t)t * n_out + o] = dot_fd(wrow, X + (size_t)t * n_in, n_in);
    }
}

/* ---- step 2c: RoPE on one head, rotate-half pairing (i, i+hd/2), angle p * theta^(-2i/hd) ---- */
void hqo_rope(double *v, int32_t head_dim, int32_t pos, double theta) {
    int32_t half = head_dim / 2;
    for (int32_t i = 0; i < half; ++i) {
        double phi = (double)pos * pow(theta, -2.0 * (double)i / (double)head_dim);
        double c = cos(phi), s = sin(phi);
        double a = v[i], b = v[i + half];
        v[i] = a * c - b * s;
        v[i + half] = b * c + a * s;
    }
}

/* ---- step 2g: silu(z) = z / (1 + exp(-z)) (reading 11) -------------------------------------- */
double hqo_silu(double z) { return z / (1.0 + exp(-z)); }

/* ---- step 2e: one query head against n_ctx cached positions ---------------------------------
 * s_r = <q, K[r]> / sqrt(hd); P = softmax(s) with max subtraction; o = sum_r P_r V[r].
 * K, V: row r at K + r*stride.  probs (optional) receives P. */
void hqo_attend(const double *q, const double *K, const double *V, int32_t n_ctx, int32_t stride,
                int32_t head_dim, double *o, double *probs) {
    double *s = (double *)malloc(sizeof(double) * (size_t)n_ctx);
    double scale = 1.0 / sqrt((double)head_dim);
    double m = -INFINITY;
    for (int32_t r = 0; r < n_ctx; ++r) {
        double acc = 0.0;
        for (int32_t i = 0; i < head_dim; ++i) acc += q[i] * K[(size_t)r * stride + i];
        s[r] = acc * scale;
        if (s[r] > m) m = s[r];
    }
    double l = 0.0;
    for (int32_t r = 0; r < n_ctx; ++r) { s[r] = exp(s[r] - m); l += s[r]; }
    for (int32_t r = 0; r < n_ctx; ++r) s[r] /= l;
    for (int32_t i = 0; i < head_dim; ++i) o[i] = 0.0;
    for (int32_t r = 0; r < n_ctx; ++r)
        for (int32_t i = 0; i < head_dim; ++i) o[i] += s[r] * V[(size_t)r * stride + i];
    if (probs) memcpy(probs, s, sizeof(double) * (size_t)n_ctx);
    free(s);
}

/* ---- step 3: greedy argmax, lowest index wins ties (reading 13) ----------------------------- */
int32_t hqo_argmax(const double *v, int32_t n) {
    int32_t best = 0;
    for (int32_t i = 1; i < n; ++i) if (v[i] > v[best]) best = i;
    return best;
}

/* top-2 margin (largest minus second largest), used by the teacher-forced argmax rule */
double hqo_top2_margin(const double *v, int32_t n) {
    double a = -INFINITY, b = -INFINITY;
    for (int32_t i = 0; i < n; ++i) {
        if (v[i] > a) { b = a; a = v[i]; }
        else if (v[i] > b) b = v[i];
    }
    return a - b;
}

/* ---- model object ---------------------------------------------------------------------------- */
hqo_model *hqo_create(const hqo_config *c, const hqo_weights *w) {
    if (c->n_heads % c->n_kv_heads != 0 || c->head_dim % 2 != 0) return NULL;
    hqo_model *m = (hqo_model *)calloc(1, sizeof(hqo_model));
    m->c = *c;
    m->w = *w;
    int L = c->n_layers;
    m->ptrs = (const float **)malloc(sizeof(float *) * 9 * (size_t)L);
    const float *const *src[9] = {w->attn_norm, w->wq, w->wk, w->wv, w->wo,
                                  w->ffn_norm, w->w_gate, w->w_up, w->w_down};
    for (int j = 0; j < 9; ++j)
        for (int l = 0; l < L; ++l) m->ptrs[j * L + l] = src[j][l];
    m->w.attn_norm = m->ptrs + 0 * L; m->w.wq = m->ptrs + 1 * L; m->w.wk = m->ptrs + 2 * L;
    m->w.wv = m->ptrs + 3 * L;        m->w.wo = m->ptrs + 4 * L; m->w.ffn_norm = m->ptrs + 5 * L;
    m->w.w_gate = m->ptrs + 6 * L;    m->w.w_up = m->ptrs + 7 * L; m->w.w_down = m->ptrs + 8 * L;
    size_t kv = (size_t)L * c->max_seq * c->n_kv_heads * c->head_dim;
    m->kcache = (double *)malloc(sizeof(double) * kv);
    m->vcache = (double *)malloc(sizeof(double) * kv);
    m->seq_len = 0;
    return m;
}

void hqo_destroy(hqo_model *m) {
    if (!m) return;
    free(m->ptrs); free(m->kcache); free(m->vcache); free(m);
}

void hqo_reset(hqo_model *m) { m->seq_len = 0; }
int32_t hqo_seq_len(const hqo_model *m) { return m->seq_len; }

/*
 * Feed T tokens at positions seq_len .. seq_len+T-1 (SURVEY.md §8(c) "Algorithm", steps 1-3,
 * for each position in order; written layer by layer, which changes nothing because position p
 * only ever reads cache rows 0..p).  T = 1 is one decode step; T = prompt length is prefill.
 *
 * mode 0: nothing, 1: last position only, 2: all T positions.
 *   hidden_out: mode 1 -> [n_layers][hidden],  mode 2 -> [T][n_layers][hidden]   (step 2h)
 *   logits_out: mode 1 -> [vocab],             mode 2 -> [T][vocab]              (step 3)
 * Returns 0, or -1 on capacity overflow / bad token (state unchanged).
 */
int32_t hqo_forward(hqo_model *m, const int32_t *tokens, int32_t T, int32_t hidden_mode,
                    double *hidden_out, int32_t logits_mode, double *logits_out) {
    const hqo_config *c = &m->c;
    const int32_t d = c->hidden, H = c->n_heads, Hkv = c->n_kv_heads, hd = c->head_dim;
    const int32_t G = H / Hkv, qd = H * hd, kvd = Hkv * hd, F = c->ffn, L = c->n_layers;
    const int32_t p0 = m->seq_len;
    if (T <= 0 || p0 + T > c->max_seq) return -1;
    for (int32_t t = 0; t < T; ++t) if (tokens[t] < 0 || tokens[t] >= c->vocab) return -1;

    double *x = (double *)malloc(sizeof(double) * (size_t)T * d);
    double *h = (double *)malloc(sizeof(double) * (size_t)T * d);
    double *q = (double *)malloc(sizeof(double) * (size_t)T * qd);
    double *k = (double *)malloc(sizeof(double) * (size_t)T * kvd);
    double *v = (double *)malloc(sizeof(double) * (size_t)T * kvd);
    double *o = (double *)malloc(sizeof(double) * (size_t)T * qd);
    double *y = (double *)malloc(sizeof(double) * (size_t)T * d);
    double *g = (double *)malloc(sizeof(double) * (size_t)T * F);
    double *u = (double *)malloc(sizeof(double) * (size_t)T * F);

    /* step 1: x <- E[token] */
    for (int32_t t = 0; t < T; ++t)
        for (int32_t i = 0; i < d; ++i)
            x[(size_t)t * d + i] = (double)m->w.tok_embedding[(size_t)tokens[t] * d + i];

    for (int32_t l = 0; l < L; ++l) {
        double *Kl = m->kcache + (size_t)l * c->max_seq * kvd;
        double *Vl = m->vcache + (size_t)l * c->max_seq * kvd;
        /* 2a */
        for (int32_t t = 0; t < T; ++t)
            hqo_rmsnorm(x + (size_t)t * d, m->w.attn_norm[l], d, c->rms_eps, h + (size_t)t * d);
        /* 2b */
        hqo_matmul(m->w.wq[l], h, T, qd, d, q);
        hqo_matmul(m->w.wk[l], h, T, kvd, d, k);
        hqo_matmul(m->w.wv[l], h, T, kvd, d, v);
        /* 2c, 2d */
        for (int32_t t = 0; t < T; ++t) {
            int32_t p = p0 + t;
            for (int32_t j = 0; j < H; ++j) hqo_rope(q + (size_t)t * qd + j * hd, hd, p, c->rope_theta);
            for (int32_t j = 0; j < Hkv; ++j) hqo_rope(k + (size_t)t * kvd + j * hd, hd, p, c->rope_theta);
            memcpy(Kl + (size_t)p * kvd, k + (size_t)t * kvd, sizeof(double) * kvd);
            memcpy(Vl + (size_t)p * kvd, v + (size_t)t * kvd, sizeof(double) * kvd);
        }
        /* 2e: query head j uses KV head floor(j / G) (reading 8); position p sees rows 0..p */
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
        for (int32_t t = 0; t < T; ++t)
            for (int32_t j = 0; j < H; ++j) {
                int32_t kappa = j / G;
                hqo_attend(q + (size_t)t * qd + j * hd, Kl + kappa * hd, Vl + kappa * hd,
                           p0 + t + 1, kvd, hd, o + (size_t)t * qd + j * hd, NULL);
            }
        /* 2f */
        hqo_matmul(m->w.wo[l], o, T, d, qd, y);
        for (size_t i = 0; i < (size_t)T * d; ++i) x[i] += y[i];
        /* 2g */
        for (int32_t t = 0; t < T; ++t)
            hqo_rmsnorm(x + (size_t)t * d, m->w.ffn_norm[l], d, c->rms_eps, h + (size_t)t * d);
        hqo_matmul(m->w.w_gate[l], h, T, F, d, g);
        hqo_matmul(m->w.w_up[l], h, T, F, d, u);
        for (size_t i = 0; i < (size_t)T * F; ++i) g[i] = hqo_silu(g[i]) * u[i];
        hqo_matmul(m->w.w_down[l], g, T, d, F, y);
        for (size_t i = 0; i < (size_t)T * d; ++i) x[i] += y[i];
        /* 2h */
        if (hidden_mode == 2)
            for (int32_t t = 0; t < T; ++t)
                memcpy(hidden_out + ((size_t)t * L + l) * d, x + (size_t)t * d, sizeof(double) * d);
        else if (hidden_mode == 1)
            memcpy(hidden_out + (size_t)l * d, x + (size_t)(T - 1) * d, sizeof(double) * d);
    }

    /* step 3 */
    if (logits_mode == 2) {
        for (int32_t t = 0; t < T; ++t)
            hqo_rmsnorm(x + (size_t)t * d, m->w.final_norm, d, c->rms_eps, h + (size_t)t * d);
        hqo_matmul(m->w.lm_head, h, T, c->vocab, d, logits_out);
    } else if (logits_mode == 1) {
        hqo_rmsnorm(x + (size_t)(T - 1) * d, m->w.final_norm, d, c->rms_eps, h);
        hqo_matmul(m->w.lm_head, h, 1, c->vocab, d, logits_out);
    }

    m->seq_len = p0 + T;
    free(x); free(h); free(q); free(k); free(v); free(o); free(y); free(g); free(u);
    return 0;
}

/* read back one cached K or V row (test access): which 0 = K, 1 = V */
void hqo_get_kv(const hqo_model *m, int32_t which, int32_t layer, int32_t pos, double *out) {
    int32_t kvd = m->c.n_kv_heads * m->c.head_dim;
    const double *src = (which ? m->vcache : m->kcache) + ((size_t)layer * m->c.max_seq + pos) * kvd;
    memcpy(out, src, sizeof(double) * kvd);
}
