/*
 * hq_host.h — C ABI of libhq_host: the host-side runtime path in front of the mouth model.
 *
 * PAPER.md:L70 (section 4, "Runtime phase"): "a router maps the incoming question to a stored key.  A deterministic
 * renderer produces the factual answer line from the stored entry — this step involves no model and takes effectively
 * zero time.  A 1B-class model ... then streams the answer".  PAPER.md:L137-144 (section 6.3): the router that works on
 * the 563-entry store is BM25 over a "deliberately naive linear scan" (p50 2.40 ms on the author's laptop), followed by a
 * confidence gate: "queries whose margin falls below a threshold (tau = 0.05) are escalated rather than answered".
 * PAPER.md:L152 (section 6.4): the answer must reach the mouth "as a bare line following a structural marker".
 *
 * The paper discloses neither the store format, nor the BM25 variant, nor the marker; the readings
 * taken here are listed in DESIGN.md section 10.  Everything in this library runs on the HOST; all pointers are HOST
 * pointers; strings are NUL-terminated UTF-8 (tokenised as ASCII: letters and digits, lower-cased).  Every call returns
 * 0 or a negative code (-1 invalid argument, -2 capacity); no exceptions, no abort().
 */
#ifndef HQ_HOST_H_
#define HQ_HOST_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hqh_store hqh_store; /* opaque, library-owned */

/* Build the store over n_entries (key text, answer line) pairs; both arrays are copied.  The key text (stored key plus
 * its aliases, "keys and aliases for retrieval") is what the router indexes; the answer line is what the
 * renderer emits verbatim.  BM25 parameters k1, b (Robertson/Sparck Jones; DESIGN.md section 10 uses 1.2 and 0.75). */
int32_t hqh_store_create(const char *const *key_text, const char *const *answer_line, int32_t n_entries, double k1, double b,
                         hqh_store **out);
void hqh_store_destroy(hqh_store *s);
int32_t hqh_store_size(const hqh_store *s);

/* BM25 linear scan: scores every entry against the query and returns the top_k (<= 8) entries, best
 * first, ties broken by the lower entry index.  ids_out / scores_out: arrays of top_k; entries with score 0 still rank
 * (by index) so that the arrays are always full when n_entries >= top_k.
 *   score(q, d) = sum over DISTINCT query terms t of idf(t) * tf(t, d) * (k1 + 1) / (tf(t, d) + k1 * (1 - b + b * |d| / avgdl))
 *   idf(t) = ln(1 + (N - df(t) + 0.5) / (df(t) + 0.5)) */
int32_t hqh_route(const hqh_store *s, const char *query, int32_t top_k, int32_t *ids_out, double *scores_out);

/* Confidence gate: margin = (s1 - s2) / s1 of the two best scores (0 when s1 <= 0); returns 1 = answer
 * from the store, 0 = escalate (margin < tau).  margin_out may be NULL. */
int32_t hqh_gate(double s1, double s2, double tau, double *margin_out);

/* Deterministic renderer: writes "<marker>\n<answer line>\n" for entry id into buf (capacity
 * cap bytes including the NUL); returns the length written (without the NUL) or -2 when it does not fit. */
int32_t hqh_render(const hqh_store *s, int32_t id, char *buf, int32_t cap);
const char *hqh_marker(void); /* the structural marker line, static storage */

/* Synthetic tokeniser for the (random-weight) mouth model: words of letters/digits are cut into pieces of <= 4
 * characters, every other non-blank character is a piece of its own, a newline is a piece; piece -> FNV-1a 64 hash mod
 * vocab.  Returns the number of tokens written (<= cap) or -2.  Stands in for the undisclosed tokenizer of the paper's
 * MiniCPM5-1B; only the token COUNT matters for timing. */
int32_t hqh_tokenize(const char *text, int32_t vocab, int32_t *tokens_out, int32_t cap);

#ifdef __cplusplus
}
#endif
#endif /* HQ_HOST_H_ */
