// hq_host.cpp — host-side runtime path (include/hq_host.h): BM25 linear-scan router, margin gate, marker-line renderer,
// synthetic tokeniser.  Plain C++17, no dependencies; single-threaded per call (the paper measures one user).
#include "../../include/hq_host.h"

#include <math.h>
#include <string.h>

#include <algorithm>
#include <new>
#include <string>
#include <unordered_map>
#include <vector>

namespace {

// lower-cased runs of ASCII letters and digits
void split_terms(const char *text, std::vector<std::string> &out) {
    out.clear();
    std::string cur;
    for (const unsigned char *p = reinterpret_cast<const unsigned char *>(text); *p; ++p) {
        const unsigned char c = *p;
        const bool alnum = (c >= '0' && c <= '9') || (c >= 'a' && c <= 'z') || (c >= 'A' && c <= 'Z');
        if (alnum) {
            cur.push_back((char)((c >= 'A' && c <= 'Z') ? c - 'A' + 'a' : c));
        } else if (!cur.empty()) {
            out.push_back(cur);
            cur.clear();
        }
    }
    if (!cur.empty()) out.push_back(cur);
}

struct Posting { int32_t term; int32_t tf; };

}  // namespace

struct hqh_store {
    double k1, b, avgdl;
    std::vector<std::string> answers;
    std::unordered_map<std::string, int32_t> term_id;
    std::vector<int32_t> df;                       // documents containing the term
    std::vector<std::vector<Posting>> docs;        // per entry: its distinct terms and their counts (sorted by term id)
    std::vector<int32_t> doc_len;                  // terms per entry (with repeats)
};

extern "C" int32_t hqh_store_create(const char *const *key_text, const char *const *answer_line, int32_t n, double k1, double b,
                                    hqh_store **out) {
    if (!out) return -1;
    *out = nullptr;
    if (!key_text || !answer_line || n <= 0 || !(k1 >= 0.0) || !(b >= 0.0 && b <= 1.0)) return -1;
    for (int32_t i = 0; i < n; ++i)
        if (!key_text[i] || !answer_line[i]) return -1;
    hqh_store *s = new (std::nothrow) hqh_store();
    if (!s) return -2;
    s->k1 = k1;
    s->b = b;
    s->answers.reserve(n);
    s->docs.resize(n);
    s->doc_len.resize(n);
    std::vector<std::string> terms;
    long long total = 0;
    for (int32_t i = 0; i < n; ++i) {
        s->answers.emplace_back(answer_line[i]);
        split_terms(key_text[i], terms);
        s->doc_len[i] = (int32_t)terms.size();
        total += (long long)terms.size();
        std::unordered_map<int32_t, int32_t> tf;
        for (const std::string &t : terms) {
            auto it = s->term_id.find(t);
            int32_t id;
            if (it == s->term_id.end()) {
                id = (int32_t)s->df.size();
                s->term_id.emplace(t, id);
                s->df.push_back(0);
            } else {
                id = it->second;
            }
            ++tf[id];
        }
        for (const auto &kv : tf) {
            s->docs[i].push_back(Posting{kv.first, kv.second});
            ++s->df[kv.first];
        }
        std::sort(s->docs[i].begin(), s->docs[i].end(), [](const Posting &a, const Posting &c) { return a.term < c.term; });
    }
    s->avgdl = (double)total / (double)n;
    *out = s;
    return 0;
}

extern "C" void hqh_store_destroy(hqh_store *s) { delete s; }
extern "C" int32_t hqh_store_size(const hqh_store *s) { return s ? (int32_t)s->answers.size() : -1; }

extern "C" int32_t hqh_route(const hqh_store *s, const char *query, int32_t top_k, int32_t *ids_out, double *scores_out) {
    if (!s || !query || !ids_out || !scores_out || top_k <= 0 || top_k > 8 || top_k > (int32_t)s->answers.size()) return -1;
    std::vector<std::string> terms;
    split_terms(query, terms);
    // distinct query terms known to the store, with their idf, in ascending term id (the order of summation)
    std::vector<std::pair<int32_t, double>> q;
    const double N = (double)s->answers.size();
    for (const std::string &t : terms) {
        auto it = s->term_id.find(t);
        if (it == s->term_id.end()) continue;
        bool seen = false;
        for (const auto &e : q) seen = seen || e.first == it->second;
        if (!seen) q.emplace_back(it->second, log(1.0 + (N - (double)s->df[it->second] + 0.5) / ((double)s->df[it->second] + 0.5)));
    }
    std::sort(q.begin(), q.end(), [](const std::pair<int32_t, double> &a, const std::pair<int32_t, double> &c) { return a.first < c.first; });
    int32_t best_id[8];
    double best_sc[8];
    int32_t filled = 0;
    // "a deliberately naive linear scan": every entry is scored
    for (int32_t d = 0; d < (int32_t)s->docs.size(); ++d) {
        const std::vector<Posting> &doc = s->docs[d];
        const double norm = s->k1 * (1.0 - s->b + s->b * (double)s->doc_len[d] / s->avgdl);
        double score = 0.0;
        size_t j = 0;
        for (const auto &e : q) {   // both lists ascend by term id
            while (j < doc.size() && doc[j].term < e.first) ++j;
            if (j < doc.size() && doc[j].term == e.first) {
                const double tf = (double)doc[j].tf;
                score += e.second * tf * (s->k1 + 1.0) / (tf + norm);
            }
        }
        // insert into the top-k (strictly better score wins; equal scores keep the lower index first)
        int32_t pos = filled;
        while (pos > 0 && score > best_sc[pos - 1]) --pos;
        if (pos < top_k) {
            const int32_t last = filled < top_k ? filled : top_k - 1;
            for (int32_t m = last; m > pos; --m) { best_id[m] = best_id[m - 1]; best_sc[m] = best_sc[m - 1]; }
            best_id[pos] = d;
            best_sc[pos] = score;
            if (filled < top_k) ++filled;
        }
    }
    for (int32_t i = 0; i < top_k; ++i) { ids_out[i] = best_id[i]; scores_out[i] = best_sc[i]; }
    return 0;
}

extern "C" int32_t hqh_gate(double s1, double s2, double tau, double *margin_out) {
    const double margin = s1 > 0.0 ? (s1 - s2) / s1 : 0.0;
    if (margin_out) *margin_out = margin;
    return margin < tau ? 0 : 1;
}

static const char kMarker[] = "@@ANSWER";
extern "C" const char *hqh_marker(void) { return kMarker; }

extern "C" int32_t hqh_render(const hqh_store *s, int32_t id, char *buf, int32_t cap) {
    if (!s || !buf || id < 0 || id >= (int32_t)s->answers.size() || cap <= 0) return -1;
    const std::string &a = s->answers[id];
    const size_t need = sizeof(kMarker) - 1 + 1 + a.size() + 1;
    if (need + 1 > (size_t)cap) return -2;
    char *p = buf;
    memcpy(p, kMarker, sizeof(kMarker) - 1); p += sizeof(kMarker) - 1;
    *p++ = '\n';
    memcpy(p, a.data(), a.size()); p += a.size();
    *p++ = '\n';
    *p = '\0';
    return (int32_t)need;
}

extern "C" int32_t hqh_tokenize(const char *text, int32_t vocab, int32_t *tokens_out, int32_t cap) {
    if (!text || !tokens_out || vocab <= 0 || cap < 0) return -1;
    int32_t n = 0;
    auto emit = [&](const unsigned char *p, size_t len) -> bool {
        unsigned long long h = 14695981039346656037ull;   // FNV-1a 64
        for (size_t i = 0; i < len; ++i) { h ^= p[i]; h *= 1099511628211ull; }
        if (n >= cap) return false;
        tokens_out[n++] = (int32_t)(h % (unsigned long long)vocab);
        return true;
    };
    const unsigned char *p = reinterpret_cast<const unsigned char *>(text);
    while (*p) {
        const unsigned char c = *p;
        const bool alnum = (c >= '0' && c <= '9') || (c >= 'a' && c <= 'z') || (c >= 'A' && c <= 'Z');
        if (alnum) {
            size_t len = 0;
            while (len < 4) {
                const unsigned char e = p[len];
                if (!((e >= '0' && e <= '9') || (e >= 'a' && e <= 'z') || (e >= 'A' && e <= 'Z'))) break;
                ++len;
            }
            if (!emit(p, len)) return -2;
            p += len;
        } else if (c == ' ' || c == '\t' || c == '\r') {
            ++p;
        } else {
            if (!emit(p, 1)) return -2;
            ++p;
        }
    }
    return n;
}
