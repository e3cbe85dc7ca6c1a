"""Seeded synthetic store and query set shaped like the paper's (section 6.3: 563 entries built from
17 documents, probed with 1,126 queries "generated from distinctive vocabulary in the source documents"; answer lines of
~70 tokens typical and at most ~230).  Input generator only: no routing, scoring or rendering here.
The paper's own store and queries are private; nothing of them is reproduced."""
from __future__ import annotations

from typing import List, Tuple

import numpy as np

N_ENTRIES, N_QUERIES, N_DOCUMENTS = 563, 1126, 17

_SYL = ["ka", "ro", "mi", "ten", "vu", "sol", "dar", "pe", "lin", "go", "sha", "bur", "ne", "qui", "tam", "zo", "fel", "ix",
        "mor", "ul", "ba", "cre", "dun", "eph", "ga", "hol", "jin", "ky", "lo", "mar", "nu", "os"]


def _word(rng: np.random.Generator, n_syl: int) -> str:
    return "".join(_SYL[i] for i in rng.integers(0, len(_SYL), n_syl))


def make_store(seed: int = 563) -> Tuple[List[str], List[str], List[str], List[int]]:
    """Returns (key_text [563], answer_line [563], queries [1126], query_target [1126])."""
    rng = np.random.default_rng(seed)
    common = [_word(rng, 1 + int(rng.integers(0, 2))) for _ in range(60)]             # frequent, uninformative words
    doc_vocab = [[_word(rng, 2) for _ in range(40)] for _ in range(N_DOCUMENTS)]      # per-document topic words
    keys, answers, distinct = [], [], []
    for e in range(N_ENTRIES):
        doc = e % N_DOCUMENTS
        own = [_word(rng, 3) + str(int(rng.integers(0, 100))) for _ in range(int(rng.integers(2, 5)))]   # distinctive vocabulary
        topic = [doc_vocab[doc][i] for i in rng.integers(0, 40, int(rng.integers(2, 5)))]
        filler = [common[i] for i in rng.integers(0, 60, int(rng.integers(3, 8)))]
        key = own + topic + filler
        alias = [own[int(rng.integers(0, len(own)))]] + [doc_vocab[doc][int(rng.integers(0, 40))]] + \
                [common[int(rng.integers(0, 60))] for _ in range(2)]
        rng.shuffle(key)
        keys.append(" ".join(key) + " ; " + " ".join(alias))
        n_words = int(np.clip(rng.lognormal(np.log(38), 0.55), 8, 135))               # ~60-70 tokens typical, <= ~230
        words = [(_word(rng, int(rng.integers(1, 4))) if rng.random() < 0.85 else str(int(rng.integers(0, 10000))))
                 for _ in range(n_words)]
        answers.append(" ".join(words) + ".")
        distinct.append((own, topic))
    queries, targets = [], []
    for q in range(N_QUERIES):
        e = q % N_ENTRIES
        own, topic = distinct[e]
        picks = [own[int(rng.integers(0, len(own)))]]
        if rng.random() < 0.6:
            picks.append(own[int(rng.integers(0, len(own)))])
        if rng.random() < 0.7:
            picks.append(topic[int(rng.integers(0, len(topic)))])
        # a sixth of the queries only carry topic words: several entries of the document match, the margin is small
        if rng.random() < 0.16:
            picks = [topic[int(rng.integers(0, len(topic)))] for _ in range(2)]
        noise = [common[int(rng.integers(0, 60))] for _ in range(int(rng.integers(2, 6)))]
        words = picks + noise
        rng.shuffle(words)
        queries.append("what about " + " ".join(words) + " ?")
        targets.append(e)
    return keys, answers, queries, targets
