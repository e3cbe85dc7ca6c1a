"""CPU oracle of the host runtime path — TEST INFRASTRUCTURE, NOT PRODUCT.

Plain, slow Python restating what SURVEY.md 8(f)-3 asks of the host path, in the paper's order (section 4
"Runtime phase": route -> render -> speak; section 6.3: BM25 over a naive linear scan, margin gate with
tau = 0.05; section 6.4: bare answer line after a structural marker).  The BM25 definition is the textbook
one (Robertson & Zaragoza 2009, "The Probabilistic Relevance Framework", eq. 3.15 with the non-negative idf
ln(1 + (N - df + 0.5) / (df + 0.5))), written out term by term.  Shares no code with paper_2606_12154_b200/.
"""
from __future__ import annotations

import math
import re
from typing import Dict, List, Sequence, Tuple


def terms(text: str) -> List[str]:
    """Lower-cased runs of ASCII letters and digits."""
    return re.findall(r"[0-9a-z]+", text.lower().encode("ascii", "ignore").decode())


class Store:
    def __init__(self, key_text: Sequence[str], answer_line: Sequence[str], k1: float = 1.2, b: float = 0.75):
        self.k1, self.b = k1, b
        self.answers = list(answer_line)
        self.docs = [terms(k) for k in key_text]
        self.N = len(self.docs)
        self.avgdl = sum(len(d) for d in self.docs) / self.N
        self.df: Dict[str, int] = {}
        for d in self.docs:
            for t in set(d):
                self.df[t] = self.df.get(t, 0) + 1

    def idf(self, t: str) -> float:
        df = self.df.get(t, 0)
        return math.log(1.0 + (self.N - df + 0.5) / (df + 0.5))

    def score(self, query: str, d: int) -> float:
        """BM25 of entry d for the query: sum over the DISTINCT query terms that occur in the store."""
        doc = self.docs[d]
        total = 0.0
        for t in sorted(set(terms(query)), key=lambda t: (t not in self.df, t)):
            if t not in self.df:
                continue
            tf = doc.count(t)
            if tf == 0:
                continue
            total += self.idf(t) * tf * (self.k1 + 1.0) / (tf + self.k1 * (1.0 - self.b + self.b * len(doc) / self.avgdl))
        return total

    def route(self, query: str, top_k: int = 3) -> Tuple[List[int], List[float]]:
        """Linear scan; best first, ties to the lower entry index."""
        scored = [(self.score(query, d), d) for d in range(self.N)]
        scored.sort(key=lambda sd: (-sd[0], sd[1]))
        return [d for _, d in scored[:top_k]], [s for s, _ in scored[:top_k]]

    def render(self, entry: int, marker: str = "@@ANSWER") -> str:
        return marker + "\n" + self.answers[entry] + "\n"


def gate(s1: float, s2: float, tau: float = 0.05) -> Tuple[bool, float]:
    """(answer from the store?, margin): margin = (s1 - s2) / s1; escalate when it falls below tau."""
    margin = (s1 - s2) / s1 if s1 > 0 else 0.0
    return margin >= tau, margin


def tokenize(text: str, vocab: int) -> List[int]:
    """Synthetic tokeniser: alphanumeric words in pieces of <= 4 characters, other non-blank characters alone."""
    out = []
    for piece in re.findall(r"[0-9A-Za-z]{1,4}|[^0-9A-Za-z \t\r]", text.encode("ascii", "ignore").decode()):
        h = 14695981039346656037
        for c in piece.encode():
            h = ((h ^ c) * 1099511628211) & 0xFFFFFFFFFFFFFFFF
        out.append(h % vocab)
    return out
