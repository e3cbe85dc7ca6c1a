"""Host runtime path (include/hq_host.h): the oracle (oracle/host_oracle.py) against what the BM25
definition and the paper fix, then libhq_host.so against the oracle on the synthetic 563-entry store, query by query.
All CPU: no test here needs a GPU."""
import math
import os
import re
import subprocess

import numpy as np
import pytest

from oracle import host_oracle as ho

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


# ---- oracle pins ---------------------------------------------------------------------------------------
def test_bm25_worked_example():
    """Three documents, worked by hand (k1 = 1.2, b = 0.75, avgdl = 3, idf = ln(1 + 1.5 / 2.5) = ln 1.6 for both terms):
    d0 'apple banana'            : apple tf 1, |d| 2 -> ln1.6 * 2.2 / (1 + 0.9)
    d1 'apple apple cherry'      : apple tf 2, cherry tf 1, |d| 3 -> ln1.6 * (4.4 / 3.2 + 2.2 / 2.2)
    d2 'banana cherry cherry date': cherry tf 2, |d| 4 -> ln1.6 * 4.4 / (2 + 1.5)"""
    s = ho.Store(["apple banana", "apple apple cherry", "banana cherry cherry date"], ["a", "b", "c"])
    assert s.avgdl == 3.0 and s.df == {"apple": 2, "banana": 2, "cherry": 2, "date": 1}
    assert abs(s.idf("apple") - 0.47000362924573563) < 1e-15
    want = [0.5442147286003255, 1.1162586194586221, 0.5908617053374962]
    for d in range(3):
        assert abs(s.score("Apple, cherry?", d) - want[d]) < 1e-12
    ids, scores = s.route("apple cherry", 3)
    assert ids == [1, 2, 0] and abs(scores[0] - want[1]) < 1e-12


def test_bm25_properties():
    docs = ["x y z", "x x y z w", "q r s t u v", "x"]
    s = ho.Store(docs, ["-"] * 4)
    # rarer terms weigh more; a repeated term saturates (tf 2 scores less than twice tf 1 at equal length)
    assert s.idf("w") > s.idf("y") > s.idf("x")
    t = ho.Store(["a b", "a a"], ["-", "-"])
    assert t.score("a", 0) < t.score("a", 1) < 2 * t.score("a", 0)
    # the same tf in a longer document scores lower; unknown terms and repeated query terms change nothing
    u = ho.Store(["a b", "a b c d e f"], ["-", "-"])
    assert u.score("a", 0) > u.score("a", 1)
    assert s.score("nothing here", 0) == 0.0 and s.score("x", 2) == 0.0
    assert s.score("x x x y", 0) == s.score("y x", 0)
    # b = 0: no length normalisation; k1 = 0: binary model (idf only)
    v = ho.Store(["a b", "a b c d e f"], ["-", "-"], k1=1.2, b=0.0)
    assert v.score("a", 0) == v.score("a", 1)
    w = ho.Store(["a a a b", "a c"], ["-", "-"], k1=0.0, b=0.75)
    assert abs(w.score("a", 0) - w.idf("a")) < 1e-15 and abs(w.score("a", 1) - w.idf("a")) < 1e-15
    # ties go to the lower index; zero scores still rank by index
    z = ho.Store(["m n", "m n", "o"], ["-"] * 3)
    assert z.route("m", 3)[0] == [0, 1, 2]


def test_gate_threshold():
    """margin below tau = 0.05 escalates."""
    assert ho.gate(1.0, 0.96) == (False, pytest.approx(0.04))
    assert ho.gate(1.0, 0.94)[0] is True and ho.gate(2.0, 1.0) == (True, 0.5)
    assert ho.gate(0.0, 0.0) == (False, 0.0)            # nothing matched: escalate
    ok, m = ho.gate(1.0, 0.95)
    assert abs(m - 0.05) < 1e-15                        # at the threshold the decision is whatever IEEE gives; both sides agree (below)


def test_renderer_and_tokenizer_pins():
    s = ho.Store(["k"], ["the VRAM slack is 312 MiB."])
    assert s.render(0) == "@@ANSWER\nthe VRAM slack is 312 MiB.\n"          # bare line after a structural marker, verbatim
    # FNV-1a 64 published vectors: "" -> cbf29ce484222325, "a" -> af63dc4c8601ec8c, "foobar" -> 85944171f73967e8
    assert ho.tokenize("a", 1 << 62) == [0xaf63dc4c8601ec8c % (1 << 62)]
    assert ho.tokenize("foobar", 1000) == [ho.tokenize("foob", 1000)[0], ho.tokenize("ar", 1000)[0]]   # pieces of <= 4 characters
    assert len(ho.tokenize("Hello, world 12345!\nab", 50000)) == 2 + 1 + 2 + 2 + 1 + 1 + 1   # Hell o , worl d 1234 5 ! \\n ab
    assert ho.terms("VRAM-slack: 312MiB") == ["vram", "slack", "312mib"]


# ---- libhq_host.so against the oracle ----------------------------------------------------------------
@pytest.fixture(scope="module")
def hostlib():
    from paper_2606_12154_b200 import build
    build.build_host()
    from paper_2606_12154_b200 import hostlib
    return hostlib


@pytest.fixture(scope="module")
def synthetic_store():
    from datagen import store as ds
    return ds.make_store()


def test_host_header_binding_library_agree(hostlib):
    src = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "hq_host.h")).read(), flags=re.S)
    declared = sorted(set(re.findall(r"\b(hqh_[a-z_0-9]+)\s*\(", src)))
    assert declared == sorted(hostlib.DECLARED_SYMBOLS)
    out = subprocess.check_output(["nm", "-D", "--defined-only", os.path.join(ROOT, "paper_2606_12154_b200", "libhq_host.so")]).decode()
    assert set(declared) <= set(re.findall(r" T (hqh_[a-z_0-9]+)", out))


def test_route_gate_render_match_the_oracle_on_the_563_entry_store(hostlib, synthetic_store):
    keys, answers, queries, targets = synthetic_store
    assert len(keys) == 563 and len(queries) == 1126
    S, O = hostlib.Store(keys, answers), ho.Store(keys, answers)
    top1 = top3 = gated = 0
    for q, t in zip(queries, targets):
        ids, sc = S.route(q, 3)
        oids, osc = O.route(q, 3)
        assert list(ids) == oids, q                               # index work: exact
        assert np.allclose(sc, osc, rtol=1e-12, atol=0)
        ok, margin = hostlib.gate(sc[0], sc[1])
        ook, omargin = ho.gate(osc[0], osc[1])
        if abs(omargin - 0.05) > 1e-9:
            assert ok == ook
        assert abs(margin - omargin) < 1e-12
        top1 += int(ids[0] == t)
        top3 += int(t in ids)
        gated += int(not ok)
    for e in range(0, 563, 7):
        assert S.render(e) == O.render(e, hostlib.marker())       # byte work: exact
        assert list(hostlib.tokenize(S.render(e), 128256)) == ho.tokenize(O.render(e), 128256)
    # the synthetic query set is shaped like the paper's (most queries route, a minority trips the gate)
    n = len(queries)
    assert top1 / n > 0.8 and top3 / n >= top1 / n and 0.01 < gated / n < 0.3
    print(f"synthetic store: top-1 {top1 / n:.3f}, top-3 {top3 / n:.3f}, gated {gated / n:.3f}")


def test_host_edge_cases(hostlib):
    S = hostlib.Store(["alpha beta", "gamma"], ["one", "two"])
    ids, sc = S.route("", 2)
    assert list(ids) == [0, 1] and list(sc) == [0.0, 0.0]        # empty query: nothing scores, order by index
    assert hostlib.gate(0.0, 0.0) == (False, 0.0)
    with pytest.raises(ValueError):
        S.route("alpha", 3)                                       # top_k > entries
    with pytest.raises(ValueError):
        S.render(2)
    with pytest.raises(ValueError):
        hostlib.Store([], [])
    assert list(hostlib.tokenize("", 100)) == []
    long_answer = "w " * 40000
    T = hostlib.Store(["k"], [long_answer])
    with pytest.raises(ValueError):
        T.render(0)                                               # does not fit the binding's 64 KiB buffer: -2, no overflow
