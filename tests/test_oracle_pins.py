"""Pins for the CPU oracle (oracle/hq_oracle.c) against what the definitions fix.

Nothing in the paper prints a value this path must reproduce, so the oracle
is pinned to closed forms, invariants, special cases, brute force and an independent float64
torch re-expression — SURVEY.md §8(c) "What pins the oracle".  Golden constants below are textbook
values (cos 1, sin 1, sigmoid(1)), not outputs of any code in this repository.
"""
import math

import numpy as np
import pytest
import torch
import torch.nn.functional as F

import datagen
import oracle

rng = np.random.default_rng(1234)


# ------------------------------------------------------------------ RoPE ----------------------------
def test_rope_position_zero_is_identity():
    v = rng.standard_normal(64)
    assert np.array_equal(oracle.rope(v, 0, 10000.0), v)


def test_rope_worked_value_hd2():
    # hd=2, p=1: (1,0) -> (cos 1, sin 1) = (0.5403023058681398, 0.8414709848078965)
    out = oracle.rope(np.array([1.0, 0.0]), 1, 10000.0)
    assert abs(out[0] - 0.5403023058681398) < 1e-15 and abs(out[1] - 0.8414709848078965) < 1e-15
    # (0,1) -> (-sin 1, cos 1): fixes the sign of the rotation
    out = oracle.rope(np.array([0.0, 1.0]), 1, 10000.0)
    assert abs(out[0] + 0.8414709848078965) < 1e-15 and abs(out[1] - 0.5403023058681398) < 1e-15


def test_rope_pairing_and_frequencies_hd4():
    # hd=4, theta=10000: pair (0,2) turns by p*1, pair (1,3) by p*theta^(-2/4) = p/100
    p = 3
    out = oracle.rope(np.array([1.0, 1.0, 0.0, 0.0]), p, 10000.0)
    want = [math.cos(3.0), math.cos(0.03), math.sin(3.0), math.sin(0.03)]
    assert np.allclose(out, want, atol=1e-15)


def test_rope_norm_preserved_and_relative():
    q, k = rng.standard_normal(64), rng.standard_normal(64)
    for theta in (10000.0, 500000.0):
        r = oracle.rope(q, 1234, theta)
        assert np.allclose(q[:32] ** 2 + q[32:] ** 2, r[:32] ** 2 + r[32:] ** 2, rtol=1e-12)
        a = oracle.rope(q, 17, theta) @ oracle.rope(k, 5, theta)
        b = oracle.rope(q, 1017, theta) @ oracle.rope(k, 1005, theta)
        c = oracle.rope(q, 12, theta) @ k
        assert abs(a - b) < 1e-9 and abs(a - c) < 1e-9


# ------------------------------------------------------------------ attention ------------------------
def test_attention_rows_sum_to_one_and_shift_invariance():
    q, K, V = rng.standard_normal(64), rng.standard_normal((37, 64)), rng.standard_normal((37, 64))
    o, p = oracle.attend(q, K, V, return_probs=True)
    assert abs(p.sum() - 1.0) < 1e-12 and np.all(p > 0)
    # adding a constant vector c*q/|q|^2-direction shift to all scores: K + 1 (x) u with <q,u> = const
    u = q / (q @ q)
    o2, p2 = oracle.attend(q, K + 5.0 * u[None, :], V, return_probs=True)
    assert np.allclose(p, p2, atol=1e-12) and np.allclose(o, o2, atol=1e-12)


def test_attention_context_one_returns_v0():
    q, K, V = rng.standard_normal(64), rng.standard_normal((1, 64)), rng.standard_normal((1, 64))
    assert np.allclose(oracle.attend(q, K, V), V[0], atol=0, rtol=0)
    assert np.allclose(oracle.attend(100 * q, K, V), V[0], atol=0, rtol=0)


def test_attention_brute_force_numpy_and_scale():
    hd = 64
    q, K, V = rng.standard_normal(hd), rng.standard_normal((9, hd)), rng.standard_normal((9, hd))
    s = (K @ q) * 0.125                       # 1/sqrt(64) exactly (reading 9)
    e = np.exp(s - s.max())
    want = (e / e.sum()) @ V
    assert np.allclose(oracle.attend(q, K, V), want, atol=1e-13)
    # uniform case: q = 0 gives the mean of V
    assert np.allclose(oracle.attend(np.zeros(hd), K, V), V.mean(axis=0), atol=1e-13)
    # a dominant key selects its value
    K2 = K.copy(); K2[4] = 50 * q
    assert np.allclose(oracle.attend(q, K2, V), V[4], atol=1e-9)


def test_attention_matches_torch_sdpa():
    q, K, V = rng.standard_normal(64), rng.standard_normal((21, 64)), rng.standard_normal((21, 64))
    want = F.scaled_dot_product_attention(torch.tensor(q)[None, None, None], torch.tensor(K)[None, None],
                                          torch.tensor(V)[None, None])[0, 0, 0].numpy()
    assert np.allclose(oracle.attend(q, K, V), want, atol=1e-12)


# ------------------------------------------------------------------ RMSNorm / SiLU / argmax ----------
def test_rmsnorm_closed_forms():
    d, eps = 256, 1e-5
    g = (1 + 0.1 * rng.standard_normal(d)).astype(np.float32)
    c = 0.37
    out = oracle.rmsnorm(np.full(d, c), g, eps)
    assert np.allclose(out, g.astype(np.float64) * c / math.sqrt(c * c + eps), rtol=1e-14)
    x = rng.standard_normal(d)
    ones = np.ones(d, dtype=np.float32)
    y = oracle.rmsnorm(x, ones, eps)
    ms = (x ** 2).mean()
    assert abs(math.sqrt((y ** 2).mean()) - 1 / math.sqrt(1 + eps / ms)) < 1e-14
    # scale invariance as eps -> 0, and eps sits inside the sqrt: x = 0 gives 0 (not NaN)
    assert np.allclose(oracle.rmsnorm(x, g, 0.0), oracle.rmsnorm(7.5 * x, g, 0.0), rtol=1e-13)
    assert np.array_equal(oracle.rmsnorm(np.zeros(d), g, eps), np.zeros(d))
    # tiny x: output ~ x / sqrt(eps)
    assert np.allclose(oracle.rmsnorm(1e-9 * x, ones, eps), 1e-9 * x / math.sqrt(eps), rtol=1e-9)
    assert np.allclose(y, F.rms_norm(torch.tensor(x), (d,), torch.ones(d, dtype=torch.float64), eps).numpy(),
                       rtol=1e-13)


def test_silu_values():
    assert oracle.silu(0.0) == 0.0
    assert abs(oracle.silu(1.0) - 0.7310585786300049) < 1e-15     # sigmoid(1)
    assert abs(oracle.silu(-1.0) + 0.2689414213699951) < 1e-15    # -sigmoid(-1)
    assert abs(oracle.silu(40.0) - 40.0) < 1e-12 and abs(oracle.silu(-40.0)) < 1e-12


def test_matmul_orientation():
    W = rng.standard_normal((5, 3)).astype(np.float32)
    X = rng.standard_normal((2, 3))
    assert np.allclose(oracle.matmul(W, X), X @ W.astype(np.float64).T, atol=1e-14)
    E = np.zeros((1, 3)); E[0, 2] = 1.0            # picks column 2 of W: y = W x with W [out, in]
    assert np.allclose(oracle.matmul(W, E)[0], W[:, 2], atol=0)


def test_argmax_ties_lowest_index_and_margin():
    v = np.array([0.5, 2.0, -1.0, 2.0, 1.5, 2.0])
    assert oracle.argmax(v) == 1 and oracle.top2_margin(v) == 0.0
    w = rng.standard_normal(1000)
    assert oracle.argmax(w) == int(np.argmax(w))
    s = np.sort(w)
    assert abs(oracle.top2_margin(w) - (s[-1] - s[-2])) < 1e-15
    w[[10, 700]] = 9.0
    assert oracle.argmax(w) == 10


# ------------------------------------------------------------------ whole model ----------------------
def _small_model(H=4, Hkv=2, L=2, d=64, hd=16, Fdim=96, V=50, seed=7, zero_out=False, max_seq=32,
                 theta=10000.0):
    r = np.random.default_rng(seed)
    def mat(o, i):
        return (0.08 * r.standard_normal((o, i))).astype(np.float32)
    layers = []
    for _ in range(L):
        layers.append({
            "attn_norm": (1 + 0.05 * r.standard_normal(d)).astype(np.float32),
            "wq": mat(H * hd, d), "wk": mat(Hkv * hd, d), "wv": mat(Hkv * hd, d),
            "wo": np.zeros((d, H * hd), np.float32) if zero_out else mat(d, H * hd),
            "ffn_norm": (1 + 0.05 * r.standard_normal(d)).astype(np.float32),
            "w_gate": mat(Fdim, d), "w_up": mat(Fdim, d),
            "w_down": np.zeros((d, Fdim), np.float32) if zero_out else mat(d, Fdim)})
    kw = dict(n_layers=L, hidden=d, n_heads=H, n_kv_heads=Hkv, head_dim=hd, ffn=Fdim, vocab=V,
              rms_eps=1e-5, rope_theta=theta, max_seq=max_seq,
              embedding=mat(V, d), final_norm=(1 + 0.05 * r.standard_normal(d)).astype(np.float32),
              layers=layers)
    return kw


def torch_reference(kw, tokens):
    """Independent float64 re-expression with torch library ops: F.rms_norm, complex-number RoPE,
    F.scaled_dot_product_attention(is_causal=True) on explicitly repeated K/V, F.silu.
    Full-sequence, no KV cache.  Returns hidden [T, L, d], logits [T, V]."""
    t64 = lambda a: torch.tensor(np.asarray(a, dtype=np.float64))
    H, Hkv, hd, d = kw["n_heads"], kw["n_kv_heads"], kw["head_dim"], kw["hidden"]
    T = len(tokens)
    E = t64(kw["embedding"])
    x = E[torch.tensor(np.asarray(tokens, dtype=np.int64))]
    pos = torch.arange(T, dtype=torch.float64)
    inv = kw["rope_theta"] ** (-torch.arange(0, hd, 2, dtype=torch.float64) / hd)
    rot = torch.polar(torch.ones(T, hd // 2, dtype=torch.float64), pos[:, None] * inv[None, :])

    def rope(z):  # z [T, heads, hd]; pair (i, i + hd/2) is one complex number
        zc = torch.complex(z[..., : hd // 2], z[..., hd // 2:]) * rot[:, None, :]
        return torch.cat([zc.real, zc.imag], dim=-1)

    hidden = []
    for lw in kw["layers"]:
        h = F.rms_norm(x, (d,), t64(lw["attn_norm"]), kw["rms_eps"])
        q = rope((h @ t64(lw["wq"]).T).view(T, H, hd))
        k = rope((h @ t64(lw["wk"]).T).view(T, Hkv, hd))
        v = (h @ t64(lw["wv"]).T).view(T, Hkv, hd)
        k = k.repeat_interleave(H // Hkv, dim=1)
        v = v.repeat_interleave(H // Hkv, dim=1)
        o = F.scaled_dot_product_attention(q.transpose(0, 1)[None], k.transpose(0, 1)[None],
                                           v.transpose(0, 1)[None], is_causal=True)[0]
        x = x + o.transpose(0, 1).reshape(T, H * hd) @ t64(lw["wo"]).T
        h2 = F.rms_norm(x, (d,), t64(lw["ffn_norm"]), kw["rms_eps"])
        x = x + (F.silu(h2 @ t64(lw["w_gate"]).T) * (h2 @ t64(lw["w_up"]).T)) @ t64(lw["w_down"]).T
        hidden.append(x)
    logits = F.rms_norm(x, (d,), t64(kw["final_norm"]), kw["rms_eps"]) @ E.T
    return torch.stack(hidden, dim=1).numpy(), logits.numpy()


def _rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def test_small_model_matches_torch_float64_route():
    kw = _small_model()
    toks = rng.integers(0, kw["vocab"], 12)
    m = oracle.Model(**kw)
    hid, lg = m.forward(toks, hidden="all", logits="all")
    rh, rl = torch_reference(kw, toks)
    assert _rel(hid, rh) < 1e-12 and _rel(lg, rl) < 1e-12


def test_configs0_matches_torch_float64_route(tiny_weights, tiny_tokens):
    """configs[0] (fp32 weights verbatim, reading 2) against the independent torch route."""
    s = datagen.TINY
    m = oracle.Model.from_datagen(tiny_weights, max_seq=64, use_raw_fp32=True)
    hid, lg = m.forward(tiny_tokens, hidden="all", logits="all")
    raw = tiny_weights.raw
    kw = dict(n_heads=s.n_heads, n_kv_heads=s.n_kv_heads, head_dim=s.head_dim, hidden=s.hidden,
              rms_eps=s.rms_eps, rope_theta=s.rope_theta, embedding=raw[datagen.TID_EMBEDDING],
              final_norm=raw[datagen.TID_FINAL_NORM],
              layers=[{k: raw[datagen.layer_tid(l, k)] for k in datagen.LAYER_TENSORS}
                      for l in range(s.n_layers)])
    rh, rl = torch_reference(kw, tiny_tokens)
    assert _rel(hid, rh) < 1e-12 and _rel(lg, rl) < 1e-12
    assert np.array_equal(lg.argmax(axis=1), rl.argmax(axis=1))


def test_incremental_decode_equals_full_sequence(tiny_weights, tiny_tokens):
    """KV-cache decode one token at a time == one full-sequence pass == chunked prefill."""
    m = oracle.Model.from_datagen(tiny_weights, max_seq=64)
    hid_full, lg_full = m.forward(tiny_tokens, hidden="all", logits="all")
    m.reset()
    for t, tok in enumerate(tiny_tokens):
        h, lg = m.forward([tok], hidden="last", logits="last")
        assert _rel(h, hid_full[t]) < 1e-13 and _rel(lg, lg_full[t]) < 1e-13
    m.reset()
    m.forward(tiny_tokens[:13], logits="none")
    h, lg = m.forward(tiny_tokens[13:], hidden="all", logits="all")
    assert _rel(h, hid_full[13:]) < 1e-13 and _rel(lg, lg_full[13:]) < 1e-13
    assert m.seq_len == 32


def test_causality_bit_identical_prefix(tiny_weights, tiny_tokens):
    m = oracle.Model.from_datagen(tiny_weights, max_seq=64)
    hid_a, lg_a = m.forward(tiny_tokens, hidden="all", logits="all")
    toks = tiny_tokens.copy(); toks[20] = (toks[20] + 1) % datagen.TINY.vocab
    m.reset()
    hid_b, lg_b = m.forward(toks, hidden="all", logits="all")
    assert np.array_equal(hid_a[:20], hid_b[:20]) and np.array_equal(lg_a[:20], lg_b[:20])
    assert not np.array_equal(hid_a[20], hid_b[20]) and not np.array_equal(hid_a[31], hid_b[31])


def test_gqa_equals_mha_on_repeated_kv():
    kw = _small_model(H=4, Hkv=2)
    toks = rng.integers(0, kw["vocab"], 9)
    _, lg_gqa = oracle.Model(**kw).forward(toks, logits="all")
    kw2 = dict(kw); kw2["n_kv_heads"] = 4
    hd = kw["head_dim"]
    rep = lambda w: np.repeat(w.reshape(2, hd, -1), 2, axis=0).reshape(4 * hd, -1)  # head j <- kv j//2
    kw2["layers"] = [dict(l, wk=rep(l["wk"]), wv=rep(l["wv"])) for l in kw["layers"]]
    _, lg_mha = oracle.Model(**kw2).forward(toks, logits="all")
    assert _rel(lg_gqa, lg_mha) < 1e-13
    # and Hkv == H equals the independent torch multi-head route
    _, rl = torch_reference(kw2, toks)
    assert _rel(lg_mha, rl) < 1e-12


def test_zero_output_projections_special_case():
    """W_o = W_d = 0: residual is the embedding; logits_j = <e_j, RMSNorm(e_t; g_f)> (closed form),
    hidden_l = e_t for every layer."""
    kw = _small_model(zero_out=True)
    toks = rng.integers(0, kw["vocab"], 6)
    hid, lg = oracle.Model(**kw).forward(toks, hidden="all", logits="all")
    E = kw["embedding"].astype(np.float64)
    for t, tok in enumerate(toks):
        e = E[tok]
        assert np.array_equal(hid[t, 0], e) and np.array_equal(hid[t, 1], e)
        want = E @ (e / math.sqrt((e ** 2).mean() + 1e-5) * kw["final_norm"].astype(np.float64))
        assert np.allclose(lg[t], want, atol=1e-13)


def test_tied_embedding_zero_proj_predicts_input_token(tiny_weights, tiny_tokens):
    """With tied embeddings, gains ~ 1 and zeroed W_o, W_d the greedy next token is the input token
    (|e_t|^2 ~ d * 0.02^2 dominates the cross terms)."""
    s = datagen.TINY
    layers = []
    for l, t in enumerate(tiny_weights.layers):
        lw = {k: datagen.bf16_bits_to_f32(v) for k, v in t.items()}
        lw["wo"] = np.zeros_like(lw["wo"]); lw["w_down"] = np.zeros_like(lw["w_down"])
        layers.append(lw)
    m = oracle.Model(n_layers=s.n_layers, hidden=s.hidden, n_heads=s.n_heads, n_kv_heads=s.n_kv_heads,
                     head_dim=s.head_dim, ffn=s.ffn, vocab=s.vocab, rms_eps=s.rms_eps,
                     rope_theta=s.rope_theta, max_seq=64,
                     embedding=datagen.bf16_bits_to_f32(tiny_weights.embedding),
                     final_norm=datagen.bf16_bits_to_f32(tiny_weights.final_norm), layers=layers)
    _, lg = m.forward(tiny_tokens, logits="all")
    assert np.array_equal(lg.argmax(axis=1), tiny_tokens)


def test_permutation_symmetries():
    kw = _small_model()
    toks = rng.integers(0, kw["vocab"], 8)
    _, base = oracle.Model(**kw).forward(toks, logits="all")
    # permute FFN units
    perm = rng.permutation(kw["ffn"])
    kw2 = dict(kw)
    kw2["layers"] = [dict(l, w_gate=l["w_gate"][perm], w_up=l["w_up"][perm], w_down=l["w_down"][:, perm])
                     for l in kw["layers"]]
    _, lg = oracle.Model(**kw2).forward(toks, logits="all")
    assert _rel(lg, base) < 1e-12
    # permute heads consistently: swap KV groups (q heads 0,1 <-> 2,3; kv heads 0 <-> 1)
    hd = kw["head_dim"]
    qp = np.concatenate([np.arange(2 * hd, 4 * hd), np.arange(0, 2 * hd)])
    kp = np.concatenate([np.arange(hd, 2 * hd), np.arange(0, hd)])
    kw3 = dict(kw)
    kw3["layers"] = [dict(l, wq=l["wq"][qp], wk=l["wk"][kp], wv=l["wv"][kp], wo=l["wo"][:, qp])
                     for l in kw["layers"]]
    _, lg = oracle.Model(**kw3).forward(toks, logits="all")
    assert _rel(lg, base) < 1e-12


def test_kv_cache_holds_rotated_k_and_raw_v():
    kw = _small_model()
    toks = rng.integers(0, kw["vocab"], 5)
    m = oracle.Model(**kw)
    hid, _ = m.forward(toks, hidden="all", logits="none")
    # layer-0 K row at position 3 == RoPE(Wk RMSNorm(e_tok)), V row == Wv RMSNorm(e_tok)
    e = kw["embedding"][toks[3]].astype(np.float64)
    h = oracle.rmsnorm(e, kw["layers"][0]["attn_norm"], 1e-5)
    k = kw["layers"][0]["wk"].astype(np.float64) @ h
    v = kw["layers"][0]["wv"].astype(np.float64) @ h
    hd = kw["head_dim"]
    k_rot = np.concatenate([oracle.rope(k[j * hd:(j + 1) * hd], 3, kw["rope_theta"]) for j in range(2)])
    assert np.allclose(m.kv_row("k", 0, 3), k_rot, atol=1e-14)
    assert np.allclose(m.kv_row("v", 0, 3), v, atol=1e-14)


def test_capacity_and_bad_token_rejected():
    kw = _small_model(max_seq=8)
    m = oracle.Model(**kw)
    with pytest.raises(ValueError):
        m.forward(np.zeros(9, dtype=np.int32))
    with pytest.raises(ValueError):
        m.forward([kw["vocab"]])
    assert m.seq_len == 0
    m.forward(np.zeros(8, dtype=np.int32))
    with pytest.raises(ValueError):
        m.forward([0])


def test_greedy_protocol(tiny_weights, tiny_tokens):
    """configs[0]: 32-token prompt, 16 greedy steps -> 17 emitted tokens, 48 cached positions."""
    m = oracle.Model.from_datagen(tiny_weights, max_seq=64)
    r = m.greedy(tiny_tokens, 16)
    assert r["tokens"].shape == (17,) and m.seq_len == 48
    m.reset()
    seq = np.concatenate([tiny_tokens, r["tokens"][:-1]])
    _, lg = m.forward(seq, logits="all")
    assert np.array_equal(lg[31:].argmax(axis=1), r["tokens"])
    assert _rel(lg[31:], r["logits"]) < 1e-13
