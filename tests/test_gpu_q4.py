"""4-bit weight-only decode: the GPU quantiser against the hq4 oracle bit for bit, then the HQ_Q4
model against the quantisation-aware oracle (oracle.Model over the ORACLE's dequantised weights) with BASELINE.json's
tolerances."""
import numpy as np
import pytest

import datagen
import oracle
from oracle import q4_oracle as q4

pytestmark = pytest.mark.gpu

TOL_HIDDEN, TOL_LOGITS, MARGIN, MAXABS_LOGIT = 1e-2, 2e-2, 0.1, 0.05
KERNEL_PER_ROW = 8
TINYQ = datagen.Shape("tinyq", 2, 256, 4, 2, 64, 768, 4096, 1e-5, 10000.0)   # configs[0] with ffn a multiple of 128


def rel_l2(got, want):
    got, want = np.asarray(got, dtype=np.float64), np.asarray(want, dtype=np.float64)
    return float(np.linalg.norm(got - want) / np.linalg.norm(want))


def q4_oracle_model(weights, max_seq):
    """The quantisation-aware oracle: FFN matrices and the tied embedding / LM head replaced by the ORACLE quantiser's
    dequantised values; attention weights and gains as they are."""
    s, f = weights.shape, datagen.bf16_bits_to_f32
    dq = lambda bits: q4.dequantize(*q4.quantize(f(bits)))
    layers = []
    for t in weights.layers:
        d = {k: f(v) for k, v in t.items()}
        for k in ("w_gate", "w_up", "w_down"):
            d[k] = dq(t[k])
        layers.append(d)
    return oracle.Model(n_layers=s.n_layers, hidden=s.hidden, n_heads=s.n_heads, n_kv_heads=s.n_kv_heads, head_dim=s.head_dim,
                        ffn=s.ffn, vocab=s.vocab, rms_eps=s.rms_eps, rope_theta=s.rope_theta, max_seq=max_seq,
                        embedding=dq(weights.embedding), final_norm=f(weights.final_norm), layers=layers)


def test_quantizer_bit_exact():
    """hq_quantize_q4 / hq_dequantize_q4 against the oracle: codes, exponent bytes and dequantised values identical."""
    import torch
    import paper_2606_12154_b200 as hq
    w = datagen.make_weights(TINYQ)
    rng = np.random.default_rng(4)
    special = np.zeros((8, 64), dtype=np.float32)
    special[0, :4] = [7.0, -3.0, 1.0, 0.0]                       # e = 0
    special[1, :4] = [7.5, 1.0, 3.0, -5.0]                       # e = 1, ties to even
    special[2, 0] = 0.875                                         # exactly 7 * 2^-3
    special[3, 0] = 0.8828125                                     # the next bf16 above it -> e = -2
    special[4, 32:36] = [-7.0 * 32, 100.0, 0.5, -0.25]           # second group of the row
    special[5, :] = rng.normal(0, 1e-30, 64)                     # tiny magnitudes
    special[6, :] = rng.normal(0, 1e20, 64)                      # huge magnitudes
    cases = [datagen.bf16_bits_to_f32(w.layers[0]["w_gate"]), datagen.bf16_bits_to_f32(w.layers[1]["w_down"]),
             datagen.bf16_bits_to_f32(w.embedding)[:512], datagen.bf16_bits_to_f32(datagen.f32_to_bf16_bits(special))]
    for x in cases:
        qo, eo = q4.quantize(x)
        codes_o, exps_o = q4.pack(qo, eo)
        t = torch.from_numpy(datagen.f32_to_bf16_bits(x).view(np.int16)).cuda().view(torch.bfloat16)
        codes, exps = hq.quantize_q4(t)
        assert np.array_equal(codes.cpu().numpy(), codes_o) and np.array_equal(exps.cpu().numpy(), exps_o)
        d = hq.dequantize_q4(codes, exps).float().cpu().numpy()
        assert np.array_equal(d, q4.dequantize(qo, eo))


def run_q4(weights, prompt, n_steps, max_seq, path, sample_every=1):
    import paper_2606_12154_b200 as hq
    om = q4_oracle_model(weights, max_seq)
    gm = hq.Model.from_bf16_bits_q4(weights.shape, weights.embedding, weights.final_norm, weights.layers, max_seq=max_seq,
                                    flags=hq.FLAG_CAPTURE_HIDDEN | path)
    L = weights.shape.n_layers
    stats = {"hidden": 0.0, "logits": 0.0, "argmax_checked": 0, "positions": 0}
    h, lg = om.forward(prompt, hidden="last", logits="last")
    tok = gm.prefill(prompt)
    for i in range(n_steps + 1):
        want_tok, margin = oracle.argmax(lg), oracle.top2_margin(lg)
        if i % sample_every == 0 or i == n_steps:
            for l in range(L):
                e = rel_l2(gm.get_hidden(l)[0].cpu().numpy(), h[l])
                stats["hidden"] = max(stats["hidden"], e)
                assert e <= TOL_HIDDEN, f"step {i}: hidden after layer {l} rel-L2 {e:.3e}"
            got = gm.decode_logits()[0].cpu().numpy()
            e = rel_l2(got, lg)
            stats["logits"] = max(stats["logits"], e)
            assert e <= TOL_LOGITS and np.max(np.abs(got - lg)) <= MAXABS_LOGIT, f"step {i}: logits rel-L2 {e:.3e}"
            stats["positions"] += 1
        if margin > MARGIN:
            assert int(tok[0]) == want_tok, f"step {i}: argmax differs at margin {margin:.3f}"
            stats["argmax_checked"] += 1
        if i == n_steps:
            break
        h, lg = om.forward([want_tok], hidden="last", logits="last")
        tok = gm.decode_step(tokens_in=[want_tok])
    return stats, om


@pytest.mark.parametrize("path", [0, KERNEL_PER_ROW])
def test_tiny_q4_prefill_and_decode(path):
    w = datagen.make_weights(TINYQ)
    prompt = datagen.tokens(1000, TINYQ.vocab, 32)
    stats, om = run_q4(w, prompt, 16, 64, path)
    # the quantised model really differs from the bf16 one (otherwise this test would pass on the unquantised path)
    ob = oracle.Model.from_datagen(w, max_seq=64)
    _, lb = ob.forward(prompt, logits="last")
    om.reset()
    _, lq = om.forward(prompt, logits="last")
    assert rel_l2(lq, lb) > 0.05
    print("tiny q4 parity:", stats)
    assert stats["positions"] == 17


def test_tiny_q4_chunked_and_batched():
    """The tensor-core paths compute with the dequantised bf16 copies: chunked prefill (tensor-core, GEMV walk) and a
    batched decode step agree with the quantisation-aware oracle too."""
    import paper_2606_12154_b200 as hq
    w = datagen.make_weights(TINYQ)
    toks = datagen.tokens(1005, TINYQ.vocab, 44)
    om = q4_oracle_model(w, 64)
    _, lg = om.forward(toks, logits="all")
    gm = hq.Model.from_bf16_bits_q4(w.shape, w.embedding, w.final_norm, w.layers, max_seq=64, max_batch=2)
    gm.prefill(toks[:17]); gm.prefill(toks[17:20]); gm.prefill(toks[20:40])
    assert rel_l2(gm.decode_logits()[0].cpu().numpy(), lg[39]) <= TOL_LOGITS
    gm.decode_step(tokens_in=[int(toks[40])])
    assert rel_l2(gm.decode_logits()[0].cpu().numpy(), lg[40]) <= TOL_LOGITS
    gm.kv_reset()
    gm.prefill(np.stack([toks[:40], toks[:40]]))
    gm.decode_step(tokens_in=[int(toks[40])] * 2)
    got = gm.decode_logits(batch=2).cpu().numpy()
    assert rel_l2(got[0], lg[40]) <= TOL_LOGITS and rel_l2(got[1], lg[40]) <= TOL_LOGITS


def test_1b_q4_teacher_forced():
    """configs[1] shape with hq4 FFN + LM head: 256-token prompt (tcgen05 GEMMs over the dequantised copies), then 32
    teacher-forced decode steps through the 4-bit streaming GEMV."""
    w = datagen.make_weights(datagen.ONE_B)
    prompt = datagen.tokens(1001, datagen.ONE_B.vocab, 256)
    stats, _ = run_q4(w, prompt, 32, 320, 0, sample_every=8)
    print("1b q4 parity:", stats)
    assert stats["positions"] == 5
