"""GPU parity: libhq (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Tolerances are BASELINE.json north_star's: relative L2 <= 1e-2 per-layer hidden
state, <= 2e-2 on logits, teacher-forced greedy argmax identical wherever the oracle's top-2 logit
margin exceeds 0.1 (SURVEY.md §8(c) readings 13-15)."""
import numpy as np
import pytest

import datagen
import oracle

pytestmark = pytest.mark.gpu

TOL_HIDDEN, TOL_LOGITS, MARGIN = 1e-2, 2e-2, 0.1


def rel_l2(got, want):
    got, want = np.asarray(got, dtype=np.float64), np.asarray(want, dtype=np.float64)
    return float(np.linalg.norm(got - want) / np.linalg.norm(want))


def gpu_model(weights, max_seq, flags=None, max_batch=1, no_mega=None):
    """Batch-1 decode paths, all held to the same tolerances.  no_mega=None: the default (per-step kernels with QKV +
    attention + O of a layer in one launch); True: one kernel per step of the path (hq_decode.cu only, HQ_FLAG_NO_MEGA);
    False: the persistent kernel (hq_mega.cu, HQ_FLAG_MEGA)."""
    import paper_2606_12154_b200 as hq
    f = hq.FLAG_CAPTURE_HIDDEN if flags is None else flags
    if no_mega is not None:
        f |= hq.FLAG_NO_MEGA if no_mega else hq.FLAG_MEGA
    return hq.Model.from_bf16_bits(weights.shape, weights.embedding, weights.final_norm, weights.layers,
                                   max_seq=max_seq, max_batch=max_batch, flags=f)


def check_position(gm, want_hidden, want_logits, where, stats):
    L = want_hidden.shape[0]
    for l in range(L):
        e = rel_l2(gm.get_hidden(l)[0].cpu().numpy(), want_hidden[l])
        stats["hidden"] = max(stats.get("hidden", 0.0), e)
        assert e <= TOL_HIDDEN, f"{where}: hidden after layer {l} rel-L2 {e:.3e}"
    lg = gm.decode_logits()[0].cpu().numpy()
    e = rel_l2(lg, want_logits)
    stats["logits"] = max(stats.get("logits", 0.0), e)
    assert e <= TOL_LOGITS, f"{where}: logits rel-L2 {e:.3e}"
    return lg


def run_teacher_forced(gm, om, prompt, n_steps, check_every=1):
    """Prefill + n_steps teacher-forced steps: the GPU is fed the ORACLE's greedy tokens."""
    ref = om.greedy(prompt, n_steps, hidden="last")
    stats = {"argmax_checked": 0}
    tok = gm.prefill(prompt)
    lg = check_position(gm, ref["hidden"][0], ref["logits"][0], "prefill", stats)
    if ref["margins"][0] > MARGIN:
        assert int(tok[0]) == int(ref["tokens"][0]) == int(lg.argmax())
        stats["argmax_checked"] += 1
    for i in range(1, n_steps + 1):
        out = gm.decode_step(tokens_in=[int(ref["tokens"][i - 1])])
        if i % check_every == 0 or i == n_steps:
            check_position(gm, ref["hidden"][i], ref["logits"][i], f"step {i}", stats)
        if ref["margins"][i] > MARGIN:
            assert int(out[0]) == int(ref["tokens"][i]), f"step {i}: argmax differs at margin {ref['margins'][i]:.3f}"
            stats["argmax_checked"] += 1
    assert gm.seq_len() == om.seq_len == len(prompt) + n_steps
    return ref, stats


# ---------------------------------------------------------------------------------------------------
# configs[0]: tiny model, 32-token prompt, 16 greedy steps
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("no_mega", [None, False, True])
def test_tiny_prefill_and_decode(tiny_weights, tiny_tokens, no_mega):
    gm = gpu_model(tiny_weights, max_seq=64, no_mega=no_mega)
    om = oracle.Model.from_datagen(tiny_weights, max_seq=64)
    ref, stats = run_teacher_forced(gm, om, tiny_tokens, 16)
    assert stats["argmax_checked"] >= 8
    print("tiny parity:", stats)


@pytest.mark.parametrize("no_mega", [None, False, True])
def test_tiny_every_prompt_position(tiny_weights, tiny_tokens, no_mega):
    """configs[0] additionally compares all prompt positions (chunked prefill, one token at a time)."""
    gm = gpu_model(tiny_weights, max_seq=64, no_mega=no_mega)
    om = oracle.Model.from_datagen(tiny_weights, max_seq=64)
    hid, lg = om.forward(tiny_tokens, hidden="all", logits="all")
    stats = {}
    for t, tok in enumerate(tiny_tokens):
        first = gm.prefill([int(tok)])
        got = check_position(gm, hid[t], lg[t], f"prompt position {t}", stats)
        if oracle.top2_margin(lg[t]) > MARGIN:
            assert int(first[0]) == oracle.argmax(lg[t]) == int(got.argmax())
    print("tiny per-position parity:", stats)


def test_tiny_free_running_matches_teacher_forced(tiny_weights, tiny_tokens):
    """Device-fed greedy decode (what the bench times) emits the oracle's tokens when margins are wide,
    and graph replay / direct launch / no-PDL variants agree bit for bit."""
    import paper_2606_12154_b200 as hq
    om = oracle.Model.from_datagen(tiny_weights, max_seq=64)
    ref = om.greedy(tiny_tokens, 16)
    for family in (0, hq.FLAG_MEGA, hq.FLAG_NO_MEGA):
        outs = []
        for flags in (0, hq.FLAG_NO_GRAPH, hq.FLAG_NO_PDL, hq.FLAG_NO_GRAPH | hq.FLAG_NO_PDL):
            gm = gpu_model(tiny_weights, max_seq=64, flags=flags | family)
            first = gm.prefill(tiny_tokens)
            toks = gm.decode_run(16)[:, 0]
            lg = gm.decode_logits()[0].cpu().numpy()
            outs.append((int(first[0]), toks.copy(), lg))
            # streaming one step per call emits the same tokens as the single multi-step call
            gm.kv_reset()
            gm.prefill(tiny_tokens)
            one_by_one = np.array([int(gm.decode_step()[0]) for _ in range(16)])
            assert np.array_equal(one_by_one, toks) and np.array_equal(gm.decode_logits()[0].cpu().numpy(), lg)
        for o in outs[1:]:
            assert o[0] == outs[0][0] and np.array_equal(o[1], outs[0][1]) and np.array_equal(o[2], outs[0][2])
        got = np.concatenate([[outs[0][0]], outs[0][1]])
        if ref["margins"].min() > MARGIN:
            assert np.array_equal(got, ref["tokens"])


def test_tiny_kv_reset_and_reuse(tiny_weights, tiny_tokens):
    gm = gpu_model(tiny_weights, max_seq=64)
    gm.prefill(tiny_tokens)
    a = gm.decode_run(4)
    la = gm.decode_logits().cpu().numpy()
    gm.kv_reset()
    assert gm.seq_len() == 0
    gm.prefill(tiny_tokens)
    b = gm.decode_run(4)
    lb = gm.decode_logits().cpu().numpy()
    assert np.array_equal(a, b) and np.array_equal(la, lb)


@pytest.mark.parametrize("no_mega", [None, False, True])
def test_tiny_ragged_lengths(tiny_weights, no_mega):
    """Context lengths around the 16/32/64/128 tile and split boundaries of the attention kernels: the
    prompt goes through prefill, then ONE decode step attends over n+1 positions (decode attention)."""
    toks = datagen.tokens(4242, datagen.TINY.vocab, 202)
    om = oracle.Model.from_datagen(tiny_weights, max_seq=256)
    _, lg = om.forward(toks, logits="all")
    gm = gpu_model(tiny_weights, max_seq=256, no_mega=no_mega)
    checked = 0
    for n in (1, 2, 15, 16, 17, 31, 33, 63, 64, 65, 127, 128, 129, 191, 200):
        gm.kv_reset()
        gm.prefill(toks[:n])
        e = rel_l2(gm.decode_logits()[0].cpu().numpy(), lg[n - 1])
        assert e <= TOL_LOGITS, f"prompt length {n}: logits rel-L2 {e:.3e}"
        gm.decode_step(tokens_in=[int(toks[n])])
        e = rel_l2(gm.decode_logits()[0].cpu().numpy(), lg[n])
        assert e <= TOL_LOGITS, f"decode at context {n + 1}: logits rel-L2 {e:.3e}"
        checked += 1
    assert checked == 15


def test_error_paths(tiny_weights, tiny_tokens):
    import paper_2606_12154_b200 as hq
    gm = gpu_model(tiny_weights, max_seq=40)
    with pytest.raises(hq.HQError) as e:
        gm.decode_step()
    assert e.value.code == -3                                  # decode before prefill
    with pytest.raises(hq.HQError) as e:
        gm.prefill(np.zeros(41, dtype=np.int32))
    assert e.value.code == -2                                  # capacity
    with pytest.raises(hq.HQError) as e:
        gm.prefill([datagen.TINY.vocab])
    assert e.value.code == -1                                  # token out of range
    with pytest.raises(hq.HQError) as e:
        gm.prefill(np.zeros((1, 0), dtype=np.int32))
    assert e.value.code == -1                                  # empty input
    assert gm.seq_len() == 0                                   # state unchanged by failures
    gm.prefill(tiny_tokens)
    gm.decode_run(8)
    with pytest.raises(hq.HQError) as e:
        gm.decode_step()
    assert e.value.code == -2 and gm.seq_len() == 40           # full cache
    with pytest.raises(hq.HQError) as e:
        gpu_model(tiny_weights, max_seq=40, flags=0).get_hidden(0)
    assert e.value.code == -3


# ---------------------------------------------------------------------------------------------------
# configs[1]: 1B model, 256-token prompt, 128 greedy steps (full size, the launch config bench times)
# ---------------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def one_b_weights():
    return datagen.make_weights(datagen.ONE_B)


@pytest.mark.parametrize("no_mega", [None, False, True])
def test_1b_config1_teacher_forced(one_b_weights, no_mega):
    s = datagen.ONE_B
    prompt = datagen.tokens(1001, s.vocab, 256)
    gm = gpu_model(one_b_weights, max_seq=512, no_mega=no_mega)
    om = oracle.Model.from_datagen(one_b_weights, max_seq=512)
    ref, stats = run_teacher_forced(gm, om, prompt, 128, check_every=8)
    frac = float((ref["margins"] > MARGIN).mean())
    print("1b config[1] parity:", stats, "positions with margin>0.1: %.2f" % frac)
    assert stats["argmax_checked"] >= 16


def test_1b_config2_long_context_sampled(one_b_weights):
    """configs[2] at full size: 2,048-token prompt (one tensor-core pass, causal flash attention over 32 query tiles),
    then teacher-forced decode steps at context 2,048+ (8 context splits per KV head in the attention block).  The
    oracle is run on the first steps only (sampled outputs; 256 steps would cost minutes of CPU)."""
    s = datagen.ONE_B
    prompt = datagen.tokens(1002, s.vocab, 2048)
    gm = gpu_model(one_b_weights, max_seq=2304)
    om = oracle.Model.from_datagen(one_b_weights, max_seq=2304)
    ref, stats = run_teacher_forced(gm, om, prompt, 6, check_every=1)
    print("1b config[2] parity:", stats)
    assert stats["argmax_checked"] >= 2


# ---------------------------------------------------------------------------------------------------
# batched serving (configs[3] shape on the tiny model): tensor-core prefill + batched decode
# ---------------------------------------------------------------------------------------------------
def run_batched(gm, weights, prompts, n_steps, max_seq, check_every=1):
    """Every sequence is run alone through the oracle (reading 17); the GPU runs them as one batch,
    teacher-forced with the oracle's tokens.  Returns worst errors."""
    B, T = prompts.shape
    refs = []
    for b in range(B):
        om = oracle.Model.from_datagen(weights, max_seq=max_seq)
        refs.append(om.greedy(prompts[b], n_steps, hidden="last"))
    stats = {"hidden": 0.0, "logits": 0.0, "argmax_checked": 0}
    L = weights.shape.n_layers

    def check(i, toks):
        lg = gm.decode_logits(batch=B).cpu().numpy()
        hid = [gm.get_hidden(l, batch=B).cpu().numpy() for l in range(L)]
        for b in range(B):
            e = rel_l2(lg[b], refs[b]["logits"][i])
            stats["logits"] = max(stats["logits"], e)
            assert e <= TOL_LOGITS, f"seq {b} pos {i}: logits rel-L2 {e:.3e}"
            for l in range(L):
                e = rel_l2(hid[l][b], refs[b]["hidden"][i][l])
                stats["hidden"] = max(stats["hidden"], e)
                assert e <= TOL_HIDDEN, f"seq {b} pos {i} layer {l}: hidden rel-L2 {e:.3e}"
            if refs[b]["margins"][i] > MARGIN:
                assert int(toks[b]) == int(refs[b]["tokens"][i]), f"seq {b} pos {i}"
                stats["argmax_checked"] += 1

    first = gm.prefill(prompts)
    check(0, first)
    for i in range(1, n_steps + 1):
        out = gm.decode_step(tokens_in=[int(refs[b]["tokens"][i - 1]) for b in range(B)])
        if i % check_every == 0 or i == n_steps:
            check(i, out[:B])
    assert gm.seq_len() == T + n_steps
    return refs, stats


def test_tiny_batched_prefill_and_decode(tiny_weights):
    B, T, steps = 3, 24, 10
    prompts = datagen.tokens(1003, datagen.TINY.vocab, B * T).reshape(B, T)
    gm = gpu_model(tiny_weights, max_seq=64, max_batch=4)
    refs, stats = run_batched(gm, tiny_weights, prompts, steps, 64)
    print("tiny batched parity:", stats)
    assert stats["argmax_checked"] >= B * 4


def test_1b_config3_batch8_sampled(one_b_weights):
    """configs[3] at full size: 8 sequences x 192-token prompts in one tensor-core pass (1,536 rows), then batched
    decode steps (tcgen05 GEMMs with a 32-token tile, split-K across the SMs).  Sampled: the first steps only."""
    s = datagen.ONE_B
    B, T, steps = 8, 192, 3
    prompts = datagen.tokens(1003, s.vocab, B * T).reshape(B, T)
    gm = gpu_model(one_b_weights, max_seq=T + 192, max_batch=B)
    refs, stats = run_batched(gm, one_b_weights, prompts, steps, T + 192)
    print("1b config[3] parity:", stats)
    assert stats["argmax_checked"] >= B


def test_tiny_batch_invariance(tiny_weights):
    """Sequence 0's logits do not depend on its neighbours beyond rounding (reading 17)."""
    T = 20
    prompts = datagen.tokens(1004, datagen.TINY.vocab, 4 * T).reshape(4, T)
    gm = gpu_model(tiny_weights, max_seq=64, max_batch=4)
    gm.prefill(prompts)
    gm.decode_run(3, batch=4)
    a = gm.decode_logits(batch=4)[0].cpu().numpy()
    gm.kv_reset()
    other = prompts.copy()
    other[1:] = prompts[1:][::-1]
    gm.prefill(other[:2])
    gm.decode_run(3, batch=2)
    b = gm.decode_logits(batch=2)[0].cpu().numpy()
    assert rel_l2(a, b) < 1e-4


def test_tiny_chunked_prefill_matches_single_pass(tiny_weights):
    toks = datagen.tokens(1005, datagen.TINY.vocab, 60)
    gm = gpu_model(tiny_weights, max_seq=64)
    gm.prefill(toks)
    a = gm.decode_logits()[0].cpu().numpy()
    gm.kv_reset()
    gm.prefill(toks[:17]); gm.prefill(toks[17:20]); gm.prefill(toks[20:])   # tensor-core, GEMV, tensor-core
    b = gm.decode_logits()[0].cpu().numpy()
    assert rel_l2(b, a) < 2e-3
    om = oracle.Model.from_datagen(tiny_weights, max_seq=64)
    _, lg = om.forward(toks, logits="last")
    assert rel_l2(a, lg) <= TOL_LOGITS and rel_l2(b, lg) <= TOL_LOGITS
