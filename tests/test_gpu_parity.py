"""GPU parity: libhq (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Tolerances are BASELINE.json north_star's: relative L2 <= 1e-2 per-layer hidden
state, <= 2e-2 on logits, teacher-forced greedy argmax identical wherever the oracle's top-2 logit
margin exceeds 0.1 (SURVEY.md §8(c) readings 13-15).  Beside every relative-L2 bound stands a
max-abs bound (one wrong element among 128,256 logits moves the norm by less than the tolerance):
|delta logit| <= 0.05, half the argmax margin."""
import numpy as np
import pytest

import datagen
import oracle

pytestmark = pytest.mark.gpu

TOL_HIDDEN, TOL_LOGITS, MARGIN = 1e-2, 2e-2, 0.1
MAXABS_LOGIT = 0.05       # absolute, per logit (logits of these models are O(1))
MAXABS_HIDDEN_REL = 0.05  # per element, relative to the largest |element| of the oracle's vector
TOL_KV = 1e-2             # cached K/V rows (fp16 storage: 2^-11 relative rounding per element)

KERNEL_PER_ROW = 8        # HQ_FLAG_KERNEL_PER_ROW
PATHS = [pytest.param(0, id="attention-block"), pytest.param(KERNEL_PER_ROW, id="kernel-per-row")]


def rel_l2(got, want):
    got, want = np.asarray(got, dtype=np.float64), np.asarray(want, dtype=np.float64)
    return float(np.linalg.norm(got - want) / np.linalg.norm(want))


def max_abs(got, want):
    return float(np.max(np.abs(np.asarray(got, dtype=np.float64) - np.asarray(want, dtype=np.float64))))


def gpu_model(weights, max_seq, flags=None, max_batch=1, path=0):
    """path = 0: the default batch-1 decode path (cluster attention block per layer + streaming GEMVs);
    KERNEL_PER_ROW: one kernel per row of SURVEY.md §8(a) (hq_decode.cu only).  Same tolerances."""
    import paper_2606_12154_b200 as hq
    f = hq.FLAG_CAPTURE_HIDDEN if flags is None else flags
    gm = hq.Model.from_bf16_bits(weights.shape, weights.embedding, weights.final_norm, weights.layers,
                                 max_seq=max_seq, max_batch=max_batch, flags=f | path)
    want = "kernel-per-row" if path else "attention-block-cluster"
    assert gm.decode_path() == want, gm.decode_path()
    return gm


def check_vectors(hid, lg, want_hidden, want_logits, where, stats):
    for l in range(want_hidden.shape[0]):
        e = rel_l2(hid[l], want_hidden[l])
        a = max_abs(hid[l], want_hidden[l]) / float(np.max(np.abs(want_hidden[l])))
        stats["hidden"] = max(stats.get("hidden", 0.0), e)
        stats["hidden_maxabs_rel"] = max(stats.get("hidden_maxabs_rel", 0.0), a)
        assert e <= TOL_HIDDEN, f"{where}: hidden after layer {l} rel-L2 {e:.3e}"
        assert a <= MAXABS_HIDDEN_REL, f"{where}: hidden after layer {l} max-abs / max|x| {a:.3e}"
    e, a = rel_l2(lg, want_logits), max_abs(lg, want_logits)
    stats["logits"] = max(stats.get("logits", 0.0), e)
    stats["logits_maxabs"] = max(stats.get("logits_maxabs", 0.0), a)
    assert e <= TOL_LOGITS, f"{where}: logits rel-L2 {e:.3e}"
    assert a <= MAXABS_LOGIT, f"{where}: logits max-abs {a:.3e}"


def check_position(gm, want_hidden, want_logits, where, stats):
    hid = [gm.get_hidden(l)[0].cpu().numpy() for l in range(want_hidden.shape[0])]
    lg = gm.decode_logits()[0].cpu().numpy()
    check_vectors(hid, lg, want_hidden, want_logits, where, stats)
    return lg


def check_kv_rows(gm, om, positions, stats, seq=0):
    """Cache rows (rotated K, raw V) of the given positions, every layer, against the oracle's cache."""
    for pos in positions:
        for l in range(om.n_layers):
            for which in ("k", "v"):
                got = gm.kv_row(which, l, pos, seq).float().cpu().numpy()
                want = om.kv_row(which, l, pos)
                e = rel_l2(got, want)
                stats["kv"] = max(stats.get("kv", 0.0), e)
                assert e <= TOL_KV, f"{which} row layer {l} position {pos}: rel-L2 {e:.3e}"
        stats["kv_rows"] = stats.get("kv_rows", 0) + 1


def oracle_reference(weights, prompt, n_steps, max_seq, sample_every=1):
    """Greedy oracle run: tokens and top-2 margins at every step, hidden states and
    logits at step 0 (the prefill), every sample_every-th step and the last one."""
    om = oracle.Model.from_datagen(weights, max_seq=max_seq)
    h, lg = om.forward(prompt, hidden="last", logits="last")
    ref = {"tokens": [], "margins": [], "sampled": {}, "om": om, "prompt": np.asarray(prompt), "n_steps": n_steps}
    for i in range(n_steps + 1):
        ref["tokens"].append(oracle.argmax(lg))
        ref["margins"].append(oracle.top2_margin(lg))
        if i % sample_every == 0 or i == n_steps:
            ref["sampled"][i] = (h, lg)
        if i == n_steps:
            break
        h, lg = om.forward([ref["tokens"][-1]], hidden="last", logits="last")
    ref["tokens"] = np.array(ref["tokens"], dtype=np.int32)
    ref["margins"] = np.array(ref["margins"])
    return ref


def run_teacher_forced(gm, ref):
    """Prefill + n_steps teacher-forced steps: the GPU is fed the ORACLE's greedy tokens; argmax is compared at
    every step of margin > 0.1, hidden states and logits at the sampled steps."""
    stats = {"argmax_checked": 0, "positions": 0}
    tok = gm.prefill(ref["prompt"])
    for i in range(ref["n_steps"] + 1):
        if i:
            tok = gm.decode_step(tokens_in=[int(ref["tokens"][i - 1])])
        if i in ref["sampled"]:
            lg = check_position(gm, ref["sampled"][i][0], ref["sampled"][i][1], f"step {i}", stats)
            stats["positions"] += 1
            if ref["margins"][i] > MARGIN:
                assert int(lg.argmax()) == int(ref["tokens"][i])
        if ref["margins"][i] > MARGIN:
            assert int(tok[0]) == int(ref["tokens"][i]), f"step {i}: argmax differs at margin {ref['margins'][i]:.3f}"
            stats["argmax_checked"] += 1
    assert gm.seq_len() == ref["om"].seq_len == len(ref["prompt"]) + ref["n_steps"]
    return stats


# ---------------------------------------------------------------------------------------------------
# configs[0]: tiny model, 32-token prompt, 16 greedy steps
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("path", PATHS)
def test_tiny_prefill_and_decode(tiny_weights, tiny_tokens, path):
    gm = gpu_model(tiny_weights, max_seq=64, path=path)
    ref = oracle_reference(tiny_weights, tiny_tokens, 16, 64)
    stats = run_teacher_forced(gm, ref)
    assert stats["argmax_checked"] >= 8 and stats["positions"] == 17
    # every cached row: positions 0..31 written by the tensor-core prefill pass (rows 0..T-2 of that pass are seen by
    # nothing else directly), 32..47 by the decode path's fused RoPE + append
    check_kv_rows(gm, ref["om"], range(48), stats)
    print("tiny parity:", stats)


@pytest.mark.parametrize("path", PATHS)
def test_tiny_every_prompt_position(tiny_weights, tiny_tokens, path):
    """configs[0] additionally compares all prompt positions (chunked prefill, one token at a time: the GEMV walk)."""
    gm = gpu_model(tiny_weights, max_seq=64, path=path)
    om = oracle.Model.from_datagen(tiny_weights, max_seq=64)
    hid, lg = om.forward(tiny_tokens, hidden="all", logits="all")
    stats = {}
    for t, tok in enumerate(tiny_tokens):
        first = gm.prefill([int(tok)])
        got = check_position(gm, hid[t], lg[t], f"prompt position {t}", stats)
        if oracle.top2_margin(lg[t]) > MARGIN:
            assert int(first[0]) == oracle.argmax(lg[t]) == int(got.argmax())
    print("tiny per-position parity:", stats)


def test_tiny_every_row_of_a_tensor_core_pass(tiny_weights, tiny_tokens):
    """Rows 0..T-1 of ONE tcgen05 prefill pass against the oracle: growing prefixes of the prompt (every prefix of
    >= 8 tokens is one tensor-core pass whose last row is compared: hidden states, logits) plus the K/V rows of all
    rows of the longest pass."""
    om = oracle.Model.from_datagen(tiny_weights, max_seq=64)
    hid, lg = om.forward(tiny_tokens, hidden="all", logits="all")
    gm = gpu_model(tiny_weights, max_seq=64)
    stats = {}
    for n in range(8, len(tiny_tokens) + 1):
        gm.kv_reset()
        gm.prefill(tiny_tokens[:n])
        check_position(gm, hid[n - 1], lg[n - 1], f"pass of {n} rows, last row", stats)
    check_kv_rows(gm, om, range(len(tiny_tokens)), stats)
    print("tiny tensor-core rows:", stats)


def test_tiny_free_running_matches_teacher_forced(tiny_weights, tiny_tokens):
    """Device-fed greedy decode (what the bench times) emits the oracle's tokens when margins are wide,
    and graph replay / direct launch / no-PDL variants agree bit for bit."""
    import paper_2606_12154_b200 as hq
    om = oracle.Model.from_datagen(tiny_weights, max_seq=64)
    ref = om.greedy(tiny_tokens, 16)
    for family in (0, KERNEL_PER_ROW):
        outs = []
        for flags in (0, hq.FLAG_NO_GRAPH, hq.FLAG_NO_PDL, hq.FLAG_NO_GRAPH | hq.FLAG_NO_PDL):
            gm = gpu_model(tiny_weights, max_seq=64, flags=flags, path=family)
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


@pytest.mark.parametrize("path", PATHS)
def test_tiny_ragged_lengths(tiny_weights, path):
    """Context lengths around the 16/32/64/128 tile and split boundaries of the attention kernels: the
    prompt goes through prefill, then ONE decode step attends over n+1 positions (decode attention)."""
    toks = datagen.tokens(4242, datagen.TINY.vocab, 202)
    om = oracle.Model.from_datagen(tiny_weights, max_seq=256)
    _, lg = om.forward(toks, logits="all")
    gm = gpu_model(tiny_weights, max_seq=256, path=path)
    checked = 0
    for n in (1, 2, 7, 8, 15, 16, 17, 31, 33, 63, 64, 65, 127, 128, 129, 191, 200):
        gm.kv_reset()
        gm.prefill(toks[:n])
        e = rel_l2(gm.decode_logits()[0].cpu().numpy(), lg[n - 1])
        assert e <= TOL_LOGITS, f"prompt length {n}: logits rel-L2 {e:.3e}"
        gm.decode_step(tokens_in=[int(toks[n])])
        e = rel_l2(gm.decode_logits()[0].cpu().numpy(), lg[n])
        assert e <= TOL_LOGITS, f"decode at context {n + 1}: logits rel-L2 {e:.3e}"
        assert max_abs(gm.decode_logits()[0].cpu().numpy(), lg[n]) <= MAXABS_LOGIT
        checked += 1
    assert checked == 17


@pytest.fixture(scope="module")
def tiny_long_reference(tiny_weights):
    """Tiny model, 4,300 positions: the oracle's logits at every position (one pass, seconds)."""
    toks = datagen.tokens(4243, datagen.TINY.vocab, 4300)
    om = oracle.Model.from_datagen(tiny_weights, max_seq=4304)
    hid, lg = om.forward(toks, hidden="all", logits="all")
    return toks, hid, lg, om


@pytest.mark.parametrize("path", PATHS)
def test_tiny_long_context_decode(tiny_weights, tiny_long_reference, path):
    """Decode attention beyond 2,048 cached positions: attn_decode_kernel (kernel-per-row path) then takes more than
    one 128-position tile per split (second mbarrier phase, tile buffer reuse); the attention block takes ring tiles
    beyond its first one.  Contexts straddle the 16 x 128 boundary and the ring-tile boundaries."""
    toks, hid, lg, om = tiny_long_reference
    gm = gpu_model(tiny_weights, max_seq=4304, path=path)
    stats = {}
    for n in (449, 504, 505, 2047, 2048, 2049, 2175, 2290, 4095, 4096, 4097, 4290):
        gm.kv_reset()
        gm.prefill(toks[:n])
        for j in range(3):     # three decode steps at contexts n+1 .. n+3
            gm.decode_step(tokens_in=[int(toks[n + j])])
            check_position(gm, hid[n + j], lg[n + j], f"decode at context {n + j + 1}", stats)
    check_kv_rows(gm, om, (0, 1000, 2047, 2048, 4095, 4290, 4291, 4292), stats)
    print("tiny long-context parity:", stats)


def test_tiny_long_context_batched(tiny_weights, tiny_long_reference):
    """Batched decode (B2: attn_decode_kernel + attn_combine) at > 4,096 cached positions (three 128-position tiles per
    split), and a batched prefill of 2 x 4,150 rows = five tensor-core passes (pass capacity 2,048 rows)."""
    toks, hid, lg, om = tiny_long_reference
    gm = gpu_model(tiny_weights, max_seq=4304, max_batch=2)
    n = 4150
    prompts = np.stack([toks[:n], toks[100:n + 100]])
    om2 = oracle.Model.from_datagen(tiny_weights, max_seq=4304)
    hid2, lg2 = om2.forward(toks[100:n + 104], hidden="all", logits="all")
    gm.prefill(prompts)
    stats = {}
    lgs = gm.decode_logits(batch=2).cpu().numpy()
    check_vectors([gm.get_hidden(l, batch=2)[0].cpu().numpy() for l in range(2)], lgs[0], hid[n - 1], lg[n - 1], "prefill seq 0", stats)
    check_vectors([gm.get_hidden(l, batch=2)[1].cpu().numpy() for l in range(2)], lgs[1], hid2[n - 1], lg2[n - 1], "prefill seq 1", stats)
    for j in range(3):
        gm.decode_step(tokens_in=[int(toks[n + j]), int(toks[100 + n + j])])
        lgs = gm.decode_logits(batch=2).cpu().numpy()
        hs = [gm.get_hidden(l, batch=2).cpu().numpy() for l in range(2)]
        check_vectors([h[0] for h in hs], lgs[0], hid[n + j], lg[n + j], f"seq 0 step {j}", stats)
        check_vectors([h[1] for h in hs], lgs[1], hid2[n + j], lg2[n + j], f"seq 1 step {j}", stats)
    check_kv_rows(gm, om2, (0, 2047, 2048, 4149, 4150, 4152), stats, seq=1)
    print("tiny long-context batched parity:", stats)


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
# 1B model at BASELINE.json's full sizes, in the launch configuration bench.py times.  The oracle runs once per
# config (module-scoped references shared by the decode paths).
# ---------------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def one_b_weights():
    return datagen.make_weights(datagen.ONE_B)


@pytest.fixture(scope="module")
def ref_config1(one_b_weights):
    """configs[1]: 256-token prompt, 128 greedy steps; hidden/logits at every 8th step."""
    return oracle_reference(one_b_weights, datagen.tokens(1001, datagen.ONE_B.vocab, 256), 128, 512, sample_every=8)


@pytest.fixture(scope="module")
def ref_config2(one_b_weights):
    """configs[2]: 2,048-token prompt, all 256 greedy steps; hidden/logits at every 16th step."""
    return oracle_reference(one_b_weights, datagen.tokens(1002, datagen.ONE_B.vocab, 2048), 256, 2304, sample_every=16)


@pytest.mark.parametrize("path", PATHS)
def test_1b_config1_teacher_forced(one_b_weights, ref_config1, path):
    gm = gpu_model(one_b_weights, max_seq=512, path=path)
    stats = run_teacher_forced(gm, ref_config1)
    check_kv_rows(gm, ref_config1["om"], (0, 37, 127, 128, 255, 256, 300, 383), stats)
    frac = float((ref_config1["margins"] > MARGIN).mean())
    print("1b config[1] parity:", stats, "positions with margin>0.1: %.2f" % frac)
    assert stats["argmax_checked"] >= 16 and stats["positions"] == 17


@pytest.mark.parametrize("path", PATHS)
def test_1b_window_131072(one_b_weights, ref_config1, path):
    """PAPER.md:L170 (section 6.6, "context length is free"): the largest window of the paper's sweep, 131,072 positions
    (4 GiB of KV cache, a 32 MiB RoPE table), with the configs[1] query in it: same tolerances, first 16 decode steps."""
    ref = dict(ref_config1)
    ref["n_steps"] = 16
    ref["sampled"] = {i: v for i, v in ref_config1["sampled"].items() if i <= 16}
    gm = gpu_model(one_b_weights, max_seq=131072, path=path)
    stats = {"argmax_checked": 0, "positions": 0}
    tok = gm.prefill(ref["prompt"])
    for i in range(17):
        if i:
            tok = gm.decode_step(tokens_in=[int(ref["tokens"][i - 1])])
        if i in ref["sampled"]:
            check_position(gm, ref["sampled"][i][0], ref["sampled"][i][1], f"step {i}", stats)
            stats["positions"] += 1
        if ref["margins"][i] > MARGIN:
            assert int(tok[0]) == int(ref["tokens"][i])
            stats["argmax_checked"] += 1
    check_kv_rows(gm, ref_config1["om"], (0, 255, 256, 270), stats)
    assert gm.seq_len() == 256 + 16 and stats["positions"] == 3
    print("1b window 131,072 parity:", stats)


def test_tiny_window_131072_high_positions(tiny_weights):
    """Positions deep inside a 131,072 window: the tiny model's oracle walks 9,000 positions (RoPE angles up to 9,000 rad
    at theta = 1e4), the GPU prefills them in 2,048-row passes and decodes at positions 9,000+ (kernel-per-row and
    attention block: 1,126 cached positions per cluster CTA, 5 ring tiles)."""
    n = 9000
    toks = datagen.tokens(4244, datagen.TINY.vocab, n + 4)
    om = oracle.Model.from_datagen(tiny_weights, max_seq=n + 8)
    hid, lg = om.forward(toks, hidden="all", logits="all")
    for path in (0, KERNEL_PER_ROW):
        gm = gpu_model(tiny_weights, max_seq=131072, path=path)
        gm.prefill(toks[:n])
        stats = {}
        check_position(gm, hid[n - 1], lg[n - 1], "prefill", stats)
        for j in range(3):
            gm.decode_step(tokens_in=[int(toks[n + j])])
            check_position(gm, hid[n + j], lg[n + j], f"decode at position {n + j}", stats)
        check_kv_rows(gm, om, (0, 4095, 8999, 9000, 9002), stats)
        print("tiny window 131,072, positions 9,000+:", stats)


@pytest.mark.parametrize("path", PATHS)
def test_1b_config2_long_context(one_b_weights, ref_config2, path):
    """configs[2] at full size and full length: 2,048-token prompt (one tensor-core pass, causal flash attention over
    32 query tiles), then all 256 teacher-forced decode steps at contexts 2,049..2,304 — the attention block streams
    ring tiles beyond its first one, attn_decode_kernel (kernel-per-row) two 128-position tiles per split."""
    gm = gpu_model(one_b_weights, max_seq=2304, path=path)
    stats = run_teacher_forced(gm, ref_config2)
    check_kv_rows(gm, ref_config2["om"], (0, 1023, 2047, 2048, 2303), stats)
    print("1b config[2] parity:", stats)
    assert stats["argmax_checked"] >= 32 and stats["positions"] == 17


# ---------------------------------------------------------------------------------------------------
# batched serving (configs[3], configs[4]): tensor-core prefill + batched decode
# ---------------------------------------------------------------------------------------------------
def run_batched(gm, weights, prompts, n_steps, max_seq, sample_every=1, check_seqs=None):
    """Every CHECKED sequence is run alone through the oracle (reading 17); the GPU runs all of them as one batch.
    Checked sequences are teacher-forced with the oracle's tokens, the others are fed the GPU's own (sequences are
    independent, so what the neighbours are fed cannot matter)."""
    B, T = prompts.shape
    check_seqs = list(range(B)) if check_seqs is None else list(check_seqs)
    refs = {b: oracle_reference(weights, prompts[b], n_steps, max_seq, sample_every) for b in check_seqs}
    stats = {"argmax_checked": 0, "positions": 0}
    L = weights.shape.n_layers

    def check(i, toks):
        if any(i in refs[b]["sampled"] for b in check_seqs):
            lg = gm.decode_logits(batch=B).cpu().numpy()
            hid = [gm.get_hidden(l, batch=B).cpu().numpy() for l in range(L)]
            for b in check_seqs:
                h_ref, lg_ref = refs[b]["sampled"][i]
                check_vectors([hid[l][b] for l in range(L)], lg[b], h_ref, lg_ref, f"seq {b} step {i}", stats)
                stats["positions"] += 1
        for b in check_seqs:
            if refs[b]["margins"][i] > MARGIN:
                assert int(toks[b]) == int(refs[b]["tokens"][i]), f"seq {b} step {i}"
                stats["argmax_checked"] += 1

    toks = gm.prefill(prompts)
    check(0, toks)
    for i in range(1, n_steps + 1):
        feed = [int(refs[b]["tokens"][i - 1]) if b in refs else int(toks[b]) for b in range(B)]
        toks = gm.decode_step(tokens_in=feed)[:B].copy()
        check(i, toks)
    assert gm.seq_len() == T + n_steps
    return refs, stats


def test_tiny_batched_prefill_and_decode(tiny_weights):
    B, T, steps = 3, 24, 10
    prompts = datagen.tokens(1003, datagen.TINY.vocab, B * T).reshape(B, T)
    gm = gpu_model(tiny_weights, max_seq=64, max_batch=4)
    refs, stats = run_batched(gm, tiny_weights, prompts, steps, 64)
    for b in range(B):
        check_kv_rows(gm, refs[b]["om"], range(0, T + steps, 5), stats, seq=b)
    print("tiny batched parity:", stats)
    assert stats["argmax_checked"] >= B * 4


def test_tiny_batch32(tiny_weights):
    """max_batch = 32 (the widest token tile of batched decode), every sequence checked."""
    B, T, steps = 32, 40, 4
    prompts = datagen.tokens(1006, datagen.TINY.vocab, B * T).reshape(B, T)
    gm = gpu_model(tiny_weights, max_seq=64, max_batch=32)
    refs, stats = run_batched(gm, tiny_weights, prompts, steps, 64)
    print("tiny batch-32 parity:", stats)
    assert stats["positions"] == B * (steps + 1)


@pytest.mark.parametrize("B", [8, 9, 16])
def test_tiny_batch_token_tiles(tiny_weights, B):
    """Batched decode with <= 8 / <= 16 sequences runs its GEMMs on 8- / 16-row token tiles (a full 8-row tile, a ragged and a
    full 16-row tile; tiny ffn = 688 keeps the two-accumulator SwiGLU form on 32 rows); every sequence checked, and the K/V
    rows that the one-launch decode attention appends."""
    T, steps = 30, 6
    prompts = datagen.tokens(1010 + B, datagen.TINY.vocab, B * T).reshape(B, T)
    gm = gpu_model(tiny_weights, max_seq=64, max_batch=B)
    refs, stats = run_batched(gm, tiny_weights, prompts, steps, 64)
    for b in (0, B - 1):
        check_kv_rows(gm, refs[b]["om"], range(T - 2, T + steps), stats, seq=b)
    print(f"tiny batch-{B} parity:", stats)
    assert stats["positions"] == B * (steps + 1)


@pytest.mark.parametrize("n_heads,n_kv_heads", [(4, 4), (8, 1), (6, 2)])
def test_gqa_group_sizes_batched(n_heads, n_kv_heads):
    """Group sizes other than the models' (G = 1: plain multi-head attention, one warp per CTA of the decode attention;
    G = 8: the widest CTA; G = 3): batched prefill + decode against the oracle, every sequence, and the appended K/V rows."""
    import dataclasses
    import paper_2606_12154_b200 as hq
    shape = dataclasses.replace(datagen.TINY, name=f"tiny-h{n_heads}-kv{n_kv_heads}", n_heads=n_heads, n_kv_heads=n_kv_heads)
    weights = datagen.make_weights(shape, seed=datagen.WEIGHT_SEED + n_heads)
    B, T, steps = 3, 20, 5
    prompts = datagen.tokens(1020 + n_heads, shape.vocab, B * T).reshape(B, T)
    gm = hq.Model.from_bf16_bits(shape, weights.embedding, weights.final_norm, weights.layers, max_seq=64, max_batch=4,
                                 flags=hq.FLAG_CAPTURE_HIDDEN)
    refs, stats = run_batched(gm, weights, prompts, steps, 64)
    for b in range(B):
        check_kv_rows(gm, refs[b]["om"], range(T - 1, T + steps), stats, seq=b)
    print(f"GQA {n_heads}/{n_kv_heads} batched parity:", stats)
    assert stats["positions"] == B * (steps + 1)


def test_1b_config3_batch8(one_b_weights):
    """configs[3] at full size and full length: 8 sequences x 192-token prompts in one tensor-core pass (1,536 rows),
    then all 192 batched decode steps (tcgen05 GEMMs with a 32-token tile); hidden/logits every 16th step, argmax at
    every step of margin > 0.1, for every sequence."""
    s = datagen.ONE_B
    B, T, steps = 8, 192, 192
    prompts = datagen.tokens(1003, s.vocab, B * T).reshape(B, T)
    gm = gpu_model(one_b_weights, max_seq=T + steps, max_batch=B)
    refs, stats = run_batched(gm, one_b_weights, prompts, steps, T + steps, sample_every=16)
    check_kv_rows(gm, refs[B - 1]["om"], (0, 191, 192, 383), stats, seq=B - 1)
    print("1b config[3] parity:", stats)
    assert stats["argmax_checked"] >= 8 * 24 and stats["positions"] == 8 * 13


def test_1b_config4_batch32_ctx512(one_b_weights):
    """configs[4] corner: batch 32 x context 512 (16,384 prompt rows = 8 tensor-core passes), then 3 batched decode
    steps.  Sampled: the oracle runs sequences 0 and 31."""
    s = datagen.ONE_B
    B, T, steps = 32, 512, 3
    prompts = datagen.tokens(1004, s.vocab, B * T).reshape(B, T)
    gm = gpu_model(one_b_weights, max_seq=T + 8, max_batch=B)
    refs, stats = run_batched(gm, one_b_weights, prompts, steps, T + 8, check_seqs=(0, B - 1))
    check_kv_rows(gm, refs[B - 1]["om"], (0, 255, 511, 512, 514), stats, seq=B - 1)
    print("1b config[4] B=32 ctx=512 parity:", stats)
    assert stats["positions"] == 2 * (steps + 1)


@pytest.fixture(scope="module")
def ref_ctx4096(one_b_weights):
    """configs[4] corner, context 4,096: one 4,096-token prompt + 3 greedy steps (the oracle's attention is a plain
    double loop: ~4 minutes of CPU for this one sequence, so it is shared by the three tests below)."""
    s = datagen.ONE_B
    prompt = datagen.tokens(1005, s.vocab, 4096)
    return oracle_reference(one_b_weights, prompt, 3, 4104)


@pytest.mark.parametrize("path", PATHS)
def test_1b_config4_batch1_ctx4096(one_b_weights, ref_ctx4096, path):
    """Batch 1 at context 4,096: the prompt is two tensor-core passes (pass capacity 2,048 rows), decode attention
    reads 4,097+ cached positions (attention block: 512 per CTA = its first tile + 2 ring tiles; attn_decode_kernel:
    3 tiles per split)."""
    gm = gpu_model(one_b_weights, max_seq=4104, path=path)
    stats = run_teacher_forced(gm, ref_ctx4096)
    check_kv_rows(gm, ref_ctx4096["om"], (0, 2047, 2048, 4095, 4096, 4098), stats)
    print("1b config[4] B=1 ctx=4096 parity:", stats)
    assert stats["positions"] == 4


def test_1b_config4_batch2_ctx4096(one_b_weights, ref_ctx4096):
    """Batched decode at context 4,096 (attn_decode_kernel: three 128-position tiles per split, B2) after a batched
    prefill of 8,192 rows (4 passes).  Both sequences carry the same prompt and are held to the one oracle run (that
    neighbours do not leak into one another is what test_1b_config3_batch8, test_1b_config4_batch32_ctx512 and
    test_tiny_long_context_batched check with distinct prompts)."""
    ref = ref_ctx4096
    gm = gpu_model(one_b_weights, max_seq=4104, max_batch=2)
    stats = {"argmax_checked": 0, "positions": 0}
    toks = gm.prefill(np.stack([ref["prompt"], ref["prompt"]]))
    L = datagen.ONE_B.n_layers
    for i in range(4):
        if i:
            toks = gm.decode_step(tokens_in=[int(ref["tokens"][i - 1])] * 2)[:2].copy()
        lg = gm.decode_logits(batch=2).cpu().numpy()
        hid = [gm.get_hidden(l, batch=2).cpu().numpy() for l in range(L)]
        for b in range(2):
            check_vectors([hid[l][b] for l in range(L)], lg[b], ref["sampled"][i][0], ref["sampled"][i][1],
                          f"seq {b} step {i}", stats)
            stats["positions"] += 1
            if ref["margins"][i] > MARGIN:
                assert int(toks[b]) == int(ref["tokens"][i])
                stats["argmax_checked"] += 1
    check_kv_rows(gm, ref["om"], (0, 2048, 4095, 4098), stats, seq=1)
    print("1b config[4] B=2 ctx=4096 parity:", stats)


def test_workspace_guards(tiny_weights, tiny_tokens):
    """compute-sanitizer is closed on this pool (profiles/r02_sanitizers.md), so out-of-bounds WRITES are looked for
    directly: 1 MiB canary regions in front of and behind the workspace must survive every path — tensor-core prefill
    (single and multi-pass), both batch-1 decode paths up to the last cache slot, batched decode at max_batch, the
    dense verification pass."""
    import paper_2606_12154_b200 as hq
    w = tiny_weights
    for path in (0, KERNEL_PER_ROW):
        gm = hq.Model.from_bf16_bits(w.shape, w.embedding, w.final_norm, w.layers, max_seq=80, max_batch=4,
                                     flags=hq.FLAG_CAPTURE_HIDDEN | hq.FLAG_VERIFY | path, guard_bytes=1 << 20)
        gm.prefill(tiny_tokens)
        gm.decode_run(48)                                   # fills the cache to its last slot (32 + 48 = 80)
        assert gm.seq_len() == 80 and gm.guards_intact()
        gm.kv_reset()
        gm.prefill(np.stack([tiny_tokens] * 4))
        gm.decode_run(48, batch=4)
        assert gm.guards_intact()
        gm.kv_reset()
        gm.verify_relay(tiny_tokens[:20], tiny_tokens[20:])
        assert gm.guards_intact()
    big = hq.Model.from_bf16_bits(w.shape, w.embedding, w.final_norm, w.layers, max_seq=4200, max_batch=2, guard_bytes=1 << 20)
    big.prefill(datagen.tokens(7, datagen.TINY.vocab, 2 * 4190).reshape(2, 4190))     # five tensor-core passes
    big.decode_run(10, batch=2)
    assert big.seq_len() == 4200 and big.guards_intact()


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


def test_large_magnitude_activations(tiny_weights):
    """ADVICE (round 1): the fp16 vectors between kernels (KV cache, SwiGLU vector) must not overflow on outlier
    activations.  The tiny model with W_gate x256, W_up x512 and W_v x16 pushes the SwiGLU vector past the fp16 range
    (|a| up to ~1e5 > 65,504) and the cached V rows to O(100); results stay finite and within tolerance of the oracle."""
    import copy
    w = copy.deepcopy(tiny_weights)
    scale = {"w_gate": 256.0, "w_up": 512.0, "wv": 16.0}
    for l in range(w.shape.n_layers):
        for k, f in scale.items():
            v = datagen.bf16_bits_to_f32(w.layers[l][k]) * f     # power of two: exact in bf16
            w.layers[l][k] = datagen.f32_to_bf16_bits(v)
    toks = datagen.tokens(1007, datagen.TINY.vocab, 24)
    om = oracle.Model.from_datagen(w, max_seq=32)
    ref = om.greedy(toks, 4, hidden="last")
    assert np.abs(ref["hidden"]).max() > 1e3      # the case really has large activations
    for path in (0, KERNEL_PER_ROW):
        gm = gpu_model(w, max_seq=32, path=path)
        gm.prefill(toks)
        for i in range(5):
            if i:
                gm.decode_step(tokens_in=[int(ref["tokens"][i - 1])])
            lg = gm.decode_logits()[0].cpu().numpy()
            assert np.isfinite(lg).all()
            assert rel_l2(lg, ref["logits"][i]) <= TOL_LOGITS, (path, i, rel_l2(lg, ref["logits"][i]))


# ---------------------------------------------------------------------------------------------------
# verbatim-relay verification in one dense pass (hq_verify_relay)
# ---------------------------------------------------------------------------------------------------
def test_tiny_verify_relay(tiny_weights):
    """The oracle's own greedy continuation is the 'answer line': one dense pass accepts all of it; a corrupted token
    stops the acceptance exactly there, and streaming decode continues from the model's own token.  Envelope seed 2003:
    every oracle margin of the continuation is > 0.6, so the argmax decisions are not rounding-sensitive."""
    import paper_2606_12154_b200 as hq
    V = datagen.TINY.vocab
    env = datagen.tokens(2003, V, 24)
    om = oracle.Model.from_datagen(tiny_weights, max_seq=64)
    ref = om.greedy(env, 20)
    assert ref["margins"].min() > MARGIN
    answer = ref["tokens"][:16]
    for path in (0, KERNEL_PER_ROW):
        gm = gpu_model(tiny_weights, max_seq=64, flags=hq.FLAG_CAPTURE_HIDDEN | hq.FLAG_VERIFY, path=path)
        # (a) everything accepted; the waiting token is the model's choice after the whole answer
        assert gm.verify_relay(env, answer) == 16
        assert gm.seq_len() == 24 + 16
        lg = gm.decode_logits()[0].cpu().numpy()
        assert rel_l2(lg, ref["logits"][16]) <= TOL_LOGITS and max_abs(lg, ref["logits"][16]) <= MAXABS_LOGIT
        assert int(gm.decode_step()[0]) == int(ref["tokens"][17]) and int(gm.decode_step()[0]) == int(ref["tokens"][18])
        # (b) a wrong token at answer position 5: five accepted, streaming resumes with the model's own token 5
        bad = answer.copy()
        bad[5] = (bad[5] + 1) % V
        gm.kv_reset()
        assert gm.verify_relay(env, bad) == 5
        assert gm.seq_len() == 24 + 5
        lg = gm.decode_logits()[0].cpu().numpy()
        assert rel_l2(lg, ref["logits"][5]) <= TOL_LOGITS
        out = [int(gm.decode_step()[0]) for _ in range(4)]
        assert out == [int(t) for t in ref["tokens"][6:10]], (out, ref["tokens"][6:10])
        assert gm.seq_len() == 24 + 5 + 4
        # (c) appended to a cache that already holds the head of the envelope (chunked), first token wrong -> 0 accepted
        gm.kv_reset()
        gm.prefill(env[:10])
        bad0 = answer.copy()
        bad0[0] = (bad0[0] + 7) % V
        assert gm.verify_relay(env[10:], bad0) == 0 and gm.seq_len() == 24
        assert int(gm.decode_step()[0]) == int(ref["tokens"][1])
        # the cached rows of envelope + accepted prefix are the oracle's
        check_kv_rows(gm, om, (0, 9, 10, 23, 24), {})
    with pytest.raises(hq.HQError) as e:
        gpu_model(tiny_weights, max_seq=64).verify_relay(env, answer)
    assert e.value.code == -3          # model created without HQ_FLAG_VERIFY


def test_1b_verify_relay(one_b_weights, ref_config1):
    """configs[1] shape: 256-token envelope + the oracle's first 100 greedy tokens as the answer line, verified in one
    dense pass (356 rows through the tcgen05 GEMMs, LM head over 101 positions)."""
    import paper_2606_12154_b200 as hq
    ref = ref_config1
    answer = ref["tokens"][:100]
    wide = ref["margins"][:101] > MARGIN
    first_narrow = int(np.argmin(wide)) if not wide.all() else 101      # first answer position the GPU may legitimately miss
    gm = gpu_model(one_b_weights, max_seq=512, flags=hq.FLAG_VERIFY)
    acc = gm.verify_relay(ref["prompt"], answer)
    assert acc >= min(first_narrow, 100), (acc, first_narrow)
    if acc in ref["sampled"]:
        assert rel_l2(gm.decode_logits()[0].cpu().numpy(), ref["sampled"][acc][1]) <= TOL_LOGITS
    # corrupt a position in front of the first narrow margin: acceptance stops exactly there
    j = min(first_narrow, 100) - 1
    if j >= 1:
        bad = answer.copy()
        bad[j] = (bad[j] + 1) % datagen.ONE_B.vocab
        gm.kv_reset()
        assert gm.verify_relay(ref["prompt"], bad) == j
        assert gm.seq_len() == 256 + j
        assert int(gm.decode_step()[0]) == int(ref["tokens"][j + 1]) or ref["margins"][j + 1] <= MARGIN
    print("1b verify relay: accepted", acc, "of 100; first narrow margin at", first_narrow)
