#!/usr/bin/env python
"""bench.py — headline benchmark of the hq hot path on B200.

Metric (BASELINE.json): batch-1 decode tokens/s of the 1B bf16 model (as a fraction of the HBM
roofline), with envelope-prefill TTFT next to it.  Workload = BASELINE.json configs[1]: 256-token
random prompt, then 128 greedy decode steps.  One bench "step" = one whole query (kv_reset, prefill,
128 decode steps).  See DESIGN.md "Measurement" for the byte model behind the roofline object.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl hq|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
        --master-port P bench.py --gpus N --steps K --warmup W

N > 1 runs N independent replicas (no collective on the data path).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

PROMPT_LEN, DECODE_STEPS = 256, 128
METRIC, UNIT = "decode_tokens_per_s_batch1_1b_bf16", "tokens/s"
WORKLOAD = "configs[1]: 1B Llama-style bf16, batch 1, 256-token random prompt, 128 greedy decode steps"
FALLBACK_HBM_GBS = 6650.0  # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


def weight_bytes(s) -> int:
    return 2 * s.n_params


def bytes_per_token(s, ctx: int, batch: int = 1) -> int:
    """Algorithmic HBM bytes of one decode step: weights once + embedding row +
    KV read of ctx cached tokens and write of one; 2*Hkv*hd*2 B*L per cached token."""
    kv_tok = 2 * s.n_kv_heads * s.head_dim * 2 * s.n_layers
    return weight_bytes(s) + batch * 2 * s.hidden + batch * (ctx + 1) * kv_tok


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_numbers():
    """Per-launch figures copied from the committed ncu --set full summaries (profiles/roofline_traffic.json): DRAM
    bytes and the serialised (no PDL overlap, cold) duration of the decode kernels."""
    p = os.path.join(ROOT, "profiles", "roofline_traffic.json")
    if os.path.exists(p):
        try:
            return json.load(open(p))
        except Exception:
            return {}
    return {}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons during the timed region (NVML; nvidia-smi fields)."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self.mem, self.power = [], []
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                self.mem.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_MEM))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.05)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons)}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples),
                "mem_mhz": float(np.median(self.mem)) if self.mem else None,
                "power_w_median": float(np.median(self.power)) if self.power else None,
                "power_w_max": float(np.max(self.power)) if self.power else None}


def aggregate_over_ranks(dist, dev, dec_total_ms, total_ms, ttft_ms, launches):
    """N independent replicas: the job's time is the slowest rank's, its launch
    count the sum.  dist = torch.distributed or None (single process); tensors live on dev (cuda for nccl, cpu for gloo)."""
    if dist is None:
        return dec_total_ms, total_ms, ttft_ms, launches
    import torch
    t = torch.tensor([dec_total_ms, total_ms, ttft_ms], device=dev, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ln = torch.tensor([launches], device=dev, dtype=torch.int64)
    dist.all_reduce(ln)
    a, b, c = [float(v) for v in t.tolist()]
    return a, b, c, int(ln.item())


def job_tokens_per_s(world, steps, dec_total_ms):
    """Whole-job decode throughput: tokens of all replicas / the slowest replica's decode time."""
    return world * steps * DECODE_STEPS / (dec_total_ms * 1e-3)


def oracle_sample(weights, s, prompt_len=16, steps=24):
    """cpu_baseline: the oracle as it stands on the host cores, on a bounded sample of the workload."""
    import datagen
    import oracle
    om = oracle.Model.from_datagen(weights, max_seq=prompt_len + steps + 1)
    prompt = datagen.tokens(1001, s.vocab, prompt_len)
    t0 = time.perf_counter()
    _, lg = om.forward(prompt, logits="last")
    t1 = time.perf_counter()
    tok = oracle.argmax(lg)
    for _ in range(steps):
        _, lg = om.forward([tok], logits="last")
        tok = oracle.argmax(lg)
    t2 = time.perf_counter()
    return {"value": steps / (t2 - t1), "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"same 1B weights; {prompt_len}-token prompt (prefill {t1 - t0:.2f} s, "
                      f"{prompt_len / (t1 - t0):.1f} tok/s) then {steps} greedy decode steps at context "
                      f"{prompt_len + 1}..{prompt_len + steps} ({(t2 - t1) / steps * 1e3:.0f} ms/token); the workload's context "
                      f"is 257..384 - the oracle is weight-bound, so its rate barely depends on it (full configs[1] "
                      f"timing: profiles/r02_oracle_full_config1.md)"}


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import datagen
    import oracle
    s = datagen.ONE_B
    w = datagen.make_weights(s)
    prompt_len, steps = (PROMPT_LEN, DECODE_STEPS) if args.full_config1 else (8, 8)  # default: bounded sample of the workload per bench step
    om = oracle.Model.from_datagen(w, max_seq=prompt_len + steps + 1)
    prompt = datagen.tokens(1001, s.vocab, prompt_len)

    def one():
        om.reset()
        t0 = time.perf_counter()
        _, lg = om.forward(prompt, logits="last")
        t1 = time.perf_counter()
        tok = oracle.argmax(lg)
        for _ in range(steps):
            _, lg = om.forward([tok], logits="last")
            tok = oracle.argmax(lg)
        return t1 - t0, time.perf_counter() - t1

    for _ in range(args.warmup):
        one()
    tp = td = 0.0
    for _ in range(args.steps):
        a, b = one()
        tp += a
        td += b
    value = args.steps * steps / td
    sample = (f"per step: {prompt_len}-token prompt + {steps} greedy decode steps (context {prompt_len + 1}.."
              f"{prompt_len + steps}) of the same 1B weights " +
              ("(the whole of configs[1])" if args.full_config1 else "(bounded sample of configs[1], whose context is 257..384)"))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": (tp + td) / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": WORKLOAD, "sample": sample},
            "ttft_ms": tp / args.steps * 1e3,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="hq", choices=["hq", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg")
    ap.add_argument("--full-config1", action="store_true",
                    help="with --impl reference: time the oracle on the whole of configs[1] (256-token prompt + 128 steps) per step")
    ap.add_argument("--sweep", action="store_true",
                    help="configs[4]: batch {1,4,16,32} x context {512,4096}, 128 decode steps each; one JSON line per point")
    ap.add_argument("--q4", action="store_true",
                    help="SURVEY 8(f)-1: the configs[1] query with the FFN and LM-head matrices streamed as 4-bit hq4 (hq_model_create_q4)")
    ap.add_argument("--runtime", action="store_true",
                    help="SURVEY 8(f)-3: the whole runtime path per query on the synthetic 563-entry store (route, gate, render, "
                         "tokenise, prefill, streaming decode): e2e wall, e2e tok/s, TTFT, route p50 as PAPER.md:L109 defines them")
    ap.add_argument("--window-sweep", action="store_true",
                    help="PAPER.md:L170 (section 6.6): context WINDOW 4,096 -> 131,072 with the configs[1] query; one JSON line per window")
    ap.add_argument("--gemm-timeline", action="store_true",
                    help="globaltimer stamps inside the tcgen05 GEMM (hq_debug_gemm_timeline) for the 1B prefill and batched-decode shapes; JSON lines")
    ap.add_argument("--probes", action="store_true",
                    help="memory-system probes behind the kernel design: bulk-copy size vs per-SM rate, read-only stream; JSON lines")
    ap.add_argument("--profile", type=int, default=0, metavar="N",
                    help="ncu helper: one prefill + N decode steps of the bench workload, no timing")
    ap.add_argument("--profile-batch", type=int, default=1, metavar="B",
                    help="with --profile: B sequences of the configs[3] shape (192-token prompts) instead of the batch-1 query")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import datagen
    import paper_2606_12154_b200 as hq

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
    dev = torch.device(f"cuda:{local_rank}")
    torch.cuda.set_device(dev)

    s = datagen.ONE_B
    weights = datagen.make_weights(s)
    max_seq = 1024 if args.runtime else PROMPT_LEN + DECODE_STEPS + 32
    gm = hq.Model.from_bf16_bits(s, weights.embedding, weights.final_norm, weights.layers, max_seq=max_seq,
                                 device=str(dev))
    prompt = datagen.tokens(1001, s.vocab, PROMPT_LEN)
    stream = gm.stream       # the stream libhq launches on (CUDA events must be recorded there)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    ev = lambda: torch.cuda.Event(enable_timing=True)

    def query(events=None):
        """One bench step on the device-resident path: async greedy decode, tokens stay on the GPU."""
        gm.kv_reset()
        if events:
            events[0].record(stream)
        gm.prefill(prompt, want_token=False)
        if events:
            events[1].record(stream)
        gm.decode_run(DECODE_STEPS, want_tokens=False)
        if events:
            events[2].record(stream)

    if args.sweep:
        # BASELINE.json configs[4] (and the shapes of configs[2], [3]): tokens/s, per-token latency and algorithmic HBM GB/s
        peak, _ = measured_peak()
        lay = gm.weight_tensors()
        points = [(B, ctx, 128, "configs[4]") for B in (1, 4, 16, 32) for ctx in (512, 4096)]
        points += [(1, 2048, 256, "configs[2]"), (8, 192, 192, "configs[3]")]
        for B, ctx, steps, cfg_name in points:
            if True:   # (indentation kept: one model per point)
                m = hq.Model(hq.binding.make_config(n_layers=s.n_layers, hidden=s.hidden, n_heads=s.n_heads, n_kv_heads=s.n_kv_heads,
                                            head_dim=s.head_dim, ffn=s.ffn, vocab=s.vocab, rms_eps=s.rms_eps,
                                            rope_theta=s.rope_theta, max_batch=B, max_seq=ctx + steps + 8, flags=0), *lay)
                pr = datagen.tokens(1004, s.vocab, B * ctx).reshape(B, ctx)
                ms, pf = [], []
                sampler = ClockSampler(local_rank)
                sampler.start()
                for it in range(3):
                    m.kv_reset()
                    a, b, c2 = ev(), ev(), ev()
                    a.record(m.stream)
                    m.prefill(pr, want_token=False)
                    b.record(m.stream)
                    m.decode_run(steps, want_tokens=False, batch=B)
                    c2.record(m.stream)
                    torch.cuda.synchronize(dev)
                    if it:
                        pf.append(a.elapsed_time(b))
                        ms.append(b.elapsed_time(c2))
                clk = sampler.stop()
                step_ms = float(np.mean(ms)) / steps
                bpt = bytes_per_token(s, ctx + steps // 2, B)
                print(json.dumps({"sweep": True, "config": cfg_name, "batch": B, "context": ctx, "decode_steps": steps,
                                  "clocks": clk,
                                  "tokens_per_s": B / (step_ms * 1e-3), "ms_per_step": step_ms,
                                  "prefill_ms": float(np.mean(pf)), "prefill_tokens_per_s": B * ctx / (float(np.mean(pf)) * 1e-3),
                                  "bytes_per_step": bpt, "GBps": bpt / (step_ms * 1e-3) / 1e9,
                                  "frac_of_measured_peak": bpt / (step_ms * 1e-3) / 1e9 / peak}), flush=True)
                m.close()
                del m
                torch.cuda.empty_cache()
        return

    if args.q4:
        # the paper's mouth runs at 4-bit.  Same query as the headline, FFN + LM head as hq4 (4.25 bits per
        # weight), attention weights bf16: algorithmic bytes per token = hq4 bytes + bf16 attention / norm bytes + embedding row + KV
        del gm
        torch.cuda.empty_cache()
        qm = hq.Model.from_bf16_bits_q4(s, weights.embedding, weights.final_norm, weights.layers, max_seq=max_seq, device=str(dev))
        qd = s.n_heads * s.head_dim
        attn_bytes = s.n_layers * 2 * (qd * s.hidden + 2 * s.n_kv_heads * s.head_dim * s.hidden + s.hidden * qd + 2 * s.hidden) + 2 * s.hidden
        q4_weights = s.n_layers * 3 * s.ffn * s.hidden + s.vocab * s.hidden
        q4_bytes = q4_weights // 2 + q4_weights // 32
        kv_tok = 2 * s.n_kv_heads * s.head_dim * 2 * s.n_layers
        bpt = attn_bytes + q4_bytes + 2 * s.hidden + (PROMPT_LEN + DECODE_STEPS // 2 + 1) * kv_tok
        dec, pf = [], []
        sampler = ClockSampler(local_rank)
        sampler.start()
        for it in range(3 + args.steps):
            qm.kv_reset()
            a, b, c2 = ev(), ev(), ev()
            a.record(qm.stream)
            qm.prefill(prompt, want_token=False)
            b.record(qm.stream)
            qm.decode_run(DECODE_STEPS, want_tokens=False)
            c2.record(qm.stream)
            torch.cuda.synchronize(dev)
            if it >= 3:
                pf.append(a.elapsed_time(b))
                dec.append(b.elapsed_time(c2))
        clk = sampler.stop()
        kernels = {}
        qm.kv_reset(); qm.prefill(prompt, want_token=False); qm.sync()
        for which, name in ((0, "gate_up"), (1, "lm_head"), (4, "down"), (6, "attn_block")):
            r = 16 if which == 1 else 128
            qm.bench_kernel(which, 8)
            a, b = ev(), ev()
            a.record(qm.stream)
            nbytes = qm.bench_kernel(which, r)
            b.record(qm.stream)
            torch.cuda.synchronize(dev)
            ms = a.elapsed_time(b) / r
            kernels[name] = {"us": ms * 1e3, "GBps": nbytes / ms / 1e6, "bytes_per_launch": nbytes}
        peak, _ = measured_peak()
        ms_tok = float(np.mean(dec)) / DECODE_STEPS
        print(json.dumps({"q4": True, "workload": WORKLOAD + "; FFN and LM head as hq4 (4.25 bits per weight), attention weights bf16",
                          "tokens_per_s": 1e3 / ms_tok, "ms_per_token": ms_tok, "ttft_ms": float(np.mean(pf)),
                          "bytes_per_token": bpt, "achieved_GBps": bpt / (ms_tok * 1e-3) / 1e9,
                          "frac_of_measured_peak": bpt / (ms_tok * 1e-3) / 1e9 / peak,
                          "weight_bytes_q4_model": attn_bytes + q4_bytes, "weight_bytes_bf16_model": weight_bytes(s),
                          "kernels_alone": kernels, "clocks": clk, "decode_path": qm.decode_path()}), flush=True)
        return

    if args.runtime:
        # PAPER.md:L109 (section 6.2): end-to-end throughput = tokens of the final answer / total wall time including
        # routing, retrieval and one prompt evaluation; decode rate = streaming speed once it begins; TTFT = time to first
        # token.  (No HTTP server here: the paper's "HTTP overhead" share of its 518 ms is not reproduced.)
        from datagen import store as ds
        from paper_2606_12154_b200 import build as hq_build, hostlib
        hq_build.build_host()
        keys, answers, queries, targets = ds.make_store()
        S = hostlib.Store(keys, answers)
        vm = hq.Model(gm.cfg_with_flags(hq.FLAG_VERIFY), *gm.weight_tensors())
        header = "relay the line after the marker verbatim .\n"
        out = np.empty(1, dtype=np.int32)
        rec = {k: [] for k in ("route_us", "ttft_ms", "wall_ms", "n_answer", "decode_ms", "verify_wall_ms", "n_prompt")}
        escalated = top1 = 0
        for rep in range(2):          # first sweep of 64 queries warms everything up
            qs = list(zip(queries, targets))[:64] if rep == 0 else list(zip(queries, targets))
            for q, target in qs:
                t0 = time.perf_counter()
                ids, sc = S.route(q, 3)
                t1 = time.perf_counter()
                ok, _ = hostlib.gate(sc[0], sc[1])
                if rep:
                    top1 += int(ids[0] == target)
                if not ok:
                    escalated += rep
                    continue
                line = S.render(int(ids[0]))
                env = hostlib.tokenize(header + line, s.vocab)
                ans = hostlib.tokenize(answers[int(ids[0])], s.vocab)
                gm.kv_reset()
                gm.prefill(env, want_token=True)                      # H2D envelope, first token back on the host
                t2 = time.perf_counter()
                for _ in range(len(ans) - 1):
                    gm.decode_step(want_token=True, out=out)          # streaming: one sync + 4-byte D2H per token
                t3 = time.perf_counter()
                # the same query with the answer line verified in one dense pass (hq_verify_relay)
                vm.kv_reset()
                t4 = time.perf_counter()
                vm.verify_relay(env, ans)
                t5 = time.perf_counter()
                if rep:
                    rec["route_us"].append((t1 - t0) * 1e6); rec["ttft_ms"].append((t2 - t0) * 1e3)
                    rec["wall_ms"].append((t3 - t0) * 1e3); rec["n_answer"].append(len(ans)); rec["n_prompt"].append(len(env))
                    rec["decode_ms"].append((t3 - t2) * 1e3); rec["verify_wall_ms"].append((t5 - t4 + t1 - t0) * 1e3)
        r = {k: np.array(v, dtype=np.float64) for k, v in rec.items()}
        nq = len(queries)
        print(json.dumps({
            "runtime_path": True, "store_entries": len(keys), "queries": nq, "answered": int(r["wall_ms"].size),
            "escalated_frac": escalated / nq, "top1": top1 / nq,
            "route_us_p50": float(np.percentile(r["route_us"], 50)), "route_us_p99": float(np.percentile(r["route_us"], 99)),
            "prompt_tokens_mean": float(r["n_prompt"].mean()), "answer_tokens_mean": float(r["n_answer"].mean()),
            "answer_tokens_max": int(r["n_answer"].max()),
            "ttft_ms_mean": float(r["ttft_ms"].mean()), "ttft_ms_p50": float(np.percentile(r["ttft_ms"], 50)),
            "e2e_wall_ms_mean": float(r["wall_ms"].mean()),
            "e2e_tokens_per_s": float(r["n_answer"].sum() / (r["wall_ms"].sum() * 1e-3)),
            "decode_tokens_per_s": float((r["n_answer"] - 1).sum() / (r["decode_ms"].sum() * 1e-3)),
            "verified_relay": {"e2e_wall_ms_mean": float(r["verify_wall_ms"].mean()),
                               "e2e_tokens_per_s": float(r["n_answer"].sum() / (r["verify_wall_ms"].sum() * 1e-3)),
                               "note": "route + hq_verify_relay(envelope, answer): every answer position scored in one dense pass; "
                                       "the time holds for a verbatim relay (all tokens accepted) - random weights accept none"},
            "paper_context": {"e2e_wall_ms": 518, "e2e_tok_s": 131.4, "decode_tok_s": "226-237", "ttft_ms": "29-62",
                              "route_ms_p50": 2.40, "hardware": "RTX 4060 Laptop 8 GB, 4-bit MiniCPM5-1B, HTTP included (PAPER.md:L111-120, L137)"},
            "note": "synthetic store and queries (datagen/store.py), synthetic tokeniser, random-weight 1B bf16 model; no HTTP layer"}), flush=True)
        return

    if args.window_sweep:
        # "Context length is free": the window (KV capacity, max_seq) grows 32x, the USED context stays the
        # configs[1] query (256-token envelope + 128 tokens); decode rate and TTFT must stay flat, memory grows by 32 KiB per
        # window position (the paper's 4-bit laptop setup: ~22 MiB per 1k positions)
        lay = gm.weight_tensors()
        for window in (4096, 8192, 16384, 32768, 65536, 131072):
            cfg = hq.binding.make_config(n_layers=s.n_layers, hidden=s.hidden, n_heads=s.n_heads, n_kv_heads=s.n_kv_heads,
                                         head_dim=s.head_dim, ffn=s.ffn, vocab=s.vocab, rms_eps=s.rms_eps,
                                         rope_theta=s.rope_theta, max_batch=1, max_seq=window, flags=0)
            m = hq.Model(cfg, *lay)
            dec, pf = [], []
            sampler = ClockSampler(local_rank)
            sampler.start()
            for it in range(5):
                m.kv_reset()
                a, b, c2 = ev(), ev(), ev()
                a.record(m.stream)
                m.prefill(prompt, want_token=False)
                b.record(m.stream)
                m.decode_run(DECODE_STEPS, want_tokens=False)
                c2.record(m.stream)
                torch.cuda.synchronize(dev)
                if it >= 2:
                    pf.append(a.elapsed_time(b))
                    dec.append(b.elapsed_time(c2))
            clk = sampler.stop()
            ws = hq.workspace_bytes(cfg)
            kv_bytes = 2 * s.n_layers * s.n_kv_heads * s.head_dim * 2 * window
            print(json.dumps({"window_sweep": True, "window": window, "tokens_per_s": DECODE_STEPS / (float(np.mean(dec)) * 1e-3),
                              "ttft_ms": float(np.mean(pf)), "workspace_MiB": ws / 2 ** 20, "kv_cache_MiB": kv_bytes / 2 ** 20,
                              "kv_MiB_per_1k_positions": kv_bytes / 2 ** 20 / (window / 1024), "decode_path": m.decode_path(),
                              "clocks": clk}), flush=True)
            m.close()
            del m
            torch.cuda.empty_cache()
        return

    if args.gemm_timeline:
        # Where a GEMM launch spends its time (profiles/r02_launches.md): each shape launched alone over fresh weights (three
        # sets cycled so that they come from HBM), stamps of the CTAs of the first token tile / K split, medians over CTAs.
        shapes = [("prefill gate/up", 2, s.ffn, s.hidden, 256, 128, 1), ("prefill Q|K|V", 0, 3072, s.hidden, 256, 128, 2),
                  ("prefill O", 0, s.hidden, s.hidden, 256, 128, 4), ("prefill down", 0, s.hidden, s.ffn, 256, 128, 4),
                  ("decode B=8 gate/up", 3, s.ffn, s.hidden, 8, 8, 1), ("decode B=8 down", 0, s.hidden, s.ffn, 8, 8, 9),
                  ("decode B=8 LM head", 0, s.vocab, s.hidden, 8, 8, 1),
                  ("decode B=8 gate/up, 32-token tile", 3, s.ffn, s.hidden, 8, 32, 1), ("decode B=8 down, 32-token tile", 0, s.hidden, s.ffn, 8, 32, 9),
                  ("decode B=32 LM head", 0, s.vocab, s.hidden, 32, 32, 1)]
        g = torch.Generator(device=dev).manual_seed(7)
        with torch.cuda.stream(stream):
            for name, mode, N, K, T, tile, splits in shapes:
                nset = 2 if N > 100000 else 3
                ws = [torch.randn(N, K, device=dev, generator=g).mul_(0.02).bfloat16() for _ in range(nset)]
                w2 = [torch.randn(N, K, device=dev, generator=g).mul_(0.02).bfloat16() for _ in range(nset)] if mode >= 2 else [None] * nset
                x = torch.randn(2, T, K, device=dev, generator=g).bfloat16()
                out = (torch.zeros((2, T, N), dtype=torch.bfloat16, device=dev) if mode >= 2
                       else torch.zeros((T, N), dtype=torch.float32, device=dev))
                n_ctas = (N // 64 if mode == 3 else (N + 127) // 128)
                n_ctas += n_ctas & 1 if T > 32 else 0
                tr = torch.zeros((n_ctas, 8), dtype=torch.int64, device=dev)
                for i in range(nset + 1):
                    hq.debug_gemm(mode, ws[i % nset], x, out, w2=w2[i % nset], token_tile=tile, splits=splits, stream=stream, trace=tr)
                torch.cuda.synchronize(dev)
                t = tr.cpu().numpy().astype(np.float64)
                t = t[(t[:, 4] > 0) & (t[:, 1] > 0)]   # CTA pairs: only the leader issues MMAs and stamps [1], [2]
                rel = (t[:, 1:5] - t[:, 0:1]) / 1e3
                kb = ((K + 63) // 64 + splits - 1) // splits
                med = np.median(rel, axis=0)
                print(json.dumps({"gemm_timeline": name, "mode": mode, "n_rows": N, "k": K, "tokens": T, "token_tile": tile, "splits": splits,
                                  "ctas_stamped": int(t.shape[0]), "k_blocks_per_cta": kb,
                                  "first_stage_landed_us": round(float(med[0]), 2), "last_stage_landed_us": round(float(med[1]), 2),
                                  "us_per_k_block": round(float((med[1] - med[0]) / max(kb - 1, 1)), 3),
                                  "accumulator_complete_us": round(float(med[2]), 2), "epilogue_us": round(float(med[3] - med[2]), 2),
                                  "note": "us since the CTA had its barriers and tensor memory; medians over the stamped CTAs"}), flush=True)
                del ws, w2
                torch.cuda.empty_cache()
        return

    if args.probes:
        # what one SM / the chip pulls through cp.async.bulk as a function of the copy size (hq_debug_copy_probe), and the
        # read-only LDG stream (hq_debug_read_probe); 2 GiB buffer, CUDA events on the launching stream
        buf = torch.empty(2 << 30, dtype=torch.uint8, device=dev)
        buf.zero_()
        acc = torch.zeros(1, dtype=torch.int32, device=dev)
        n_sms = torch.cuda.get_device_properties(dev).multi_processor_count
        with torch.cuda.stream(stream):
            for n_ctas in (8, 16, 64, n_sms):
                for copy in (1024, 4096, 16384, 32768, 65536):
                    sub = buf[: (256 << 20) if n_ctas <= 16 else (2 << 30)]
                    hq.copy_probe(sub, copy, n_ctas, stream=stream)
                    a, b = ev(), ev()
                    a.record(stream)
                    for _ in range(3):
                        nb = hq.copy_probe(sub, copy, n_ctas, stream=stream)
                    b.record(stream)
                    torch.cuda.synchronize(dev)
                    gbs = 3 * nb / (a.elapsed_time(b) * 1e-3) / 1e9
                    print(json.dumps({"probe": "bulk_copy", "n_ctas": n_ctas, "copy_bytes": copy, "GBps": gbs,
                                      "GBps_per_sm": gbs / n_ctas}), flush=True)
            hq.read_probe(buf, acc, stream=stream)
            a, b = ev(), ev()
            a.record(stream)
            for _ in range(5):
                hq.read_probe(buf, acc, stream=stream)
            b.record(stream)
            torch.cuda.synchronize(dev)
            print(json.dumps({"probe": "read_only_ldg", "GBps": 5 * buf.numel() / (a.elapsed_time(b) * 1e-3) / 1e9}), flush=True)
        return

    if args.profile and args.profile_batch > 1:
        B = args.profile_batch
        bm = hq.Model(hq.binding.make_config(n_layers=s.n_layers, hidden=s.hidden, n_heads=s.n_heads, n_kv_heads=s.n_kv_heads,
                                             head_dim=s.head_dim, ffn=s.ffn, vocab=s.vocab, rms_eps=s.rms_eps,
                                             rope_theta=s.rope_theta, max_batch=B, max_seq=512, flags=0), *gm.weight_tensors())
        bm.prefill(datagen.tokens(1003, s.vocab, B * 192).reshape(B, 192), want_token=False)
        bm.sync()
        before = bm.kernel_count()
        bm.decode_run(args.profile, want_tokens=False, batch=B)
        bm.sync()
        print(json.dumps({"profile": True, "batch": B, "decode_launches": bm.kernel_count() - before}), flush=True)
        return

    if args.profile:
        gm.kv_reset()
        gm.prefill(prompt, want_token=False)
        gm.sync()
        before = gm.kernel_count()
        gm.decode_run(args.profile, want_tokens=False)
        gm.sync()
        print(json.dumps({"profile": True, "decode_launches": gm.kernel_count() - before,
                          "decode_path": gm.decode_path()}), flush=True)
        return

    for _ in range(max(args.warmup, 3)):
        query()
    barrier()

    # ---- timed region: K whole queries, device timed -------------------------------------------------
    sampler = ClockSampler(local_rank)
    sampler.start()
    evs = [[ev(), ev(), ev()] for _ in range(args.steps)]
    k0 = gm.kernel_count()
    barrier()
    t_start, t_end = ev(), ev()
    t_start.record(stream)
    for i in range(args.steps):
        query(evs[i])
    t_end.record(stream)
    barrier()
    clocks = sampler.stop()
    launches = gm.kernel_count() - k0
    total_ms = t_start.elapsed_time(t_end)
    prefill_ms = [e[0].elapsed_time(e[1]) for e in evs]
    decode_ms = [e[1].elapsed_time(e[2]) for e in evs]

    # ---- e2e: same metric through the C ABI with HOST buffers, streaming one token per call ------------
    # (SURVEY.md 8(d) second pass: per-step sync + 4-byte D2H => true streaming per-token latency, p50 / p99)
    out = np.empty(1, dtype=np.int32)
    e2e_decode_s, e2e_ttft_s, tok_lat_us = [], [], []
    for _ in range(max(1, min(args.steps, 3))):
        gm.kv_reset()
        gm.sync()
        t0 = time.perf_counter()
        gm.prefill(prompt, want_token=True)                   # H2D prompt, D2H first token, sync
        t1 = time.perf_counter()
        tp = t1
        for _ in range(DECODE_STEPS):
            gm.decode_step(want_token=True, out=out)          # D2H 4 bytes + sync every token
            tn = time.perf_counter()
            tok_lat_us.append((tn - tp) * 1e6)
            tp = tn
        e2e_ttft_s.append(t1 - t0)
        e2e_decode_s.append(tp - t1)

    # ---- every decode kernel timed alone (CUDA events on the library's stream, launches back to back under PDL,
    #      cycling the 16 layers so that the weights streamed exceed L2) ------------------------------------------
    reps = 16 * 8
    per_step = {"attn_block": s.n_layers, "gate_up": s.n_layers, "down": s.n_layers, "lm_head": 1}
    kernels = {}
    gm.kv_reset(); gm.prefill(prompt, want_token=False); gm.sync()
    for which, name in ((0, "gate_up"), (1, "lm_head"), (4, "down"), (6, "attn_block")):
        r = 16 if which == 1 else reps
        gm.bench_kernel(which, 8)
        a, b = ev(), ev()
        a.record(stream)
        nbytes = gm.bench_kernel(which, r)
        b.record(stream)
        torch.cuda.synchronize(dev)
        ms = a.elapsed_time(b) / r
        kernels[name] = {"us": ms * 1e3, "GBps": nbytes / ms / 1e6, "bytes_per_launch": nbytes,
                         "launches_per_step": per_step[name]}

    # ---- read-only streaming probe: a sum-reduction over 4 GiB, the practical ceiling of a kernel that
    #      only reads HBM ------------------------------------------------------------------------------------------
    probe_gbs = None
    try:
        buf = torch.empty(4 << 30, dtype=torch.uint8, device=dev)
        buf.zero_()
        acc = torch.zeros(1, dtype=torch.int32, device=dev)
        with torch.cuda.stream(stream):
            for _ in range(2):
                hq.read_probe(buf, acc, stream=stream)
            a, b = ev(), ev()
            a.record(stream)
            for _ in range(5):
                hq.read_probe(buf, acc, stream=stream)
            b.record(stream)
        torch.cuda.synchronize(dev)
        probe_gbs = 5 * buf.numel() / (a.elapsed_time(b) * 1e-3) / 1e9
        del buf
    except Exception as e:    # e.g. not enough free memory for the probe buffer
        probe_gbs = None
        print("read probe skipped:", e, file=sys.stderr)

    # ---- aggregate over ranks (max time) -----------------------------------------------------------------
    dec_total_ms, total_ms, ttft, launches = aggregate_over_ranks(dist, dev, float(sum(decode_ms)), total_ms,
                                                                  float(np.mean(prefill_ms)), launches)

    if rank == 0:
        peak, peak_src = measured_peak()
        ncu = ncu_numbers()
        value = job_tokens_per_s(world, args.steps, dec_total_ms)
        ms_per_token = dec_total_ms / (args.steps * DECODE_STEPS)
        ctx_mid = PROMPT_LEN + DECODE_STEPS // 2
        bpt = bytes_per_token(s, ctx_mid)
        step_gbs = bpt / (ms_per_token * 1e-3) / 1e9
        e2e_value = world * DECODE_STEPS / float(np.mean(e2e_decode_s))
        # the kernel with the largest share of the step TIME, chosen from what was just measured
        dom = max(kernels, key=lambda k: kernels[k]["us"] * kernels[k]["launches_per_step"])
        kd = kernels[dom]
        label = {"attn_block": "attn_block_kernel (A2-A6 of a layer in one cluster launch: a latency chain, 8.5 % of the bytes)",
                 "gate_up": "sgemv_kernel<gate/up + SwiGLU> (43 % of the bytes per token)",
                 "down": "sgemv_kernel<down + residual> (22 % of the bytes)",
                 "lm_head": "sgemv_kernel<LM head + argmax> (21 % of the bytes)"}
        lat = np.array(tok_lat_us)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None,
            "dtype": "bf16 weights, f32 accumulate and residual stream; fp16 KV cache; activations into tensor-core MMAs "
                     "(decode GEMVs via mma.sync, prefill GEMMs via tcgen05) as two bf16 planes hi + lo; prefill attention fp16 mma.sync",
            "data": "synthetic",
            "config": {"workload": WORKLOAD, "l2": "inputs larger than L2 (2.47 GB of weights per token vs 126 MB)",
                       "multi_gpu": "independent replicas, no collective", "decode_path": gm.decode_path()},
            "ttft_ms": ttft, "ms_per_token": ms_per_token, "clocks": clocks, "gpu_launches": launches,
            "latency_us_per_token_streaming": {"p50": float(np.percentile(lat, 50)), "p99": float(np.percentile(lat, 99)),
                                               "mean": float(lat.mean()), "n": int(lat.size),
                                               "how": "hq_decode_step with a host token out: one sync + 4-byte D2H per token, host wall clock"},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": PROMPT_LEN * 4,
                    "d2h_bytes_per_step": (DECODE_STEPS + 1) * 4,
                    "ttft_ms": float(np.mean(e2e_ttft_s)) * 1e3,
                    "how": "hq_prefill(host tokens -> host first token) then 128 x hq_decode_step(host token out), "
                           "host wall clock, one sync + 4-byte D2H per token"},
            "roofline": {"bound": "hbm", "kernel": label[dom], "chosen": "largest us_per_launch x launches_per_step of kernels_alone",
                         "achieved": kd["GBps"], "peak": peak, "unit": "GB/s", "frac": kd["GBps"] / peak,
                         "traffic": ncu.get(dom + "_dram_bytes_per_launch"), "peak_source": peak_src,
                         "bytes_per_launch": kd["bytes_per_launch"], "us_per_launch": kd["us"],
                         "share_of_step_time": kd["us"] * kd["launches_per_step"] / (ms_per_token * 1e3)},
            # the kernel with the largest share of the BYTES: both its PDL-chained figure (back-to-back launches overlap the
            # predecessor's tail) and the serialised, cold-cache one from the committed ncu pass
            "roofline_gate_up": {"bound": "hbm", "kernel": label["gate_up"], "achieved": kernels["gate_up"]["GBps"], "peak": peak,
                                 "unit": "GB/s", "frac": kernels["gate_up"]["GBps"] / peak,
                                 "us_per_launch": kernels["gate_up"]["us"],
                                 "bytes_per_launch": kernels["gate_up"]["bytes_per_launch"],
                                 "traffic": ncu.get("gate_up_dram_bytes_per_launch"),
                                 "ncu_serialised_us": ncu.get("gate_up_ncu_us"),
                                 "ncu_serialised_frac": (kernels["gate_up"]["bytes_per_launch"] / (ncu["gate_up_ncu_us"] * 1e-6) / 1e9 / peak)
                                 if ncu.get("gate_up_ncu_us") else None},
            "step_roofline": {"bytes_per_token": bpt, "achieved_GBps": step_gbs, "frac_of_measured": step_gbs / peak,
                              "frac_of_8TBps_spec": step_gbs / 8000.0,
                              "read_probe_GBps": probe_gbs,
                              "frac_of_read_probe": (step_gbs / probe_gbs) if probe_gbs else None},
            "kernels_alone": kernels,
        }
        if not args.no_cpu_baseline:
            line["cpu_baseline"] = oracle_sample(weights, s)
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
