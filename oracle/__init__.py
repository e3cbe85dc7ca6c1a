"""CPU oracle binding — TEST INFRASTRUCTURE, NOT PRODUCT (see hq_oracle.c header).

Only tests/, ``__graft_entry__.smoke()`` and bench.py's ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It imports nothing from ``paper_2606_12154_b200``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hq_oracle.c")
_SO = os.path.join(_HERE, "libhq_oracle.so")

c_f32p = ctypes.POINTER(ctypes.c_float)
c_f32pp = ctypes.POINTER(c_f32p)


class _Config(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in
                ("n_layers", "hidden", "n_heads", "n_kv_heads", "head_dim", "ffn", "vocab", "max_seq")]
    _fields_ += [("rms_eps", ctypes.c_double), ("rope_theta", ctypes.c_double)]


class _Weights(ctypes.Structure):
    _fields_ = [("tok_embedding", c_f32p), ("attn_norm", c_f32pp), ("wq", c_f32pp), ("wk", c_f32pp),
                ("wv", c_f32pp), ("wo", c_f32pp), ("ffn_norm", c_f32pp), ("w_gate", c_f32pp),
                ("w_up", c_f32pp), ("w_down", c_f32pp), ("final_norm", c_f32p), ("lm_head", c_f32p)]


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        # HQO_EXTRA_CFLAGS: e.g. "-fsanitize=address,undefined -g" for the recorded sanitizer run (profiles/r02_sanitizers.md)
        extra = os.environ.get("HQO_EXTRA_CFLAGS", "").split()
        subprocess.check_call(["gcc", "-O2", "-march=x86-64-v3", "-fopenmp", "-shared", "-fPIC"] + extra +
                              ["-o", _SO, _SRC, "-lm"])
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        l = ctypes.CDLL(build())
        dp, ip = ctypes.c_void_p, ctypes.c_void_p
        l.hqo_num_threads.restype = ctypes.c_int
        l.hqo_rmsnorm.argtypes = [dp, dp, ctypes.c_int32, ctypes.c_double, dp]
        l.hqo_rmsnorm.restype = None
        l.hqo_matmul.argtypes = [dp, dp, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, dp]
        l.hqo_matmul.restype = None
        l.hqo_rope.argtypes = [dp, ctypes.c_int32, ctypes.c_int32, ctypes.c_double]
        l.hqo_rope.restype = None
        l.hqo_silu.argtypes = [ctypes.c_double]
        l.hqo_silu.restype = ctypes.c_double
        l.hqo_attend.argtypes = [dp, dp, dp, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, dp, dp]
        l.hqo_attend.restype = None
        l.hqo_argmax.argtypes = [dp, ctypes.c_int32]
        l.hqo_argmax.restype = ctypes.c_int32
        l.hqo_top2_margin.argtypes = [dp, ctypes.c_int32]
        l.hqo_top2_margin.restype = ctypes.c_double
        l.hqo_create.argtypes = [ctypes.POINTER(_Config), ctypes.POINTER(_Weights)]
        l.hqo_create.restype = ctypes.c_void_p
        l.hqo_destroy.argtypes = [ctypes.c_void_p]
        l.hqo_destroy.restype = None
        l.hqo_reset.argtypes = [ctypes.c_void_p]
        l.hqo_reset.restype = None
        l.hqo_seq_len.argtypes = [ctypes.c_void_p]
        l.hqo_seq_len.restype = ctypes.c_int32
        l.hqo_forward.argtypes = [ctypes.c_void_p, ip, ctypes.c_int32, ctypes.c_int32, dp,
                                  ctypes.c_int32, dp]
        l.hqo_forward.restype = ctypes.c_int32
        l.hqo_get_kv.argtypes = [ctypes.c_void_p, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, dp]
        l.hqo_get_kv.restype = None
        _lib = l
    return _lib


def num_threads() -> int:
    return int(lib().hqo_num_threads())


# ---- primitives (exposed so each can be pinned on its own) ---------------------------------------
def _d(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _f(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float32)


def rmsnorm(x, g, eps: float) -> np.ndarray:
    x, g = _d(x), _f(g)
    out = np.empty_like(x)
    lib().hqo_rmsnorm(x.ctypes.data, g.ctypes.data, x.size, eps, out.ctypes.data)
    return out


def matmul(W, X) -> np.ndarray:
    """Y[t, o] = <W[o], X[t]>;  W fp32 [n_out, n_in], X double [T, n_in]."""
    W, X = _f(W), _d(X)
    T, n_in = X.shape
    Y = np.empty((T, W.shape[0]), dtype=np.float64)
    lib().hqo_matmul(W.ctypes.data, X.ctypes.data, T, W.shape[0], n_in, Y.ctypes.data)
    return Y


def rope(v, pos: int, theta: float) -> np.ndarray:
    v = _d(v).copy()
    lib().hqo_rope(v.ctypes.data, v.size, pos, theta)
    return v


def silu(z: float) -> float:
    return float(lib().hqo_silu(z))


def attend(q, K, V, return_probs: bool = False):
    """One query head q[hd] against K, V [n_ctx, hd]."""
    q, K, V = _d(q), _d(K), _d(V)
    n_ctx, hd = K.shape
    o = np.empty(hd, dtype=np.float64)
    p = np.empty(n_ctx, dtype=np.float64)
    lib().hqo_attend(q.ctypes.data, K.ctypes.data, V.ctypes.data, n_ctx, hd, hd, o.ctypes.data,
                     p.ctypes.data)
    return (o, p) if return_probs else o


def argmax(v) -> int:
    v = _d(v)
    return int(lib().hqo_argmax(v.ctypes.data, v.size))


def top2_margin(v) -> float:
    v = _d(v)
    return float(lib().hqo_top2_margin(v.ctypes.data, v.size))


# ---- model -----------------------------------------------------------------------------------------
class Model:
    """Oracle model over fp32 weight arrays.

    ``layers`` is a list of dicts with keys attn_norm, wq, wk, wv, wo, ffn_norm, w_gate, w_up,
    w_down (numpy float32, nn.Linear [out, in]); ``lm_head=None`` ties it to the embedding.
    """

    def __init__(self, *, n_layers, hidden, n_heads, n_kv_heads, head_dim, ffn, vocab, rms_eps,
                 rope_theta, max_seq, embedding, final_norm, layers: Sequence[dict], lm_head=None):
        self._keep = []

        def keep(a):
            a = _f(a)
            self._keep.append(a)
            return a

        def fp(a):
            return a.ctypes.data_as(c_f32p)

        def arr(name):
            ptrs = (c_f32p * n_layers)(*[fp(keep(layers[l][name])) for l in range(n_layers)])
            self._keep.append(ptrs)
            return ctypes.cast(ptrs, c_f32pp)

        emb = keep(embedding)
        head = emb if lm_head is None else keep(lm_head)
        self.cfg = _Config(n_layers, hidden, n_heads, n_kv_heads, head_dim, ffn, vocab, max_seq,
                           rms_eps, rope_theta)
        w = _Weights(fp(emb), arr("attn_norm"), arr("wq"), arr("wk"), arr("wv"), arr("wo"),
                     arr("ffn_norm"), arr("w_gate"), arr("w_up"), arr("w_down"),
                     fp(keep(final_norm)), fp(head))
        self._h = lib().hqo_create(ctypes.byref(self.cfg), ctypes.byref(w))
        if not self._h:
            raise ValueError("hqo_create rejected the config")
        self.n_layers, self.hidden, self.vocab = n_layers, hidden, vocab
        self.kv_dim = n_kv_heads * head_dim

    @classmethod
    def from_datagen(cls, weights, max_seq: int, use_raw_fp32: bool = False) -> "Model":
        """Build from ``datagen.Weights``: the bf16-rounded values as fp32 (default) or the raw draw."""
        import datagen  # input generators only
        s = weights.shape

        def val(bits, tid):
            if use_raw_fp32:
                return weights.raw[tid]
            return datagen.bf16_bits_to_f32(bits)

        layers = []
        for l, t in enumerate(weights.layers):
            layers.append({k: val(v, datagen.layer_tid(l, k)) for k, v in t.items()})
        return cls(n_layers=s.n_layers, hidden=s.hidden, n_heads=s.n_heads, n_kv_heads=s.n_kv_heads,
                   head_dim=s.head_dim, ffn=s.ffn, vocab=s.vocab, rms_eps=s.rms_eps,
                   rope_theta=s.rope_theta, max_seq=max_seq,
                   embedding=val(weights.embedding, datagen.TID_EMBEDDING),
                   final_norm=val(weights.final_norm, datagen.TID_FINAL_NORM), layers=layers)

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h:
            lib().hqo_destroy(h)

    def reset(self):
        lib().hqo_reset(self._h)

    @property
    def seq_len(self) -> int:
        return int(lib().hqo_seq_len(self._h))

    def forward(self, tokens, hidden: str = "none", logits: str = "last"):
        """Feed ``tokens`` at the next positions.  hidden/logits in {"none", "last", "all"}.

        Returns (hidden, logits): hidden [L, d] ("last") or [T, L, d] ("all"); logits [V] or [T, V].
        """
        mode = {"none": 0, "last": 1, "all": 2}
        toks = np.ascontiguousarray(tokens, dtype=np.int32).reshape(-1)
        T = toks.size
        hm, lm = mode[hidden], mode[logits]
        hid: Optional[np.ndarray] = None
        lg: Optional[np.ndarray] = None
        if hm:
            hid = np.empty((self.n_layers, self.hidden) if hm == 1 else (T, self.n_layers, self.hidden))
        if lm:
            lg = np.empty((self.vocab,) if lm == 1 else (T, self.vocab))
        rc = lib().hqo_forward(self._h, toks.ctypes.data, T, hm, hid.ctypes.data if hm else None,
                               lm, lg.ctypes.data if lm else None)
        if rc != 0:
            raise ValueError("hqo_forward: capacity overflow, empty input or token out of range")
        return hid, lg

    def kv_row(self, which: str, layer: int, pos: int) -> np.ndarray:
        out = np.empty(self.kv_dim)
        lib().hqo_get_kv(self._h, 0 if which == "k" else 1, layer, pos, out.ctypes.data)
        return out

    def greedy(self, prompt, n_steps: int, hidden: str = "none"):
        """Prefill then ``n_steps`` greedy steps: token_0 = argmax(prefill logits);
        step i feeds token_{i-1}.  Returns dict with tokens [n_steps+1], logits [n_steps+1, V],
        hidden [n_steps+1, L, d] (if asked), margins [n_steps+1]."""
        hs, lgs, toks, margins = [], [], [], []
        h, lg = self.forward(prompt, hidden=hidden, logits="last")
        for i in range(n_steps + 1):
            toks.append(argmax(lg)); margins.append(top2_margin(lg)); lgs.append(lg); hs.append(h)
            if i == n_steps:
                break
            h, lg = self.forward([toks[-1]], hidden=hidden, logits="last")
        return {"tokens": np.array(toks, dtype=np.int32), "logits": np.stack(lgs),
                "hidden": np.stack(hs) if hidden != "none" else None, "margins": np.array(margins)}
