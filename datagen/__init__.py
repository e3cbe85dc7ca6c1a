"""Seeded synthetic inputs shared by the CPU oracle and the CUDA path (and by nothing else).

Holds no arithmetic of the method: model *shapes* (BASELINE.json `configs`), the counter-based
normal / token generators of ``hq_datagen.c`` and bf16 rounding.  See DESIGN.md "Input recipe".
"""
from __future__ import annotations

import ctypes
import dataclasses
import os
import subprocess
from typing import Dict, List

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hq_datagen.c")
_SO = os.path.join(_HERE, "libhq_datagen.so")

WEIGHT_SEED = 20260612  # SURVEY.md §8(d) seed scheme


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        extra = os.environ.get("HQO_EXTRA_CFLAGS", "").split()   # sanitizer run, see oracle/__init__.py
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC"] + extra + ["-o", _SO, _SRC, "-lm"])
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        l = ctypes.CDLL(build())
        l.hqd_mix64.restype = ctypes.c_uint64
        l.hqd_mix64.argtypes = [ctypes.c_uint64]
        l.hqd_key.restype = ctypes.c_uint64
        l.hqd_key.argtypes = [ctypes.c_uint64, ctypes.c_uint64]
        l.hqd_normal_f32.restype = None
        l.hqd_normal_f32.argtypes = [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_double,
                                     ctypes.c_double, ctypes.c_void_p, ctypes.c_size_t]
        l.hqd_tokens_i32.restype = None
        l.hqd_tokens_i32.argtypes = [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_int32,
                                     ctypes.c_void_p, ctypes.c_size_t]
        l.hqd_f32_to_bf16.restype = None
        l.hqd_f32_to_bf16.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t]
        l.hqd_bf16_to_f32.restype = None
        l.hqd_bf16_to_f32.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t]
        _lib = l
    return _lib


@dataclasses.dataclass(frozen=True)
class Shape:
    """Llama-style decoder shape (BASELINE.json configs[0] / configs[1..4])."""
    name: str
    n_layers: int
    hidden: int
    n_heads: int
    n_kv_heads: int
    head_dim: int
    ffn: int
    vocab: int
    rms_eps: float
    rope_theta: float

    @property
    def n_params(self) -> int:
        d, f = self.hidden, self.ffn
        q = self.n_heads * self.head_dim
        kv = self.n_kv_heads * self.head_dim
        per_layer = q * d + 2 * kv * d + d * q + 3 * f * d + 2 * d
        return self.n_layers * per_layer + self.vocab * d + d


TINY = Shape("tiny", 2, 256, 4, 2, 64, 688, 4096, 1e-5, 10000.0)          # configs[0]
ONE_B = Shape("1b", 16, 2048, 32, 8, 64, 8192, 128256, 1e-5, 500000.0)    # configs[1..4]
SHAPES = {"tiny": TINY, "1b": ONE_B}

# tensor ids (fixed for good: golden checksums depend on them)
TID_EMBEDDING = 0
TID_FINAL_NORM = 1
TID_TOKENS = 7
_LAYER_BASE, _LAYER_STRIDE = 16, 16
LAYER_TENSORS = ("attn_norm", "wq", "wk", "wv", "wo", "ffn_norm", "w_gate", "w_up", "w_down")


def layer_tid(layer: int, name: str) -> int:
    return _LAYER_BASE + _LAYER_STRIDE * layer + LAYER_TENSORS.index(name)


def normal_f32(seed: int, tensor_id: int, n: int, mean: float = 0.0, std: float = 0.02) -> np.ndarray:
    out = np.empty(n, dtype=np.float32)
    lib().hqd_normal_f32(seed, tensor_id, mean, std, out.ctypes.data, n)
    return out


def tokens(seed: int, vocab: int, n: int, tensor_id: int = TID_TOKENS) -> np.ndarray:
    out = np.empty(n, dtype=np.int32)
    lib().hqd_tokens_i32(seed, tensor_id, vocab, out.ctypes.data, n)
    return out


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.float32)
    out = np.empty(x.shape, dtype=np.uint16)
    lib().hqd_f32_to_bf16(x.ctypes.data, out.ctypes.data, x.size)
    return out


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    b = np.ascontiguousarray(b, dtype=np.uint16)
    out = np.empty(b.shape, dtype=np.float32)
    lib().hqd_bf16_to_f32(b.ctypes.data, out.ctypes.data, b.size)
    return out


def tensor_shapes(s: Shape) -> Dict[str, tuple]:
    q, kv = s.n_heads * s.head_dim, s.n_kv_heads * s.head_dim
    return {
        "attn_norm": (s.hidden,), "wq": (q, s.hidden), "wk": (kv, s.hidden), "wv": (kv, s.hidden),
        "wo": (s.hidden, q), "ffn_norm": (s.hidden,), "w_gate": (s.ffn, s.hidden),
        "w_up": (s.ffn, s.hidden), "w_down": (s.hidden, s.ffn),
    }


@dataclasses.dataclass
class Weights:
    """All tensors as bf16 bit patterns (uint16, nn.Linear [out, in] row-major).

    ``embedding`` doubles as the tied LM head.  ``f32(name)`` gives the exact fp32 value of the
    bf16-rounded tensor (what the oracle consumes); ``raw`` keeps the unrounded fp32 draw when
    ``keep_raw`` was asked for (configs[0] "fp32 weights").
    """
    shape: Shape
    embedding: np.ndarray
    final_norm: np.ndarray
    layers: List[Dict[str, np.ndarray]]
    raw: dict | None = None

    def nbytes(self) -> int:
        return 2 * self.shape.n_params


def make_weights(s: Shape, seed: int = WEIGHT_SEED, keep_raw: bool = False) -> Weights:
    """Matrices/embedding ~ N(0, 0.02^2); norm gains ~ 1 + N(0, 0.02^2); all bf16-rounded."""
    raw = {} if keep_raw else None

    def draw(tid: int, shp: tuple, mean: float) -> np.ndarray:
        n = int(np.prod(shp))
        x = normal_f32(seed, tid, n, mean=mean, std=0.02).reshape(shp)
        if keep_raw:
            raw[tid] = x
        return f32_to_bf16_bits(x)

    emb = draw(TID_EMBEDDING, (s.vocab, s.hidden), 0.0)
    fn = draw(TID_FINAL_NORM, (s.hidden,), 1.0)
    shapes = tensor_shapes(s)
    layers = []
    for l in range(s.n_layers):
        t = {}
        for name in LAYER_TENSORS:
            t[name] = draw(layer_tid(l, name), shapes[name], 1.0 if name.endswith("norm") else 0.0)
        layers.append(t)
    return Weights(s, emb, fn, layers, raw)
