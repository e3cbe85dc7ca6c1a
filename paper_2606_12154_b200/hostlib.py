"""ctypes binding of include/hq_host.h (libhq_host.so): router, gate, renderer, synthetic tokeniser — marshalling only."""
from __future__ import annotations

import ctypes
import os
from typing import List, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libhq_host.so")

DECLARED_SYMBOLS = ("hqh_store_create", "hqh_store_destroy", "hqh_store_size", "hqh_route", "hqh_gate", "hqh_render",
                    "hqh_marker", "hqh_tokenize")

_lib = None


def load_library():
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise ImportError(f"{_LIB_PATH} is missing: build it with `python -m paper_2606_12154_b200.build`")
        l = ctypes.CDLL(_LIB_PATH)
        vp, i32, dbl = ctypes.c_void_p, ctypes.c_int32, ctypes.c_double
        cpp = ctypes.POINTER(ctypes.c_char_p)
        l.hqh_store_create.restype = i32
        l.hqh_store_create.argtypes = [cpp, cpp, i32, dbl, dbl, ctypes.POINTER(vp)]
        l.hqh_store_destroy.restype = None
        l.hqh_store_destroy.argtypes = [vp]
        l.hqh_store_size.restype = i32
        l.hqh_store_size.argtypes = [vp]
        l.hqh_route.restype = i32
        l.hqh_route.argtypes = [vp, ctypes.c_char_p, i32, vp, vp]
        l.hqh_gate.restype = i32
        l.hqh_gate.argtypes = [dbl, dbl, dbl, ctypes.POINTER(dbl)]
        l.hqh_render.restype = i32
        l.hqh_render.argtypes = [vp, i32, ctypes.c_char_p, i32]
        l.hqh_marker.restype = ctypes.c_char_p
        l.hqh_marker.argtypes = []
        l.hqh_tokenize.restype = i32
        l.hqh_tokenize.argtypes = [ctypes.c_char_p, i32, vp, i32]
        _lib = l
    return _lib


class Store:
    """The structured store as the runtime sees it: key text (key + aliases) and the answer line per entry."""

    def __init__(self, key_text: Sequence[str], answer_line: Sequence[str], k1: float = 1.2, b: float = 0.75):
        lib = load_library()
        n = len(key_text)
        keys = (ctypes.c_char_p * n)(*[k.encode() for k in key_text])
        answers = (ctypes.c_char_p * n)(*[a.encode() for a in answer_line])
        h = ctypes.c_void_p()
        rc = lib.hqh_store_create(keys, answers, n, k1, b, ctypes.byref(h))
        if rc != 0:
            raise ValueError(f"hqh_store_create failed: {rc}")
        self._lib, self._h = lib, h
        self._buf = ctypes.create_string_buffer(1 << 16)

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h:
            self._lib.hqh_store_destroy(h)

    def __len__(self) -> int:
        return int(self._lib.hqh_store_size(self._h))

    def route(self, query: str, top_k: int = 3) -> Tuple[np.ndarray, np.ndarray]:
        ids = np.empty(top_k, dtype=np.int32)
        scores = np.empty(top_k, dtype=np.float64)
        rc = self._lib.hqh_route(self._h, query.encode(), top_k, ids.ctypes.data, scores.ctypes.data)
        if rc != 0:
            raise ValueError(f"hqh_route failed: {rc}")
        return ids, scores

    def render(self, entry: int) -> str:
        n = self._lib.hqh_render(self._h, entry, self._buf, len(self._buf))
        if n < 0:
            raise ValueError(f"hqh_render failed: {n}")
        return self._buf.raw[:n].decode()


def gate(s1: float, s2: float, tau: float = 0.05) -> Tuple[bool, float]:
    m = ctypes.c_double()
    ok = load_library().hqh_gate(s1, s2, tau, ctypes.byref(m))
    return bool(ok), m.value


def marker() -> str:
    return load_library().hqh_marker().decode()


def tokenize(text: str, vocab: int) -> np.ndarray:
    out = np.empty(max(16, 2 * len(text)), dtype=np.int32)
    n = load_library().hqh_tokenize(text.encode(), vocab, out.ctypes.data, out.size)
    if n < 0:
        raise ValueError(f"hqh_tokenize failed: {n}")
    return out[:n].copy()
