"""CPU oracle of the 4-bit weight format "hq4" — TEST INFRASTRUCTURE, NOT PRODUCT.

SURVEY.md 8(f)-1: "4-bit weight-only GEMV (group-wise int4 + scales, own format) ... needs a quantisation-aware oracle".
The paper's mouth model runs at 4-bit quantisation through a third-party runtime whose format is not
described and not used here.  The format below is this repository's own ((f)-1):

  * a weight row of K elements (K a multiple of 32) is cut into groups of 32 consecutive elements;
  * group exponent e = the smallest integer with max|w| <= 7 * 2^e (e = -126 for an all-zero group), stored as the byte
    E = e + 127;
  * code q = round-half-to-even(w / 2^e), clamped to [-8, 7], stored as the nibble q + 8; element 2j of a row sits in the
    low nibble of byte j, element 2j + 1 in the high nibble;
  * the weight the model computes with is w' = q * 2^e — exactly representable in bf16 (|q| needs 3 bits).

The quantisation-aware oracle of the model is oracle.Model over w' for the quantised matrices (plain fp64 forward): this
file only restates the quantiser, step by step, with numpy.  No code shared with paper_2606_12154_b200/.
"""
from __future__ import annotations

import numpy as np

GROUP = 32


def quantize(w: np.ndarray):
    """w: float array [N, K] (the bf16 weights as fp32/fp64 values).  Returns (q int8 [N, K] in -8..7, e int16 [N, K/32])."""
    w = np.asarray(w, dtype=np.float64)
    n, k = w.shape
    assert k % GROUP == 0
    g = w.reshape(n, k // GROUP, GROUP)
    m = np.abs(g).max(axis=-1)                               # max |w| of the group
    # smallest e with m <= 7 * 2^e: m = f * 2^x with f in [0.5, 1)  =>  m <= 0.875 * 2^(e + 3)  <=>  e >= x - 3 (f <= 0.875) or x - 2
    f, x = np.frexp(m)
    e = np.where(f <= 0.875, x - 3, x - 2).astype(np.int64)
    e = np.where(m == 0.0, -126, e)
    e = np.clip(e, -126, 120)
    q = np.rint(g / np.ldexp(1.0, e)[..., None])             # exact scaling by a power of two, round half to even
    q = np.clip(q, -8, 7)
    return q.reshape(n, k).astype(np.int8), e.astype(np.int16)


def dequantize(q: np.ndarray, e: np.ndarray) -> np.ndarray:
    """w' = q * 2^e as float32 (exact)."""
    n, k = q.shape
    g = q.reshape(n, k // GROUP, GROUP).astype(np.float64) * np.ldexp(1.0, e.astype(np.int64))[..., None]
    return g.reshape(n, k).astype(np.float32)


def pack(q: np.ndarray, e: np.ndarray):
    """The documented memory layout: codes uint8 [N, K/2] (element 2j low nibble, 2j + 1 high nibble of byte j, nibble =
    q + 8), exponent bytes uint8 [N, K/32] (e + 127)."""
    v = (q.astype(np.int16) + 8).astype(np.uint8)
    codes = (v[:, 0::2] | (v[:, 1::2] << 4)).astype(np.uint8)
    return codes, (e + 127).astype(np.uint8)
