"""Pins of the hq4 quantiser oracle (oracle/q4_oracle.py): hand-worked groups, the defining inequalities, exactness of the
dequantised values in bf16, the packed layout.  CPU only."""
import numpy as np

import datagen
from oracle import q4_oracle as q4


def group(vals):
    g = np.zeros((1, 32))
    g[0, :len(vals)] = vals
    return g


def test_hand_worked_groups():
    # max 7.0 -> e = 0 (7 <= 7 * 2^0), codes are the values themselves
    q, e = q4.quantize(group([7.0, -3.0, 1.0, 0.0]))
    assert e[0, 0] == 0 and list(q[0, :4]) == [7, -3, 1, 0]
    # max 7.5 > 7 -> e = 1; 7.5 / 2 = 3.75 -> 4; 1 / 2 = 0.5 -> 0 and 3 / 2 = 1.5 -> 2 (ties to even); -5 / 2 = -2.5 -> -2
    q, e = q4.quantize(group([7.5, 1.0, 3.0, -5.0]))
    assert e[0, 0] == 1 and list(q[0, :4]) == [4, 0, 2, -2]
    # max 0.875 = 7 * 2^-3 -> e = -3 exactly at the boundary; just above it -> e = -2
    assert q4.quantize(group([0.875]))[1][0, 0] == -3
    assert q4.quantize(group([0.875 * (1 + 2.0 ** -20)]))[1][0, 0] == -2
    # a typical weight: 0.02 = 1.28 * 2^-6 -> 7 * 2^-9 = 0.01367 < 0.02 <= 7 * 2^-8 = 0.02734 -> e = -8, code rint(5.12) = 5
    q, e = q4.quantize(group([0.02, -0.02, 0.001]))
    assert e[0, 0] == -8 and list(q[0, :3]) == [5, -5, 0]
    # all-zero group: codes 0, exponent byte 1 (e = -126)
    q, e = q4.quantize(group([]))
    assert e[0, 0] == -126 and not q.any()
    # the negative extreme never exceeds -7 in magnitude with this exponent rule (clamp to -8 is never hit)
    q, e = q4.quantize(group([-7.0 * 2.0 ** 5]))
    assert e[0, 0] == 5 and q[0, 0] == -7


def test_defining_inequalities_on_model_weights():
    w = datagen.make_weights(datagen.TINY)
    for name in ("w_gate", "w_down"):
        x = datagen.bf16_bits_to_f32(w.layers[0][name]).astype(np.float64)
        x = x[:, : x.shape[1] // 32 * 32]
        q, e = q4.quantize(x)
        m = np.abs(x.reshape(x.shape[0], -1, 32)).max(-1)
        s = np.ldexp(1.0, e.astype(np.int64))
        assert (m <= 7 * s).all() and (m > 7 * s / 2).all()            # the SMALLEST exponent that covers the group
        d = q4.dequantize(q, e).astype(np.float64)
        err = np.abs(d - x).reshape(x.shape[0], -1, 32)
        assert (err <= s[..., None] / 2).all()                           # round to nearest: at most half a step
        assert q.min() >= -7 and q.max() <= 7
        # the dequantised weights are exact bf16 values and quantise to themselves
        assert np.array_equal(datagen.bf16_bits_to_f32(datagen.f32_to_bf16_bits(d.astype(np.float32))), d.astype(np.float32))
        assert np.array_equal(q4.dequantize(*q4.quantize(d)), d.astype(np.float32))


def test_packed_layout():
    q = np.zeros((1, 32), dtype=np.int8)
    q[0, :4] = [-8, 7, 0, -1]
    codes, eb = q4.pack(q, np.array([[-8]], dtype=np.int16))
    # element 0 (-8 -> nibble 0) low and element 1 (7 -> nibble 15) high of byte 0; elements 2, 3 (0 -> 8, -1 -> 7) of byte 1
    assert codes[0, 0] == 0xF0 and codes[0, 1] == 0x78 and codes[0, 2] == 0x88 and eb[0, 0] == 119
    assert codes.shape == (1, 16) and eb.shape == (1, 1)
