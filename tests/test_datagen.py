"""Pins for the shared seeded input generators (datagen/): SURVEY.md §8(c) readings 3, 4, 5, 16."""
import hashlib
import json
import os

import numpy as np

import datagen

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "datagen_checksums.json")


def test_splitmix64_published_vectors():
    # SplitMix64 (Steele, Lea, Flood 2014; reference implementation by Vigna) seeded with 0:
    # first three outputs.  mix64(x) is its output function applied to state x + gamma.
    gamma = 0x9E3779B97F4A7C15
    l = datagen.lib()
    assert l.hqd_mix64(0) == 0xE220A8397B1DCDAF
    assert l.hqd_mix64(gamma) == 0x6E789E6AA1B965F4
    assert l.hqd_mix64((2 * gamma) & (2**64 - 1)) == 0x06C45D188009454F


def test_bf16_round_to_nearest_even_pins():
    # 0.02f = 0x3CA3D70A -> 0x3CA4 (= 0.02001953125); 1.0f -> 0x3F80; exact ties go to even.
    x = np.array([0.02, 1.0], dtype=np.float32)
    assert datagen.f32_to_bf16_bits(x).tolist() == [0x3CA4, 0x3F80]
    ties = np.array([0x3F808000, 0x3F818000, 0x3F807FFF, 0x3F808001], dtype=np.uint32).view(np.float32)
    assert datagen.f32_to_bf16_bits(ties).tolist() == [0x3F80, 0x3F82, 0x3F80, 0x3F81]
    back = datagen.bf16_bits_to_f32(np.array([0x3CA4, 0x3F80, 0xBF80], dtype=np.uint16))
    assert back.tolist() == [0.02001953125, 1.0, -1.0]


def test_bf16_roundtrip_is_nearest():
    x = datagen.normal_f32(3, 5, 20000)
    b = datagen.bf16_bits_to_f32(datagen.f32_to_bf16_bits(x))
    # nearest: error at most half a bf16 ulp (ulp <= 2^-7 |x|), and idempotent
    assert np.all(np.abs(b - x) <= np.abs(x) * 2.0 ** -8)
    assert np.abs(b - x).max() > np.abs(x).max() * 2.0 ** -11   # it does round
    assert np.array_equal(datagen.f32_to_bf16_bits(b), datagen.f32_to_bf16_bits(x))


def test_normal_moments_and_range():
    x = datagen.normal_f32(11, 3, 1_000_000).astype(np.float64)
    assert abs(x.mean()) < 1e-4
    assert abs(x.std() - 0.02) < 1e-4
    assert np.abs(x).max() <= 0.02 * np.sqrt(2 * np.log(2.0 ** 32)) + 1e-9  # |z| <= 6.66
    # fourth moment of a normal: kurtosis 3
    assert abs(((x / x.std()) ** 4).mean() - 3.0) < 0.05
    g = datagen.normal_f32(11, 4, 100_000, mean=1.0).astype(np.float64)
    assert abs(g.mean() - 1.0) < 3e-4


def test_counter_based_prefix_and_tensor_independence():
    a = datagen.normal_f32(5, 9, 100)
    b = datagen.normal_f32(5, 9, 1000)
    assert np.array_equal(a, b[:100])                      # element i depends on i only
    c = datagen.normal_f32(5, 10, 1000)
    d = datagen.normal_f32(6, 9, 1000)
    assert abs(np.corrcoef(b, c)[0, 1]) < 0.1 and abs(np.corrcoef(b, d)[0, 1]) < 0.1


def test_box_muller_matches_numpy_restatement():
    # same recipe re-evaluated with numpy uint64 arithmetic on a few elements
    seed, tid, n = 77, 21, 64
    M = np.uint64
    def mix(x):
        with np.errstate(over="ignore"):
            z = x + M(0x9E3779B97F4A7C15)
            z = (z ^ (z >> M(30))) * M(0xBF58476D1CE4E5B9)
            z = (z ^ (z >> M(27))) * M(0x94D049BB133111EB)
            return z ^ (z >> M(31))
    with np.errstate(over="ignore"):
        key = mix(M(seed) ^ (M(tid) * M(0x9E3779B97F4A7C15)))
        r = mix(key + np.arange(n, dtype=np.uint64))
    u1 = ((r >> M(32)).astype(np.float64) + 1.0) / 2.0 ** 32
    u2 = (r & M(0xFFFFFFFF)).astype(np.float64) / 2.0 ** 32
    z = np.sqrt(-2 * np.log(u1)) * np.cos(2 * np.pi * u2)
    want = (0.02 * z).astype(np.float32)
    got = datagen.normal_f32(seed, tid, n)
    assert np.allclose(got, want, rtol=1e-6, atol=1e-9)


def test_tokens_uniform_in_range():
    v = 4096
    t = datagen.tokens(1000, v, 200_000)
    assert t.min() >= 0 and t.max() < v
    counts = np.bincount(t, minlength=v)
    assert counts.min() > 0 and abs(counts.mean() - 200_000 / v) < 1e-9
    chi2 = ((counts - counts.mean()) ** 2 / counts.mean()).sum()
    assert abs(chi2 - v) < 6 * np.sqrt(2 * v)              # chi-square with ~v dof


def test_param_counts_match_survey():
    # 1,235,814,400 parameters for the 1B shape, 2,499,840 for the tiny shape
    assert datagen.ONE_B.n_params == 1_235_814_400
    assert datagen.TINY.n_params == 2_499_840


def test_gains_are_one_plus_noise(tiny_weights):
    g = datagen.bf16_bits_to_f32(tiny_weights.final_norm)
    assert abs(g.mean() - 1.0) < 0.01 and 0.005 < g.std() < 0.04
    w = datagen.bf16_bits_to_f32(tiny_weights.layers[1]["w_up"])
    assert abs(w.mean()) < 1e-3 and abs(w.std() - 0.02) < 5e-4


def test_golden_checksums(tiny_weights, tiny_tokens):
    # written by tests/golden/make_golden.py (calls datagen only); guards the generator for good
    want = json.load(open(GOLDEN))
    got = {
        "tiny.embedding": hashlib.sha256(tiny_weights.embedding.tobytes()).hexdigest(),
        "tiny.final_norm": hashlib.sha256(tiny_weights.final_norm.tobytes()).hexdigest(),
        "tiny.l1.w_down": hashlib.sha256(tiny_weights.layers[1]["w_down"].tobytes()).hexdigest(),
        "tiny.tokens32": tiny_tokens.tolist(),
    }
    assert got == want
