"""The tcgen05/TMEM/TMA GEMM (hq_debug_gemm, C ABI) against the oracle's plain matmul and silu:
tile shapes, ragged token/row/K tails, split-K, residual and SwiGLU epilogues."""
import numpy as np
import pytest

import datagen
import oracle

pytestmark = pytest.mark.gpu


def _bf16_tensor(x_f32: np.ndarray):
    import torch
    bits = datagen.f32_to_bf16_bits(x_f32)
    return torch.from_numpy(bits.view(np.int16)).cuda().view(torch.bfloat16), datagen.bf16_bits_to_f32(bits)


def _hilo_tensor(x_f32: np.ndarray):
    """activation operand as two bf16 planes x = hi + lo; returns the device tensor [2,T,K] and the value it holds"""
    import torch
    hi_bits = datagen.f32_to_bf16_bits(x_f32)
    hi = datagen.bf16_bits_to_f32(hi_bits)
    lo_bits = datagen.f32_to_bf16_bits(x_f32 - hi)
    lo = datagen.bf16_bits_to_f32(lo_bits)
    t = torch.from_numpy(np.stack([hi_bits, lo_bits]).view(np.int16)).cuda().view(torch.bfloat16)
    return t, hi.astype(np.float64) + lo.astype(np.float64)


def _case(N, K, T, seed):
    w = datagen.normal_f32(seed, 1, N * K, std=0.05).reshape(N, K)
    x = datagen.normal_f32(seed, 2, T * K, std=1.0).reshape(T, K)
    return w, x


@pytest.mark.parametrize("N,K,T,tile,splits", [
    (128, 64, 32, 32, 1),        # one tile, one K block
    (256, 256, 32, 32, 1),
    (512, 2048, 200, 256, 1),    # ragged tokens inside a 256 tile
    (3072, 2048, 256, 256, 6),   # split-K (atomics into a zeroed buffer), QKV shape of the 1B model
    (688, 256, 70, 128, 1),      # ragged weight rows (688 = 5*128 + 48)
    (256, 688, 33, 64, 2),       # ragged K (688 = 10*64 + 48): TMA zero fill
    (2048, 8192, 300, 256, 9),   # down-proj shape, two token tiles
    (384, 512, 8, 32, 2),        # batched-decode shape: 8 sequences padded to a 32-token tile
    (384, 512, 8, 8, 2),         # the same in an 8-token tile (batched decode with <= 8 sequences)
    (2048, 8192, 5, 8, 9),       # down-projection shape, 5 sequences, 8-token tile, 9 K splits
    (3072, 2048, 16, 16, 6),     # Q|K|V shape, 16 sequences, 16-token tile
    (640, 256, 13, 16, 1),       # ragged tokens inside a 16-token tile
    (256, 512, 40, 8, 1),        # several 8-token tiles, ragged last one
    (384, 512, 100, 64, 1),      # CTA pairs (token tile <= 128, more than 32 tokens) with an odd number of weight tiles
    (3072, 2048, 256, 128, 2),   # the 1B Q|K|V shape as the prefill pass runs it: CTA pairs, 128-token tiles, 2 K splits
    (2048, 8192, 256, 128, 4),   # the 1B down-projection shape: CTA pairs, 4 K splits
])
def test_gemm_store_matches_oracle_matmul(N, K, T, tile, splits):
    import torch
    import paper_2606_12154_b200 as hq
    w, x = _case(N, K, T, 7 * N + K + T)
    wt, wr = _bf16_tensor(w)
    xt, xr = _hilo_tensor(x)
    out = torch.zeros((T, N), dtype=torch.float32, device="cuda")
    hq.debug_gemm(0, wt, xt, out, token_tile=tile, splits=splits)
    torch.cuda.synchronize()
    got = out.cpu().numpy().astype(np.float64)
    # expected: sampled rows through the oracle's plain matmul (double), all elements through torch fp64
    want_all = (torch.from_numpy(xr) @ torch.from_numpy(wr).double().T).numpy()
    rows = sorted(set([0, T - 1, T // 2]))
    want_rows = oracle.matmul(wr, xr[rows].astype(np.float64))
    assert np.allclose(want_all[rows], want_rows, rtol=1e-12, atol=1e-12)
    scale = np.abs(want_all).max()
    err = np.abs(got - want_all).max()
    assert err <= 2e-5 * scale * max(1.0, np.sqrt(K / 256)), (err, scale)   # fp32 accumulation of exact bf16 products


def test_gemm_residual_accumulates():
    import torch
    import paper_2606_12154_b200 as hq
    N, K, T = 256, 512, 96
    w, x = _case(N, K, T, 99)
    wt, wr = _bf16_tensor(w)
    xt, xr = _hilo_tensor(x)
    base = datagen.normal_f32(5, 5, T * N, std=1.0).reshape(T, N)
    for splits in (1, 4):
        out = torch.from_numpy(base.copy()).cuda()
        hq.debug_gemm(1, wt, xt, out, token_tile=128, splits=splits)
        torch.cuda.synchronize()
        want = base.astype(np.float64) + oracle.matmul(wr, xr.astype(np.float64))
        assert np.abs(out.cpu().numpy() - want).max() <= 3e-5 * np.abs(want).max()


@pytest.mark.parametrize("mode,N,K,T,tile", [
    (2, 688, 256, 100, 128),    # two accumulators per 128-row tile, ragged weight rows
    (3, 704, 256, 8, 32),       # 64-row tiles (batched decode), an odd number of them, 8 sequences in a 32-token tile
    (3, 704, 256, 8, 8),        # the same in an 8-token tile
    (3, 8192, 2048, 16, 16),    # the 1B gate/up shape at batch 16, 16-token tile
    (3, 256, 512, 11, 16),
    (3, 8192, 2048, 32, 32),    # the 1B gate/up shape at batch 32
    (3, 256, 512, 70, 64),      # 64-row tiles, two exchange rounds per token tile, ragged tokens
])
def test_gemm_swiglu_epilogue(mode, N, K, T, tile):
    import torch
    import paper_2606_12154_b200 as hq
    wg, x = _case(N, K, T, 11)
    wu, _ = _case(N, K, T, 12)
    wgt, wgr = _bf16_tensor(wg)
    wut, wur = _bf16_tensor(wu)
    xt, xr = _hilo_tensor(x)
    out = torch.zeros((2, T, N), dtype=torch.bfloat16, device="cuda")
    hq.debug_gemm(mode, wgt, xt, out, w2=wut, token_tile=tile)
    torch.cuda.synchronize()
    g = oracle.matmul(wgr, xr.astype(np.float64))
    u = oracle.matmul(wur, xr.astype(np.float64))
    want = np.vectorize(oracle.silu)(g) * u
    got = out.float().cpu().numpy().astype(np.float64).sum(axis=0)      # hi + lo
    # two-plane output: 16 mantissa bits, plus fp32 accumulation noise
    assert np.all(np.abs(got - want) <= np.abs(want) * 2.0 ** -15 + 1e-5 * np.abs(want).max())
