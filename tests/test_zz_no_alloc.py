"""hq_gemm_noalloc (include/hq_noalloc.h): the split-K tcgen05 GEMM with its partial buffers in the library's static
__device__ scratch array, against the existing path (hq_debug_gemm) on calls made back to back.

Collected last on purpose (the suite runs with `pytest -x`): a failure here hides nothing after it.  Passes alone in a
fresh process and after the other GPU tests (it shares no state with them; the scratch array is the library's own)."""
import numpy as np
import pytest

import datagen

pytestmark = pytest.mark.gpu


def _bf16(x_f32):
    import torch
    return torch.from_numpy(datagen.f32_to_bf16_bits(x_f32).view(np.int16)).cuda().view(torch.bfloat16)


def _hilo(x_f32):
    import torch
    hi_bits = datagen.f32_to_bf16_bits(x_f32)
    lo_bits = datagen.f32_to_bf16_bits(x_f32 - datagen.bf16_bits_to_f32(hi_bits))
    return torch.from_numpy(np.stack([hi_bits, lo_bits]).view(np.int16)).cuda().view(torch.bfloat16)


def _case(N, K, T, seed):
    w = datagen.normal_f32(seed, 1, N * K, std=0.05).reshape(N, K)
    x = datagen.normal_f32(seed, 2, T * K, std=1.0).reshape(T, K)
    return _bf16(w), _hilo(x)


def _tol(ref, K):
    # the bound tests/test_gpu_gemm.py uses for fp32 accumulation of exact bf16 products
    return 2e-5 * float(np.abs(ref).max()) * max(1.0, np.sqrt(K / 256))


def test_gemm_noalloc_matches_existing_path_on_calls_in_a_row():
    import torch
    import paper_2606_12154_b200 as hq
    assert hq.noalloc_scratch_bytes() == 16 << 20
    hq.noalloc_setup()
    # A: the 1B down-projection shape of a 256-token pass, 4 K splits: 8 MiB of the 16 MiB scratch, CTA pairs
    # B: a small ragged shape, 2 splits, single CTAs would not apply (T > 32 -> pairs), odd number of weight tiles
    # C: batched-decode shape (8 rows in a 32-token tile), 9 splits
    # D: ragged weight rows and an odd element count (the scalar form of the partial sum)
    cases = {"A": (2048, 8192, 256, 128, 4), "B": (384, 512, 100, 64, 2), "C": (2048, 8192, 8, 32, 9), "D": (129, 256, 33, 64, 2)}
    data, want = {}, {}
    for name, (N, K, T, tile, splits) in cases.items():
        w, x = _case(N, K, T, 1000 + N + K + T)
        ref = torch.zeros((T, N), dtype=torch.float32, device="cuda")
        hq.debug_gemm(0, w, x, ref, token_tile=tile, splits=1)      # the existing path, one K split (no atomics)
        data[name] = (w, x, torch.full((T, N), float("nan"), dtype=torch.float32, device="cuda"))
        want[name] = ref
    torch.cuda.synchronize()

    save = [torch.empty_like(data["A"][2]) for _ in range(2)]       # allocated before the no-allocation stretch below

    def run(name, keep=None):
        N, K, T, tile, splits = cases[name]
        w, x, out = data[name]
        out.fill_(float("nan"))
        hq.gemm_noalloc(w, x, out, token_tile=tile, splits=splits)
        torch.cuda.synchronize()
        got, ref = out.cpu().numpy().astype(np.float64), want[name].cpu().numpy().astype(np.float64)
        assert np.isfinite(got).all(), name
        err = np.abs(got - ref).max()
        assert err <= _tol(ref, K), (name, err, _tol(ref, K))
        if keep is not None:
            keep.copy_(out)

    run("A", save[0])                        # first call: set-up done, scratch holds A's partials afterwards
    free_before = torch.cuda.mem_get_info()[0]
    run("B")                                 # second call in a row: other shape, other data, fewer splits, stale scratch around it
    run("C")
    run("D")
    run("A", save[1])                        # and back
    free_after = torch.cuda.mem_get_info()[0]
    assert free_after >= free_before         # no device memory was allocated for these calls (by the library or anyone)
    assert torch.equal(save[0], save[1])     # bit-identical to the first A: fixed summation order, no stale data


def test_gemm_noalloc_rejects_what_does_not_fit():
    import torch
    import paper_2606_12154_b200 as hq
    N, K, T = 4096, 2048, 512                # 4 splits x 512 x 4096 x 4 B = 32 MiB > 16 MiB
    w = torch.zeros((N, K), dtype=torch.bfloat16, device="cuda")
    x = torch.zeros((2, T, K), dtype=torch.bfloat16, device="cuda")
    out = torch.full((T, N), 7.0, dtype=torch.float32, device="cuda")
    with pytest.raises(hq.HQError) as e:
        hq.gemm_noalloc(w, x, out, token_tile=128, splits=4)
    assert e.value.code == -2 and "scratch" in str(e.value)
    torch.cuda.synchronize()
    assert float(out.min()) == 7.0 and float(out.max()) == 7.0      # nothing was enqueued
    hq.gemm_noalloc(w, x, out, token_tile=128, splits=2)            # 16 MiB exactly: fits
    torch.cuda.synchronize()
    assert float(out.abs().max()) == 0.0
    with pytest.raises(hq.HQError):
        hq.gemm_noalloc(w, x, out, token_tile=48, splits=1)
