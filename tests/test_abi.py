"""Host-side checks of the C-ABI boundary that need no GPU: the library builds for sm_100a, loads,
exports every symbol include/hq.h declares, does its host arithmetic, and refuses to run without a
CUDA device (no CPU fallback)."""
import ctypes
import os
import re
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def hq():
    from paper_2606_12154_b200 import build
    build.build()
    import paper_2606_12154_b200 as hq
    return hq


def header_functions():
    names = set()
    for h in ("hq.h", "hq_debug.h", "hq_noalloc.h"):
        src = open(os.path.join(ROOT, "include", h)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(hq_[a-z_0-9]+)\s*\(", src))
    return sorted(names)


def test_library_reads_no_environment_variable():
    """Every switch is an hq_config flag decided at hq_model_create; nothing below it consults the environment."""
    csrc = os.path.join(ROOT, "paper_2606_12154_b200", "csrc")
    for f in sorted(os.listdir(csrc)):
        assert "getenv" not in open(os.path.join(csrc, f)).read(), f


def test_every_product_call_cites_its_passage():
    """include/hq.h: the comment in front of every exported call names the passage that defines it."""
    src = open(os.path.join(ROOT, "include", "hq.h")).read()
    for m in re.finditer(r"/\*((?:(?!\*/).)*)\*/\s*(?:const\s+char\s*\*|int32_t|int64_t|size_t|void)\s*(hq_[a-z_0-9]+)\s*\(", src, flags=re.S):
        comment, name = m.group(1), m.group(2)
        assert re.search(r"PAPER\.md:L\d+|north_star|error convention|Counterpart of", comment), name


def test_header_and_binding_declare_the_same_symbols(hq):
    assert header_functions() == sorted(hq.DECLARED_SYMBOLS)


def test_library_exports_every_declared_symbol(hq):
    lib = hq.load_library()
    for name in header_functions():
        assert hasattr(lib, name), name
    out = subprocess.check_output(["nm", "-D", "--defined-only", os.path.join(ROOT, "paper_2606_12154_b200", "libhq.so")]).decode()
    exported = set(re.findall(r" T (hq_[a-z_0-9]+)", out))
    assert set(header_functions()) <= exported
    assert "sm_100a" in hq.version()


def test_library_contains_sm100a_sass_only(hq):
    out = subprocess.check_output(["cuobjdump", "-lelf", os.path.join(ROOT, "paper_2606_12154_b200", "libhq.so")]).decode()
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_workspace_bytes_is_host_arithmetic(hq):
    from paper_2606_12154_b200.binding import make_config
    cfg = make_config(n_layers=16, hidden=2048, n_heads=32, n_kv_heads=8, head_dim=64, ffn=8192, vocab=128256,
                      rms_eps=1e-5, rope_theta=500000.0, max_batch=1, max_seq=4352)
    n = hq.workspace_bytes(cfg)
    kv = 2 * 16 * 1 * 8 * 4352 * 64 * 2          # K and V, bf16: 32,768 B per cached token
    assert kv == 4352 * 32768
    # + fp32 logits, decode scratch and the row-batched (tensor-core) pass buffers: 2,048 rows of
    # residual, hi/lo bf16 operands, 4 split-K partial buffers each of qkv and of the deferred residual, the SwiGLU output (~275 MB)
    assert kv < n < kv + 512 * 2 ** 20
    cfg2 = make_config(n_layers=16, hidden=2048, n_heads=32, n_kv_heads=8, head_dim=64, ffn=8192, vocab=128256,
                       rms_eps=1e-5, rope_theta=500000.0, max_batch=8, max_seq=4352)
    assert hq.workspace_bytes(cfg2) > 8 * kv
    bad = make_config(n_layers=0, hidden=2048, n_heads=32, n_kv_heads=8, head_dim=64, ffn=8192, vocab=128256,
                      rms_eps=1e-5, rope_theta=500000.0)
    assert hq.workspace_bytes(bad) == 0
    assert b"non-positive" in hq.load_library().hq_last_error()


def test_noalloc_scratch_size_is_the_header_constant(hq):
    """include/hq_noalloc.h states the size of the static scratch array; the library reports the same (host arithmetic)."""
    src = open(os.path.join(ROOT, "include", "hq_noalloc.h")).read()
    m = re.search(r"#define\s+HQ_NOALLOC_SCRATCH_BYTES\s+\((\d+)u\s*<<\s*(\d+)\)", src)
    assert m, "HQ_NOALLOC_SCRATCH_BYTES not found"
    assert hq.noalloc_scratch_bytes() == int(m.group(1)) << int(m.group(2)) == 16 << 20


def test_create_rejects_bad_arguments_before_touching_cuda(hq):
    from paper_2606_12154_b200.binding import Weights, make_config
    lib = hq.load_library()
    h = ctypes.c_void_p()
    good = dict(n_layers=2, hidden=256, n_heads=4, n_kv_heads=2, head_dim=64, ffn=688, vocab=4096, rms_eps=1e-5,
                rope_theta=1e4, max_batch=1, max_seq=64)
    w = Weights()
    cfg = make_config(**good)
    assert lib.hq_model_create(ctypes.byref(cfg), ctypes.byref(w), None, 0, None, ctypes.byref(h)) == -1  # NULL workspace
    cfg = make_config(**dict(good, head_dim=128))
    assert lib.hq_model_create(ctypes.byref(cfg), ctypes.byref(w), None, 0, None, ctypes.byref(h)) == -5
    assert b"head_dim" in lib.hq_last_error()
    cfg = make_config(**dict(good, n_kv_heads=3))
    assert lib.hq_model_create(ctypes.byref(cfg), ctypes.byref(w), None, 0, None, ctypes.byref(h)) == -5
    cfg = make_config(**dict(good, max_batch=64))
    assert lib.hq_model_create(ctypes.byref(cfg), ctypes.byref(w), None, 0, None, ctypes.byref(h)) == -5
    assert lib.hq_model_create(ctypes.byref(cfg), ctypes.byref(w), None, 0, None, None) == -1
    assert h.value is None
    # NULL model handles are rejected, destroy(NULL) is a no-op
    assert lib.hq_sync(None) == -1 and lib.hq_kv_reset(None) == -1
    assert lib.hq_decode_step(None, None, None) == -1
    lib.hq_model_destroy(None)


def test_no_cpu_fallback(hq):
    """Without a CUDA device the binding raises; it never computes on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    import datagen
    w = datagen.make_weights(datagen.TINY)
    with pytest.raises(hq.HQError) as e:
        hq.Model.from_bf16_bits(w.shape, w.embedding, w.final_norm, w.layers, max_seq=64, device="cpu")
    assert e.value.code == -4


def test_product_does_not_import_oracle():
    """The product path never imports oracle/ (only tests, smoke() and bench's cpu_baseline may)."""
    pkg = os.path.join(ROOT, "paper_2606_12154_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert "hq_oracle" not in src and "hqo_" not in src, f
    opy = open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    osrc = open(os.path.join(ROOT, "oracle", "hq_oracle.c")).read()
    assert not re.search(r"^\s*(import|from)\s+paper_2606_12154_b200", opy, flags=re.M)
    assert "libhq.so" not in opy and "#include \"hq" not in osrc and "#include <cuda" not in osrc
