"""ctypes binding of include/hq.h — argument marshalling only; every step runs in libhq's kernels.

PyTorch is used for device memory (weights, workspace, outputs) and the CUDA stream, nothing else.
"""
from __future__ import annotations

import ctypes
import os
from typing import Dict, List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libhq.so")

FLAG_CAPTURE_HIDDEN = 1
FLAG_NO_GRAPH = 2
FLAG_NO_PDL = 4
FLAG_KERNEL_PER_ROW = 8
FLAG_VERIFY = 16
DTYPE_BF16, DTYPE_Q4 = 0, 1

HQ_OK, HQ_ERR_INVALID_ARG, HQ_ERR_CAPACITY, HQ_ERR_STATE, HQ_ERR_CUDA, HQ_ERR_UNSUPPORTED = 0, -1, -2, -3, -4, -5
_CODE_NAMES = {-1: "HQ_ERR_INVALID_ARG", -2: "HQ_ERR_CAPACITY", -3: "HQ_ERR_STATE", -4: "HQ_ERR_CUDA",
               -5: "HQ_ERR_UNSUPPORTED"}

# every symbol include/hq.h and include/hq_debug.h declare (tests check the headers and the library against this list)
DECLARED_SYMBOLS = (
    "hq_workspace_bytes", "hq_model_create", "hq_model_create_q4", "hq_quantize_q4", "hq_dequantize_q4", "hq_model_destroy", "hq_prefill", "hq_decode_step",
    "hq_decode_run", "hq_verify_relay", "hq_decode_logits", "hq_get_hidden", "hq_sync", "hq_seq_len", "hq_kv_reset",
    "hq_kernel_count", "hq_decode_path", "hq_bench_kernel", "hq_debug_copy_probe", "hq_debug_gemm", "hq_debug_gemm_timeline", "hq_debug_kv_row", "hq_debug_read_probe", "hq_debug_step_trace", "hq_debug_trace", "hq_last_error",
    "hq_version", "hq_noalloc_scratch_bytes", "hq_noalloc_setup", "hq_gemm_noalloc",
)


class HQError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{_CODE_NAMES.get(code, code)}: {msg}")
        self.code = code


class Config(ctypes.Structure):
    _fields_ = [("n_layers", ctypes.c_int32), ("hidden", ctypes.c_int32), ("n_heads", ctypes.c_int32),
                ("n_kv_heads", ctypes.c_int32), ("head_dim", ctypes.c_int32), ("ffn", ctypes.c_int32),
                ("vocab", ctypes.c_int32), ("rms_eps", ctypes.c_float), ("rope_theta", ctypes.c_float),
                ("max_batch", ctypes.c_int32), ("max_seq", ctypes.c_int32), ("weight_dtype", ctypes.c_int32),
                ("flags", ctypes.c_uint32)]


_vpp = ctypes.POINTER(ctypes.c_void_p)


class Weights(ctypes.Structure):
    _fields_ = [("tok_embedding", ctypes.c_void_p), ("attn_norm", _vpp), ("wq", _vpp), ("wk", _vpp),
                ("wv", _vpp), ("wo", _vpp), ("ffn_norm", _vpp), ("w_gate", _vpp), ("w_up", _vpp),
                ("w_down", _vpp), ("final_norm", ctypes.c_void_p), ("lm_head", ctypes.c_void_p)]


class WeightsQ4(ctypes.Structure):
    _fields_ = [("w_gate_codes", _vpp), ("w_gate_exps", _vpp), ("w_up_codes", _vpp), ("w_up_exps", _vpp),
                ("w_down_codes", _vpp), ("w_down_exps", _vpp), ("lm_head_codes", ctypes.c_void_p),
                ("lm_head_exps", ctypes.c_void_p)]


_lib = None


def load_library(path: Optional[str] = None):
    """Load libhq.so (in-tree).  Fails loudly when it has not been built: there is no fallback."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or _LIB_PATH
    if not os.path.exists(p):
        raise ImportError(f"{p} is missing: build it with `python -m paper_2606_12154_b200.build` "
                          "(or __graft_entry__.build()); hq has no CPU or PyTorch fallback")
    l = ctypes.CDLL(p)
    vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
    l.hq_workspace_bytes.restype = ctypes.c_size_t
    l.hq_workspace_bytes.argtypes = [ctypes.POINTER(Config)]
    l.hq_model_create.restype = i32
    l.hq_model_create.argtypes = [ctypes.POINTER(Config), ctypes.POINTER(Weights), vp, ctypes.c_size_t, vp,
                                  ctypes.POINTER(vp)]
    l.hq_model_create_q4.restype = i32
    l.hq_model_create_q4.argtypes = [ctypes.POINTER(Config), ctypes.POINTER(Weights), ctypes.POINTER(WeightsQ4), vp,
                                     ctypes.c_size_t, vp, ctypes.POINTER(vp)]
    l.hq_quantize_q4.restype = i32
    l.hq_quantize_q4.argtypes = [vp, vp, i64, i32, vp, vp]
    l.hq_dequantize_q4.restype = i32
    l.hq_dequantize_q4.argtypes = [vp, vp, vp, i64, i32, vp]
    l.hq_model_destroy.restype = None
    l.hq_model_destroy.argtypes = [vp]
    l.hq_prefill.restype = i32
    l.hq_prefill.argtypes = [vp, vp, i32, i32, vp, vp]
    l.hq_decode_step.restype = i32
    l.hq_decode_step.argtypes = [vp, vp, vp]
    l.hq_decode_run.restype = i32
    l.hq_decode_run.argtypes = [vp, i32, vp]
    l.hq_verify_relay.restype = i32
    l.hq_verify_relay.argtypes = [vp, vp, i32, i32, vp]
    l.hq_decode_logits.restype = i32
    l.hq_decode_logits.argtypes = [vp, vp]
    l.hq_get_hidden.restype = i32
    l.hq_get_hidden.argtypes = [vp, i32, vp]
    l.hq_sync.restype = i32
    l.hq_sync.argtypes = [vp]
    l.hq_seq_len.restype = i32
    l.hq_seq_len.argtypes = [vp, ctypes.POINTER(i32)]
    l.hq_kv_reset.restype = i32
    l.hq_kv_reset.argtypes = [vp]
    l.hq_kernel_count.restype = i64
    l.hq_kernel_count.argtypes = [vp]
    l.hq_decode_path.restype = ctypes.c_char_p
    l.hq_decode_path.argtypes = [vp]
    l.hq_bench_kernel.restype = i32
    l.hq_bench_kernel.argtypes = [vp, i32, i32, ctypes.POINTER(i64)]
    l.hq_debug_gemm.restype = i32
    l.hq_debug_gemm.argtypes = [vp, i32, vp, vp, vp, vp, i32, i32, i32, i32, i32]
    l.hq_noalloc_scratch_bytes.restype = ctypes.c_size_t
    l.hq_noalloc_scratch_bytes.argtypes = []
    l.hq_noalloc_setup.restype = i32
    l.hq_noalloc_setup.argtypes = []
    l.hq_gemm_noalloc.restype = i32
    l.hq_gemm_noalloc.argtypes = [vp, vp, vp, vp, i32, i32, i32, i32, i32]
    l.hq_debug_gemm_timeline.restype = i32
    l.hq_debug_gemm_timeline.argtypes = [vp, i32, vp, vp, vp, vp, i32, i32, i32, i32, i32, vp]
    l.hq_debug_copy_probe.restype = i32
    l.hq_debug_copy_probe.argtypes = [vp, vp, ctypes.c_size_t, i32, i32]
    l.hq_debug_read_probe.restype = i32
    l.hq_debug_read_probe.argtypes = [vp, vp, ctypes.c_size_t, vp]
    l.hq_debug_kv_row.restype = i32
    l.hq_debug_kv_row.argtypes = [vp, i32, i32, i32, i32, vp]
    l.hq_debug_step_trace.restype = i32
    l.hq_debug_step_trace.argtypes = [vp, vp, i32]
    l.hq_debug_trace.restype = i32
    l.hq_debug_trace.argtypes = [vp, vp, i32]
    l.hq_last_error.restype = ctypes.c_char_p
    l.hq_last_error.argtypes = []
    l.hq_version.restype = ctypes.c_char_p
    l.hq_version.argtypes = []
    if path is None:
        _lib = l
    return l


def _check(rc: int):
    if rc != HQ_OK:
        raise HQError(rc, load_library().hq_last_error().decode())


def version() -> str:
    return load_library().hq_version().decode()


def make_config(*, n_layers, hidden, n_heads, n_kv_heads, head_dim, ffn, vocab, rms_eps, rope_theta,
                max_batch=1, max_seq=4352, flags=0, weight_dtype=DTYPE_BF16) -> Config:
    return Config(n_layers, hidden, n_heads, n_kv_heads, head_dim, ffn, vocab, rms_eps, rope_theta,
                  max_batch, max_seq, weight_dtype, flags)


def quantize_q4(w, stream=None):
    """hq_quantize_q4 on a CUDA bf16 tensor [N, K]: returns (codes uint8 [N, K/2], exponent bytes uint8 [N, K/32])."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream(w.device)
    n, k = w.shape
    codes = torch.empty((n, k // 2), dtype=torch.uint8, device=w.device)
    exps = torch.empty((n, k // 32), dtype=torch.uint8, device=w.device)
    _check(load_library().hq_quantize_q4(st.cuda_stream, w.data_ptr(), n, k, codes.data_ptr(), exps.data_ptr()))
    return codes, exps


def dequantize_q4(codes, exps, stream=None):
    """hq_dequantize_q4: (codes, exponent bytes) -> CUDA bf16 tensor [N, K] of w' = q * 2^e."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream(codes.device)
    n, k = codes.shape[0], codes.shape[1] * 2
    w = torch.empty((n, k), dtype=torch.bfloat16, device=codes.device)
    _check(load_library().hq_dequantize_q4(st.cuda_stream, codes.data_ptr(), exps.data_ptr(), n, k, w.data_ptr()))
    return w


def workspace_bytes(cfg: Config) -> int:
    return int(load_library().hq_workspace_bytes(ctypes.byref(cfg)))


LAYER_TENSORS = ("attn_norm", "wq", "wk", "wv", "wo", "ffn_norm", "w_gate", "w_up", "w_down")


class Model:
    """Owns the torch device tensors (weights, workspace) and the opaque hq_model handle.

    Method names follow the C ABI: prefill, decode_step, decode_run, decode_logits, get_hidden,
    sync, seq_len, kv_reset, kernel_count, bench_kernel.
    """

    def __init__(self, cfg: Config, embedding, final_norm, layers: Sequence[Dict[str, "object"]],
                 lm_head=None, stream=None, guard_bytes: int = 0, q4=None):
        """q4 (HQ_Q4 models): dict with per-layer lists "w_gate", "w_up", "w_down" of (codes, exps) CUDA tensors and
        "lm_head": (codes, exps); the bf16 tensors passed for those matrices must be their dequantised values."""
        import torch
        if not torch.cuda.is_available():
            raise HQError(HQ_ERR_CUDA, "no CUDA device: hq has no CPU fallback")
        self._torch = torch
        self._lib = load_library()
        self.cfg = cfg
        self.device = embedding.device
        for t in [embedding, final_norm] + [l[k] for l in layers for k in LAYER_TENSORS]:
            if t.dtype != torch.bfloat16 or not t.is_cuda or not t.is_contiguous():
                raise HQError(HQ_ERR_INVALID_ARG, "weights must be contiguous CUDA bfloat16 tensors")
        self._keep = [embedding, final_norm, layers, lm_head]
        self._q4 = q4
        # a dedicated stream: CUDA graphs cannot be captured on the legacy default stream
        self.stream = stream if stream is not None else torch.cuda.Stream(self.device)
        torch.cuda.synchronize(self.device)     # weight uploads on the current stream are done
        nbytes = workspace_bytes(cfg)
        if nbytes == 0:
            _check(HQ_ERR_INVALID_ARG)
        # guard_bytes (a multiple of 256): canary regions in front of and behind the workspace (tests: guards_intact())
        self._guard = int(guard_bytes)
        self._ws_alloc = torch.empty(nbytes + 2 * self._guard, dtype=torch.uint8, device=self.device)
        if self._guard:
            self._ws_alloc[:self._guard] = 0xA5
            self._ws_alloc[self._guard + nbytes:] = 0xA5
        self.workspace = self._ws_alloc[self._guard:self._guard + nbytes]
        arrays = {}
        for k in LAYER_TENSORS:
            arr = (ctypes.c_void_p * cfg.n_layers)(*[layers[l][k].data_ptr() for l in range(cfg.n_layers)])
            arrays[k] = arr
        head = embedding if lm_head is None else lm_head
        w = Weights(embedding.data_ptr(), *[ctypes.cast(arrays[k], _vpp) for k in LAYER_TENSORS],
                    final_norm.data_ptr(), head.data_ptr())
        h = ctypes.c_void_p()
        with torch.cuda.device(self.device):     # the library creates the model on the CURRENT device
            if q4 is None:
                _check(self._lib.hq_model_create(ctypes.byref(cfg), ctypes.byref(w), self.workspace.data_ptr(),
                                                 nbytes, self.stream.cuda_stream, ctypes.byref(h)))
            else:
                qa = {}
                for name in ("w_gate", "w_up", "w_down"):
                    for j, kind in enumerate(("codes", "exps")):
                        qa[name + "_" + kind] = (ctypes.c_void_p * cfg.n_layers)(*[q4[name][l][j].data_ptr() for l in range(cfg.n_layers)])
                wq = WeightsQ4(*[ctypes.cast(qa[n + "_" + k], _vpp) for n in ("w_gate", "w_up", "w_down") for k in ("codes", "exps")],
                               q4["lm_head"][0].data_ptr(), q4["lm_head"][1].data_ptr())
                _check(self._lib.hq_model_create_q4(ctypes.byref(cfg), ctypes.byref(w), ctypes.byref(wq), self.workspace.data_ptr(),
                                                    nbytes, self.stream.cuda_stream, ctypes.byref(h)))
        self._h = h
        self.vocab, self.hidden, self.n_layers = cfg.vocab, cfg.hidden, cfg.n_layers

    # -- construction helper: bf16 bit patterns (numpy uint16) -> device tensors ---------------------
    @classmethod
    def from_bf16_bits(cls, shape, embedding_bits: np.ndarray, final_norm_bits: np.ndarray,
                       layer_bits: List[Dict[str, np.ndarray]], *, max_batch=1, max_seq=4352, flags=0,
                       device="cuda:0", stream=None, guard_bytes: int = 0) -> "Model":
        import torch

        def up(a: np.ndarray):
            t = torch.from_numpy(np.ascontiguousarray(a).view(np.int16)).to(device)
            return t.view(torch.bfloat16)

        cfg = make_config(n_layers=shape.n_layers, hidden=shape.hidden, n_heads=shape.n_heads,
                          n_kv_heads=shape.n_kv_heads, head_dim=shape.head_dim, ffn=shape.ffn,
                          vocab=shape.vocab, rms_eps=shape.rms_eps, rope_theta=shape.rope_theta,
                          max_batch=max_batch, max_seq=max_seq, flags=flags)
        layers = [{k: up(l[k]) for k in LAYER_TENSORS} for l in layer_bits]
        return cls(cfg, up(embedding_bits), up(final_norm_bits), layers, stream=stream, guard_bytes=guard_bytes)

    @classmethod
    def from_bf16_bits_q4(cls, shape, embedding_bits: np.ndarray, final_norm_bits: np.ndarray,
                          layer_bits: List[Dict[str, np.ndarray]], *, max_batch=1, max_seq=4352, flags=0,
                          device="cuda:0", guard_bytes: int = 0) -> "Model":
        """HQ_Q4 model from bf16 bit patterns: FFN matrices and the (tied) embedding / LM head are quantised to hq4 on the
        device (hq_quantize_q4) and replaced by their dequantised values (hq_dequantize_q4); attention weights stay."""
        import torch

        def up(a: np.ndarray):
            return torch.from_numpy(np.ascontiguousarray(a).view(np.int16)).to(device).view(torch.bfloat16)

        cfg = make_config(n_layers=shape.n_layers, hidden=shape.hidden, n_heads=shape.n_heads,
                          n_kv_heads=shape.n_kv_heads, head_dim=shape.head_dim, ffn=shape.ffn,
                          vocab=shape.vocab, rms_eps=shape.rms_eps, rope_theta=shape.rope_theta,
                          max_batch=max_batch, max_seq=max_seq, flags=flags, weight_dtype=DTYPE_Q4)
        layers = [{k: up(l[k]) for k in LAYER_TENSORS} for l in layer_bits]
        q4 = {"w_gate": [], "w_up": [], "w_down": []}
        for l in layers:
            for name in ("w_gate", "w_up", "w_down"):
                ce = quantize_q4(l[name])
                q4[name].append(ce)
                l[name] = dequantize_q4(*ce)
        emb = up(embedding_bits)
        q4["lm_head"] = quantize_q4(emb)
        emb = dequantize_q4(*q4["lm_head"])
        torch.cuda.synchronize()
        return cls(cfg, emb, up(final_norm_bits), layers, guard_bytes=guard_bytes, q4=q4)

    def guards_intact(self) -> bool:
        """True when no byte of the canary regions around the workspace has been written (guard_bytes > 0)."""
        self.sync()
        g, n = self._guard, self.workspace.numel()
        return bool((self._ws_alloc[:g] == 0xA5).all().item() and (self._ws_alloc[g + n:] == 0xA5).all().item())

    def cfg_with_flags(self, flags: int) -> "Config":
        """A copy of this model's config with other HQ_FLAG_* bits (for a second model over the same weights)."""
        c = Config.from_buffer_copy(self.cfg)
        c.flags = flags
        return c

    def weight_tensors(self):
        """(embedding, final_norm, layers, lm_head) device tensors this model borrows."""
        return tuple(self._keep)

    def close(self):
        h, self._h = getattr(self, "_h", None), None
        if h:
            self._lib.hq_model_destroy(h)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the C ABI, one method per call -------------------------------------------------------------
    def prefill(self, tokens, logits=None, want_token: bool = True):
        """tokens: int array [batch, n_tokens] (or [n_tokens]) on the HOST.  Returns first tokens or None."""
        toks = np.ascontiguousarray(tokens, dtype=np.int32)
        if toks.ndim == 1:
            toks = toks[None, :]
        batch, n = toks.shape
        out = np.empty(batch, dtype=np.int32) if want_token else None
        _check(self._lib.hq_prefill(self._h, toks.ctypes.data, batch, n,
                                    logits.data_ptr() if logits is not None else None,
                                    out.ctypes.data if want_token else None))
        return out

    def decode_step(self, tokens_in=None, want_token: bool = True, out: Optional[np.ndarray] = None):
        tin = None if tokens_in is None else np.ascontiguousarray(tokens_in, dtype=np.int32).reshape(-1)
        if want_token and out is None:
            out = np.empty(max(1, self.cfg.max_batch), dtype=np.int32)
        _check(self._lib.hq_decode_step(self._h, tin.ctypes.data if tin is not None else None,
                                        out.ctypes.data if want_token else None))
        return out if want_token else None

    def decode_run(self, n_steps: int, want_tokens: bool = True, batch: int = 1):
        out = np.empty((n_steps, batch), dtype=np.int32) if want_tokens else None
        _check(self._lib.hq_decode_run(self._h, n_steps, out.ctypes.data if want_tokens else None))
        return out

    def verify_relay(self, envelope, answer) -> int:
        """hq_verify_relay: envelope and answer token arrays on the HOST; returns the number of accepted answer tokens."""
        env = np.ascontiguousarray(envelope, dtype=np.int32).reshape(-1)
        ans = np.ascontiguousarray(answer, dtype=np.int32).reshape(-1)
        toks = np.concatenate([env, ans])
        out = ctypes.c_int32()
        _check(self._lib.hq_verify_relay(self._h, toks.ctypes.data, env.size, ans.size, ctypes.byref(out)))
        return out.value

    def decode_logits(self, batch: int = 1):
        t = self._torch.empty((batch, self.vocab), dtype=self._torch.float32, device=self.device)
        _check(self._lib.hq_decode_logits(self._h, t.data_ptr()))
        self.sync()      # diagnostics: the copy ran on self.stream, the caller reads on another
        return t

    def get_hidden(self, layer: int, batch: int = 1):
        t = self._torch.empty((batch, self.hidden), dtype=self._torch.float32, device=self.device)
        _check(self._lib.hq_get_hidden(self._h, layer, t.data_ptr()))
        self.sync()
        return t

    def sync(self):
        _check(self._lib.hq_sync(self._h))

    def seq_len(self) -> int:
        v = ctypes.c_int32()
        _check(self._lib.hq_seq_len(self._h, ctypes.byref(v)))
        return v.value

    def kv_reset(self):
        _check(self._lib.hq_kv_reset(self._h))

    def kernel_count(self) -> int:
        return int(self._lib.hq_kernel_count(self._h))

    def decode_path(self) -> str:
        return self._lib.hq_decode_path(self._h).decode()

    def kv_row(self, which: str, layer: int, pos: int, seq: int = 0):
        """Cached K ("k", rotated) or V ("v") of one position: fp16 device tensor [n_kv_heads * 64]."""
        t = self._torch.empty(self.cfg.n_kv_heads * 64, dtype=self._torch.float16, device=self.device)
        _check(self._lib.hq_debug_kv_row(self._h, 0 if which == "k" else 1, layer, seq, pos, t.data_ptr()))
        self.sync()
        return t

    def step_trace(self, on: bool = True):
        """Step timeline (hq_debug_step_trace): returns the int64 [slots][4] device tensor, initialised, or None (off)."""
        if not on:
            _check(self._lib.hq_debug_step_trace(self._h, None, 0))
            self._step_trace = None
            return None
        slots = 2 + 3 * self.n_layers
        t = self._torch.zeros((slots, 4), dtype=self._torch.int64, device=self.device)
        t[:, :2] = (1 << 63) - 1      # atomicMin targets (unsigned compare: below every real stamp's complement)
        self._step_trace = t
        _check(self._lib.hq_debug_step_trace(self._h, t.data_ptr(), slots))
        return t

    def debug_trace(self, cap: int = 0):
        """Switch the attention block's timeline on (cap > 0: returns the uint64 [n_ctas][cap] device tensor the next
        direct launches fill) or off (cap == 0)."""
        if cap <= 0:
            _check(self._lib.hq_debug_trace(self._h, None, 0))
            self._trace = None
            return None
        n_sms = self._torch.cuda.get_device_properties(self.device).multi_processor_count
        self._trace = self._torch.zeros((n_sms, cap), dtype=self._torch.int64, device=self.device)
        _check(self._lib.hq_debug_trace(self._h, self._trace.data_ptr(), cap))
        return self._trace

    def bench_kernel(self, which: int, reps: int) -> int:
        b = ctypes.c_int64()
        _check(self._lib.hq_bench_kernel(self._h, which, reps, ctypes.byref(b)))
        return b.value


def noalloc_scratch_bytes() -> int:
    """hq_noalloc_scratch_bytes: size of the library's static scratch array (include/hq_noalloc.h)."""
    return int(load_library().hq_noalloc_scratch_bytes())


def noalloc_setup(device=None):
    """hq_noalloc_setup for `device` (default: torch's current device): once per device, before any no-allocation region."""
    import torch
    with torch.cuda.device(device if device is not None else torch.cuda.current_device()):
        _check(load_library().hq_noalloc_setup())


def gemm_noalloc(w, x, out, *, token_tile: int = 128, splits: int = 1, stream=None):
    """hq_gemm_noalloc on torch CUDA tensors: bf16 w [N,K], bf16 x planes [2,T,K] (hi, lo), fp32 out [T,N]; allocates nothing."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream(w.device)
    n_rows, k = w.shape
    with torch.cuda.device(w.device):
        _check(load_library().hq_gemm_noalloc(st.cuda_stream, w.data_ptr(), x.data_ptr(), out.data_ptr(), n_rows, k, x.shape[1],
                                              token_tile, splits))


def read_probe(buf, result, stream=None):
    """hq_debug_read_probe: one read-only pass over the CUDA tensor buf; result = uint32/int32 CUDA tensor [1]."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream(buf.device)
    _check(load_library().hq_debug_read_probe(st.cuda_stream, buf.data_ptr(), buf.numel() * buf.element_size(),
                                              result.data_ptr()))


def copy_probe(buf, copy_bytes: int, n_ctas: int, stream=None) -> int:
    """hq_debug_copy_probe on a CUDA tensor; returns the bytes one launch streams."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream(buf.device)
    nbytes = buf.numel() * buf.element_size()
    _check(load_library().hq_debug_copy_probe(st.cuda_stream, buf.data_ptr(), nbytes, copy_bytes, n_ctas))
    return n_ctas * (nbytes // 65536 // n_ctas) * 65536


def debug_gemm(mode: int, w, x, out, *, w2=None, token_tile: int = 128, splits: int = 1, stream=None, trace=None):
    """hq_debug_gemm on torch CUDA tensors: bf16 w [N,K], bf16 x planes [2,T,K] (hi, lo); out fp32 [T,N],
    or bf16 planes [2,T,N] for modes 2 and 3.  trace: int64 CUDA tensor [CTAs, 8] -> hq_debug_gemm_timeline."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream(w.device)
    n_rows, k = w.shape
    args = (st.cuda_stream, mode, w.data_ptr(), w2.data_ptr() if w2 is not None else None,
            x.data_ptr(), out.data_ptr(), n_rows, k, x.shape[1], token_tile, splits)
    if trace is None:
        _check(load_library().hq_debug_gemm(*args))
    else:
        _check(load_library().hq_debug_gemm_timeline(*args, trace.data_ptr()))
