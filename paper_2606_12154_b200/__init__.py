"""hq — B200-native prefill + streaming decode of a 1B-class Llama-style decoder behind a C ABI.

The product is ``libhq.so`` (hand-written CUDA for sm_100a, see ``csrc/`` and ``include/hq.h``);
this package is only the argument-marshalling binding.  There is no CPU fallback: importing the
binding without a built library, or creating a model without a CUDA device, fails loudly.
"""
from .binding import (HQError, Model, FLAG_CAPTURE_HIDDEN, FLAG_NO_GRAPH, FLAG_NO_PDL, FLAG_KERNEL_PER_ROW, FLAG_VERIFY,  # noqa: F401
                      load_library, workspace_bytes, version, debug_gemm, gemm_noalloc, noalloc_setup, noalloc_scratch_bytes, read_probe, copy_probe, quantize_q4, dequantize_q4, DECLARED_SYMBOLS)
