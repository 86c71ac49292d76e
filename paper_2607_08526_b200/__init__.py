"""aria-b200: quantized DiT linear layers (W8A8 / W4A16) of arxiv/paper_2607_08526 for B200.

The product is the C-ABI library `libaria_b200.so` (include/aria.h) built from
csrc/; `binding` is its thin ctypes front end.  Importing this package loads
nothing: call `paper_2607_08526_b200.binding.lib()` (raises if the CUDA library
is missing -- there is no CPU fallback).
"""
__all__ = ["binding", "inputs"]
