"""aria_linear_w8a8_static_ws -- the W8A8 linear for callers that cannot allocate device memory.

Why the entry point exists: aria_linear_w8a8 wants a caller-provided workspace for the int8 codes and scales
that travel between its two kernels.  A real-time audio thread must not call cudaMalloc (process-wide lock,
possible device synchronisation, no latency bound); a plug-in inside an engine that already owns all GPU memory
gets out-of-memory from it; code that was only handed raw device pointers has no allocator at all.  For those
callers the scratch is a fixed 16 MiB array inside the library, shared by every call on the device.

What is checked here: the new entry point against the existing aria_linear_w8a8 on the same inputs, in the
north_star norm and tolerance the W8A8 parity tests use (tests/test_gpu_w8a8.py), on two calls in a row whose
shapes differ -- the second call finds the first call's codes and scales still in the array, at other offsets.
The file name sorts last on purpose: pytest -x stops at the first failure, so nothing can hide behind this test.
It passes alone in a fresh process (then its first call does the per-device address lookup) and after the
other tests.
"""
import ctypes

import numpy as np
import pytest
import torch

from paper_2607_08526_b200 import inputs
from aria_testutil import dev_bf16, dev_f32, host_f32, rel_err

TOL_F32 = 1e-3   # the W8A8 gate of tests/test_gpu_w8a8.py (north_star: max |diff| / max |ref| on the fp32 output)


def test_shapes_beyond_the_built_in_scratch_are_rejected_without_a_gpu():
    from paper_2607_08526_b200 import binding
    L = binding.lib()
    limit = binding.aria_static_ws_bytes()
    assert limit == 16 << 20
    buf = (ctypes.c_char * 4096)()
    p16 = (ctypes.addressof(buf) + 15) // 16 * 16
    # C3's down-projection input, 4096 x 6144 codes = 24 MiB: over the limit -> ARIA_ERR_WORKSPACE, before any CUDA call
    assert L.aria_linear_w8a8_static_ws(p16, 1, 4096, 6144, p16, p16, 1536, None, 0, 0, p16, 1, None) == -6
    # just over: 2048 x 8192 codes fill the array exactly, the scales no longer fit
    assert L.aria_linear_w8a8_static_ws(p16, 1, 2048, 8192, p16, p16, 1536, None, 0, 0, p16, 1, None) == -6
    # the usual validation still comes first
    assert L.aria_linear_w8a8_static_ws(None, 1, 4, 64, p16, p16, 16, None, 0, 0, p16, 1, None) == -1
    assert L.aria_linear_w8a8_static_ws(p16, 1, 4, 64, p16, p16, 12, None, 0, 0, p16, 1, None) == -2
    assert L.aria_linear_w8a8_static_ws(p16 + 4, 1, 4, 64, p16, p16, 16, None, 0, 0, p16, 1, None) == -3


@pytest.mark.gpu
def test_static_scratch_linear_matches_the_workspace_path_on_two_calls_in_a_row():
    from paper_2607_08526_b200 import binding as aria
    aria.lib()
    # call 1: C5's largest linear input that fits (2048 x 6144 -> 1536, GELU off), call 2: a ragged small shape with GELU
    cases = [(2048, 6144, 1536, aria.ACT_NONE, 71), (300, 416, 392, aria.ACT_GELU_ERF, 72)]
    prepared = []
    for (M, K, N, act, seed) in cases:
        bits, _ = inputs.normal_bf16((M, K), 1.0, seed, 0)
        W = inputs.normal_f32((N, K), 0.02, seed, 1)
        b = inputs.normal_f32((N,), 0.01, seed, 2)
        wq, sw = aria.aria_quantize_weights_int8(dev_f32(W))
        X, bias = dev_bf16(bits), dev_f32(b)
        ref = aria.aria_linear_w8a8(X, wq, sw, bias, act, aria.F32)           # existing path, caller's workspace
        out = torch.full_like(ref, float("nan"))
        prepared.append((X, wq, sw, bias, act, ref, out))
    torch.cuda.synchronize()
    # the two calls under test, back to back on one stream, outputs pre-allocated: nothing is allocated in between
    for (X, wq, sw, bias, act, ref, out) in prepared:
        aria.aria_linear_w8a8_static_ws(X, wq, sw, bias, act, aria.F32, out=out)
    torch.cuda.synchronize()
    for (X, wq, sw, bias, act, ref, out) in prepared:
        got, want = host_f32(out), host_f32(ref)
        assert np.isfinite(got).all()
        e = rel_err(got, want)
        assert e <= TOL_F32, e
    # an oversized shape is refused on the device too, and leaves Y alone
    M, K, N = 4096, 6144, 64
    X = torch.zeros((M, K), dtype=torch.bfloat16, device="cuda")
    wq = torch.zeros((N, K), dtype=torch.int8, device="cuda")
    sw = torch.ones((N,), dtype=torch.float32, device="cuda")
    Y = torch.full((M, N), 7.0, dtype=torch.float32, device="cuda")
    with pytest.raises(aria.AriaError, match="workspace"):
        aria.aria_linear_w8a8_static_ws(X, wq, sw, None, aria.ACT_NONE, aria.F32, out=Y)
    torch.cuda.synchronize()
    assert bool((Y == 7.0).all())
