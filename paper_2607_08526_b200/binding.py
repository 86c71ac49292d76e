"""Thin ctypes binding of libaria_b200.so (include/aria.h).  Argument marshalling only: every
step of the path runs in the library's CUDA kernels.  PyTorch is used to own device memory and
streams.  There is no fallback: a missing library or a non-sm_100 device raises.

Functions carry the C entry points' names and argument order; tensors replace pointers, the
current torch CUDA stream replaces `stream`.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import c_char_p, c_int, c_size_t, c_void_p

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libaria_b200.so")

F32, BF16 = 0, 1
ACT_NONE, ACT_GELU_ERF = 0, 1
W8A8, W4A16, W8A16 = 0, 1, 2
STEER_ADD, STEER_PROJECT = 0, 1
NORM_LAYER, NORM_RMS = 0, 1

_lib = None


class AriaError(RuntimeError):
    pass


class aria_layer(ctypes.Structure):
    _fields_ = [("K", c_int), ("N", c_int), ("act", c_int), ("in_", c_void_p), ("wq", c_void_p),
                ("w_scale", c_void_p), ("bias", c_void_p), ("out", c_void_p)]


def lib() -> ctypes.CDLL:
    """Load the CUDA library (built in-tree by `python -m paper_2607_08526_b200.build`)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise AriaError(f"{LIB_PATH} is missing: run `python -m paper_2607_08526_b200.build` "
                            "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        L.aria_version.restype = c_char_p
        L.aria_status_string.restype = c_char_p
        L.aria_status_string.argtypes = [c_int]
        L.aria_workspace_bytes.restype = c_size_t
        L.aria_workspace_bytes.argtypes = [c_int, c_int, c_int, c_int]
        L.aria_workspace_bytes_host.restype = c_size_t
        L.aria_workspace_bytes_host.argtypes = [c_int, c_int, c_int, c_int, c_int]
        L.aria_quantize_weights_int8.argtypes = [c_void_p, c_int, c_int, c_int, c_void_p, c_void_p, c_void_p]
        L.aria_quantize_act_int8.argtypes = [c_void_p, c_int, c_int, c_int, c_void_p, c_void_p, c_void_p]
        L.aria_quantize_weights_int4.argtypes = [c_void_p, c_int, c_int, c_int, c_int, c_void_p, c_void_p, c_void_p]
        L.aria_linear_w8a8.argtypes = [c_void_p, c_int, c_int, c_int, c_void_p, c_void_p, c_int, c_void_p,
                                       c_int, c_int, c_void_p, c_int, c_void_p, c_size_t, c_void_p]
        L.aria_linear_w8a8_static_ws.argtypes = [c_void_p, c_int, c_int, c_int, c_void_p, c_void_p, c_int, c_void_p,
                                                 c_int, c_int, c_void_p, c_int, c_void_p]
        L.aria_static_ws_bytes.restype = c_size_t
        L.aria_static_ws_bytes.argtypes = []
        L.aria_linear_w8a8_q.argtypes = [c_void_p, c_void_p, c_int, c_int, c_void_p, c_void_p, c_int, c_void_p,
                                         c_int, c_int, c_void_p, c_int, c_void_p]
        L.aria_linear_w4a16.argtypes = [c_void_p, c_int, c_int, c_void_p, c_void_p, c_int, c_int, c_void_p,
                                        c_int, c_void_p, c_int, c_void_p, c_size_t, c_void_p]
        L.aria_linear_w8a16.argtypes = [c_void_p, c_int, c_int, c_void_p, c_void_p, c_int, c_void_p,
                                        c_int, c_void_p, c_int, c_void_p, c_size_t, c_void_p]
        L.aria_steer.argtypes = [c_void_p, c_int, c_int, c_int, c_void_p, c_void_p, ctypes.c_float, c_int, c_void_p]
        L.aria_norm_quantize_act_int8.argtypes = [c_void_p, c_int, c_int, c_int, c_void_p, c_void_p, c_int, ctypes.c_float,
                                                  c_void_p, c_void_p, c_void_p, c_void_p]
        L.aria_attention.argtypes = [c_void_p, c_int, c_int, c_int, c_int, ctypes.c_float, c_void_p, c_void_p, c_void_p]
        L.aria_round_act_int8.argtypes = [c_void_p, c_int, c_int, c_int, c_void_p, c_int, c_void_p, c_void_p, c_void_p]
        L.aria_gemm_i8_i32.argtypes = [c_void_p, c_void_p, c_int, c_int, c_int, c_void_p, c_void_p]
        L.aria_denoiser_linears.argtypes = [ctypes.POINTER(aria_layer), c_int, c_int, c_int, c_int,
                                            c_void_p, c_size_t, c_void_p]
        L.aria_denoiser_linears_host.argtypes = L.aria_denoiser_linears.argtypes
        L.aria_stack_plan_create.argtypes = [ctypes.POINTER(aria_layer), c_int, c_int, c_int, c_int,
                                             ctypes.POINTER(c_void_p)]
        L.aria_stack_plan_run.argtypes = [c_void_p, c_void_p]
        L.aria_stack_plan_is_streaming.argtypes = [c_void_p]
        L.aria_stack_plan_fallback_fired.argtypes = [c_void_p, ctypes.POINTER(c_int)]
        L.aria_w8a8_tile_plan.argtypes = [c_int, c_int, c_int, ctypes.POINTER(c_int), ctypes.POINTER(c_int)]
        L.aria_w4a16_tile_plan.argtypes = [c_int, c_int, c_int, c_int, ctypes.POINTER(c_int), ctypes.POINTER(c_int)]
        L.aria_tensor_peak.argtypes = [c_int, c_int, c_int, ctypes.c_double, ctypes.POINTER(ctypes.c_double), c_void_p]
        L.aria_stack_plan_destroy.argtypes = [c_void_p]
        L.aria_stack_plan_destroy.restype = None
        for name in EXPORTS:
            if name not in ("aria_version", "aria_status_string", "aria_workspace_bytes",
                            "aria_workspace_bytes_host", "aria_stack_plan_destroy", "aria_static_ws_bytes"):
                getattr(L, name).restype = c_int
        _lib = L
    return _lib


EXPORTS = ("aria_linear_w8a8_q", "aria_quantize_weights_int8", "aria_quantize_weights_int4", "aria_quantize_act_int8",
           "aria_linear_w8a8", "aria_linear_w4a16", "aria_denoiser_linears",
           "aria_denoiser_linears_host", "aria_workspace_bytes", "aria_workspace_bytes_host",
           "aria_status_string", "aria_gemm_i8_i32", "aria_version", "aria_stack_plan_create",
           "aria_stack_plan_run", "aria_stack_plan_is_streaming", "aria_stack_plan_destroy",
           "aria_stack_plan_fallback_fired", "aria_w8a8_tile_plan", "aria_w4a16_tile_plan", "aria_tensor_peak", "aria_linear_w8a16", "aria_steer",
           "aria_norm_quantize_act_int8", "aria_attention", "aria_round_act_int8", "aria_linear_w8a8_static_ws",
           "aria_static_ws_bytes")


def _check(rc: int, what: str):
    if rc != 0:
        raise AriaError(f"{what}: {lib().aria_status_string(rc).decode()} ({rc})")


def _stream() -> c_void_p:
    return c_void_p(torch.cuda.current_stream().cuda_stream)


def _dt(t: torch.Tensor) -> int:
    if t.dtype == torch.float32:
        return F32
    if t.dtype == torch.bfloat16:
        return BF16
    raise AriaError(f"unsupported dtype {t.dtype}")


def _ptr(t):
    if t is None:
        return c_void_p(0)
    assert t.is_contiguous()
    return c_void_p(t.data_ptr())


def _out_dtype(code: int):
    return torch.float32 if code == F32 else torch.bfloat16


def aria_version() -> str:
    return lib().aria_version().decode()


def aria_workspace_bytes(M: int, maxK: int, maxN: int, mode: int) -> int:
    return int(lib().aria_workspace_bytes(M, maxK, maxN, mode))


def aria_workspace_bytes_host(M: int, maxK: int, maxN: int, mode: int, io: int) -> int:
    return int(lib().aria_workspace_bytes_host(M, maxK, maxN, mode, io))


def workspace(nbytes: int, device="cuda") -> torch.Tensor:
    return torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=device)


def aria_quantize_weights_int8(W: torch.Tensor):
    N, K = W.shape
    Wq = torch.empty((N, K), dtype=torch.int8, device=W.device)
    sw = torch.empty((N,), dtype=torch.float32, device=W.device)
    _check(lib().aria_quantize_weights_int8(_ptr(W), _dt(W), N, K, _ptr(Wq), _ptr(sw), _stream()),
           "aria_quantize_weights_int8")
    return Wq, sw


def aria_quantize_act_int8(X: torch.Tensor):
    M, K = X.shape
    Xq = torch.empty((M, K), dtype=torch.int8, device=X.device)
    sx = torch.empty((M,), dtype=torch.float32, device=X.device)
    _check(lib().aria_quantize_act_int8(_ptr(X), _dt(X), M, K, _ptr(Xq), _ptr(sx), _stream()),
           "aria_quantize_act_int8")
    return Xq, sx


def aria_quantize_weights_int4(W: torch.Tensor, group: int = 32):
    N, K = W.shape
    Wq4 = torch.empty((N, K // 2), dtype=torch.uint8, device=W.device)
    sg = torch.empty((N, K // group), dtype=torch.int16, device=W.device)  # fp16 bit patterns
    _check(lib().aria_quantize_weights_int4(_ptr(W), _dt(W), N, K, group, _ptr(Wq4), _ptr(sg), _stream()),
           "aria_quantize_weights_int4")
    return Wq4, sg


def aria_linear_w8a8(X, Wq, w_scale, bias=None, act: int = ACT_NONE, yt: int = BF16, ws=None, out=None):
    M, K = X.shape
    N = Wq.shape[0]
    if ws is None:
        ws = workspace(aria_workspace_bytes(M, K, N, W8A8), X.device)
    Y = out if out is not None else torch.empty((M, N), dtype=_out_dtype(yt), device=X.device)
    _check(lib().aria_linear_w8a8(_ptr(X), _dt(X), M, K, _ptr(Wq), _ptr(w_scale), N, _ptr(bias),
                                  _dt(bias) if bias is not None else F32, act, _ptr(Y), yt, _ptr(ws),
                                  ws.numel(), _stream()), "aria_linear_w8a8")
    return Y


def aria_static_ws_bytes() -> int:
    return int(lib().aria_static_ws_bytes())


def aria_linear_w8a8_static_ws(X, Wq, w_scale, bias=None, act: int = ACT_NONE, yt: int = BF16, out=None):
    """aria_linear_w8a8 for callers that cannot allocate a workspace (real-time threads, plug-ins inside an engine
    that owns all GPU memory): the Xq / sx scratch is a fixed 16 MiB array inside the library, shared by all calls
    on the device.  Shapes beyond aria_static_ws_bytes() raise (ARIA_ERR_WORKSPACE).  Pass `out` to avoid the one
    allocation this Python wrapper would otherwise make for Y."""
    M, K = X.shape
    N = Wq.shape[0]
    Y = out if out is not None else torch.empty((M, N), dtype=_out_dtype(yt), device=X.device)
    _check(lib().aria_linear_w8a8_static_ws(_ptr(X), _dt(X), M, K, _ptr(Wq), _ptr(w_scale), N, _ptr(bias),
                                            _dt(bias) if bias is not None else F32, act, _ptr(Y), yt, _stream()),
           "aria_linear_w8a8_static_ws")
    return Y


def aria_linear_w8a8_q(Xq, x_scale, Wq, w_scale, bias=None, act: int = ACT_NONE, yt: int = BF16, out=None):
    M, K = Xq.shape
    N = Wq.shape[0]
    Y = out if out is not None else torch.empty((M, N), dtype=_out_dtype(yt), device=Xq.device)
    _check(lib().aria_linear_w8a8_q(_ptr(Xq), _ptr(x_scale), M, K, _ptr(Wq), _ptr(w_scale), N, _ptr(bias),
                                    _dt(bias) if bias is not None else F32, act, _ptr(Y), yt, _stream()),
           "aria_linear_w8a8_q")
    return Y


def aria_linear_w4a16(X, Wq4, g_scale, bias=None, act: int = ACT_NONE, yt: int = BF16, ws=None, out=None,
                      group: int = 32):
    M, K = X.shape
    N = Wq4.shape[0]
    if ws is None:
        ws = workspace(aria_workspace_bytes(M, K, N, W4A16), X.device)
    Y = out if out is not None else torch.empty((M, N), dtype=_out_dtype(yt), device=X.device)
    _check(lib().aria_linear_w4a16(_ptr(X), M, K, _ptr(Wq4), _ptr(g_scale), group, N, _ptr(bias), act,
                                   _ptr(Y), yt, _ptr(ws), ws.numel(), _stream()), "aria_linear_w4a16")
    return Y


def aria_linear_w8a16(X, Wq, w_scale, bias=None, act: int = ACT_NONE, yt: int = BF16, ws=None, out=None):
    M, K = X.shape
    N = Wq.shape[0]
    if ws is None:
        ws = workspace(aria_workspace_bytes(M, K, N, W8A16), X.device)
    Y = out if out is not None else torch.empty((M, N), dtype=_out_dtype(yt), device=X.device)
    _check(lib().aria_linear_w8a16(_ptr(X), M, K, _ptr(Wq), _ptr(w_scale), N, _ptr(bias), act, _ptr(Y), yt,
                                   _ptr(ws), ws.numel(), _stream()), "aria_linear_w8a16")
    return Y


def aria_steer(H: torch.Tensor, d: torch.Tensor, strength: torch.Tensor, hbar_norm: float = 1.0, op: int = STEER_ADD):
    """In place on H [M,D]; `strength` is a 1-element fp32 DEVICE tensor read by the kernel at run time."""
    M, D = H.shape
    assert d.dtype == torch.float32 and strength.dtype == torch.float32 and strength.is_cuda
    _check(lib().aria_steer(_ptr(H), _dt(H), M, D, _ptr(d), _ptr(strength), float(hbar_norm), op, _stream()),
           "aria_steer")
    return H


def aria_norm_quantize_act_int8(X, gamma, beta=None, norm: int = NORM_LAYER, eps: float = 1e-5, want_xn: bool = False,
                                out=None):
    """Norm fused with S1.  Returns (Xq, x_scale) or (Xq, x_scale, Xn) with want_xn; `out` = (Xq, x_scale) to reuse."""
    M, K = X.shape
    assert gamma.dtype == torch.float32 and (beta is None or beta.dtype == torch.float32)
    Xq, sx = out if out is not None else (torch.empty((M, K), dtype=torch.int8, device=X.device),
                                          torch.empty((M,), dtype=torch.float32, device=X.device))
    Xn = torch.empty_like(X) if want_xn else None
    _check(lib().aria_norm_quantize_act_int8(_ptr(X), _dt(X), M, K, _ptr(gamma), _ptr(beta), norm, float(eps), _ptr(Xn),
                                             _ptr(Xq), _ptr(sx), _stream()), "aria_norm_quantize_act_int8")
    return (Xq, sx, Xn) if want_xn else (Xq, sx)


def aria_attention(QKV, B: int, S: int, H: int, Dh: int = 64, scale: float | None = None, out=None, row_absmax=None):
    """QKV bf16 [B*S, 3*H*Dh] -> O bf16 [B*S, H*Dh].  row_absmax: zeroed fp32 [B*S] tensor or None."""
    assert QKV.dtype == torch.bfloat16 and tuple(QKV.shape) == (B * S, 3 * H * Dh)
    O = out if out is not None else torch.empty((B * S, H * Dh), dtype=torch.bfloat16, device=QKV.device)
    if scale is None:
        scale = Dh ** -0.5
    _check(lib().aria_attention(_ptr(QKV), B, S, H, Dh, float(scale), _ptr(O), _ptr(row_absmax), _stream()),
           "aria_attention")
    return O


def aria_round_act_int8(X, absmax, clear: bool = False, out=None):
    M, K = X.shape
    Xq, sx = out if out is not None else (torch.empty((M, K), dtype=torch.int8, device=X.device),
                                          torch.empty((M,), dtype=torch.float32, device=X.device))
    _check(lib().aria_round_act_int8(_ptr(X), _dt(X), M, K, _ptr(absmax), int(clear), _ptr(Xq), _ptr(sx), _stream()),
           "aria_round_act_int8")
    return Xq, sx


def aria_gemm_i8_i32(Xq, Wq):
    M, K = Xq.shape
    N = Wq.shape[0]
    acc = torch.empty((M, N), dtype=torch.int32, device=Xq.device)
    _check(lib().aria_gemm_i8_i32(_ptr(Xq), _ptr(Wq), M, N, K, _ptr(acc), _stream()), "aria_gemm_i8_i32")
    return acc


def make_layers(specs):
    """specs: iterable of dicts {K, N, act, in, wq, w_scale, bias, out}; `in`/`out` may be device
    tensors, host (pinned) tensors, raw ints, or None (chained input)."""
    arr = (aria_layer * len(specs))()
    for i, s in enumerate(specs):
        def p(v):
            if v is None:
                return None
            return v if isinstance(v, int) else v.data_ptr()
        arr[i] = aria_layer(s["K"], s["N"], s.get("act", ACT_NONE), p(s.get("in")), p(s["wq"]),
                            p(s["w_scale"]), p(s.get("bias")), p(s["out"]))
    return arr


def aria_denoiser_linears(layers, M: int, mode: int, io: int, ws: torch.Tensor):
    _check(lib().aria_denoiser_linears(layers, len(layers), M, mode, io, _ptr(ws), ws.numel(), _stream()),
           "aria_denoiser_linears")


def aria_denoiser_linears_host(layers, M: int, mode: int, io: int, ws: torch.Tensor):
    _check(lib().aria_denoiser_linears_host(layers, len(layers), M, mode, io, _ptr(ws), ws.numel(),
                                            _stream()), "aria_denoiser_linears_host")


def aria_stack_plan_create(layers, M: int, mode: int, io: int) -> c_void_p:
    """Returns the opaque plan handle; the caller keeps the layers' tensors alive and calls
    aria_stack_plan_destroy."""
    plan = c_void_p(0)
    _check(lib().aria_stack_plan_create(layers, len(layers), M, mode, io, ctypes.byref(plan)),
           "aria_stack_plan_create")
    return plan


def aria_stack_plan_run(plan: c_void_p):
    _check(lib().aria_stack_plan_run(plan, _stream()), "aria_stack_plan_run")


def aria_stack_plan_is_streaming(plan: c_void_p) -> int:
    """0: per-layer path; 1: stream kernel, fp16 operands (+ armed bf16 fallback); 2: stream kernel, bf16."""
    return int(lib().aria_stack_plan_is_streaming(plan))


def aria_stack_plan_fallback_fired(plan: c_void_p) -> int:
    """Synchronises the device, then reads the last run's domain flag (0 = stayed in the fp16 domain)."""
    torch.cuda.synchronize()
    fired = c_int(0)
    _check(lib().aria_stack_plan_fallback_fired(plan, ctypes.byref(fired)), "aria_stack_plan_fallback_fired")
    return fired.value


def aria_w8a8_tile_plan(M: int, N: int, sms: int = 148):
    bn, ctas = c_int(0), c_int(0)
    _check(lib().aria_w8a8_tile_plan(M, N, sms, ctypes.byref(bn), ctypes.byref(ctas)), "aria_w8a8_tile_plan")
    return bn.value, ctas.value


def aria_w4a16_tile_plan(M: int, N: int, K: int, sms: int = 148):
    tt, s = c_int(0), c_int(0)
    _check(lib().aria_w4a16_tile_plan(M, N, K, sms, ctypes.byref(tt), ctypes.byref(s)), "aria_w4a16_tile_plan")
    return tt.value, s.value


def aria_stack_plan_destroy(plan: c_void_p):
    lib().aria_stack_plan_destroy(plan)


def aria_tensor_peak(kind: int, ctas: int = 1, iters: int = 4096, seconds: float = 0.0):
    """Tensor-pipe issue-loop peak (measurement helper): kind 0 = int8, 1 = bf16.  Returns a dict."""
    out = (ctypes.c_double * 4)()
    _check(lib().aria_tensor_peak(kind, ctas, iters, float(seconds), out, _stream()), "aria_tensor_peak")
    return {"ops_per_s": out[0], "sm_mhz": out[1], "cycles_per_mma": out[2], "launches": int(out[3])}
