"""ctypes front end of the CPU oracle (oracle/aria_oracle.c) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference leg may import this module.  It never imports the product package's
binding or CUDA library, and the product never imports it.

Every function is argument marshalling around one C routine; the arithmetic and
its citations (BASELINE.json configs C1-C5; SURVEY.md S8(c)
O1-O5) live in aria_oracle.c.  numpy arrays in, numpy arrays out.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from ctypes import POINTER, c_double, c_float, c_int, c_int8, c_int64, c_uint8, c_uint16

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "aria_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no fast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
               "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        L.oracle_bf16_bits_to_f32.restype = c_float
        L.oracle_bf16_bits_to_f32.argtypes = [c_uint16]
        L.oracle_fp16_bits_to_f32.restype = c_float
        L.oracle_fp16_bits_to_f32.argtypes = [c_uint16]
        L.oracle_f32_to_fp16_bits.restype = c_uint16
        L.oracle_f32_to_fp16_bits.argtypes = [c_float]
        L.oracle_f64_to_bf16_bits.restype = c_uint16
        L.oracle_f64_to_bf16_bits.argtypes = [c_double]
        L.oracle_gelu_erf.restype = c_double
        L.oracle_gelu_erf.argtypes = [c_double]
        L.oracle_quant_int8_rows.restype = None
        L.oracle_quant_int8_rows.argtypes = [POINTER(c_float), c_int64, c_int64, POINTER(c_int8),
                                             POINTER(c_float)]
        L.oracle_quant_int4_groups.restype = None
        L.oracle_quant_int4_groups.argtypes = [POINTER(c_float), c_int64, c_int64, c_int,
                                               POINTER(c_int8), POINTER(c_uint16), POINTER(c_uint8)]
        L.oracle_unpack_int4.restype = None
        L.oracle_unpack_int4.argtypes = [POINTER(c_uint8), c_int64, c_int64, POINTER(c_int8)]
        L.oracle_gemm_i8.restype = c_int64
        L.oracle_gemm_i8.argtypes = [POINTER(c_int8), POINTER(c_int8), c_int64, c_int64, c_int64,
                                     POINTER(c_int64)]
        L.oracle_epilogue_w8a8.restype = None
        L.oracle_epilogue_w8a8.argtypes = [POINTER(c_int64), POINTER(c_float), POINTER(c_float),
                                           POINTER(c_double), c_int, c_int64, c_int64,
                                           POINTER(c_double)]
        L.oracle_linear_w4a16.restype = None
        L.oracle_linear_w4a16.argtypes = [POINTER(c_float), POINTER(c_int8), POINTER(c_uint16),
                                          POINTER(c_double), c_int, c_int, c_int64, c_int64,
                                          c_int64, c_int, POINTER(c_double)]
        L.oracle_dequant_int4.restype = None
        L.oracle_dequant_int4.argtypes = [POINTER(c_int8), POINTER(c_uint16), c_int, c_int64,
                                          c_int64, c_int, POINTER(c_double)]
        L.oracle_linear_w8a16.restype = None
        L.oracle_linear_w8a16.argtypes = [POINTER(c_float), POINTER(c_int8), POINTER(c_float), POINTER(c_double),
                                          c_int, c_int, c_int64, c_int64, c_int64, POINTER(c_double)]
        L.oracle_steer.restype = None
        L.oracle_steer.argtypes = [POINTER(c_float), c_int64, c_int64, POINTER(c_float), c_double, c_double, c_int,
                                   POINTER(c_double)]
        L.oracle_norm_rows.restype = None
        L.oracle_norm_rows.argtypes = [POINTER(c_float), c_int64, c_int64, POINTER(c_float), POINTER(c_float), c_int,
                                       c_double, POINTER(c_double)]
        L.oracle_attention.restype = None
        L.oracle_attention.argtypes = [POINTER(c_float), c_int64, c_int64, c_int64, c_int64, c_double, POINTER(c_double)]
        L.oracle_round_out.restype = None
        L.oracle_round_out.argtypes = [POINTER(c_double), c_int64, c_int, POINTER(c_float)]
        L.oracle_num_threads.restype = c_int
        L.oracle_num_threads.argtypes = []
        _lib = L
    return _lib


def _p(a: np.ndarray, ct):
    return a.ctypes.data_as(POINTER(ct))


def _c(a, dtype) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=dtype)


ACT_NONE, ACT_GELU_ERF = 0, 1
OUT_F32, OUT_BF16 = 0, 1


def num_threads() -> int:
    return int(_load().oracle_num_threads())


# ------------------------------------------------------------- scalar helpers
def bf16_bits_to_f32(bits) -> np.ndarray:
    """bf16 bit patterns (uint16) -> fp32 values, exact."""
    b = np.asarray(bits, dtype=np.uint16)
    return (b.astype(np.uint32) << 16).view(np.float32)


def f32_to_fp16_bits(x: float) -> int:
    return int(_load().oracle_f32_to_fp16_bits(c_float(x)))


def fp16_bits_to_f32(h: int) -> float:
    return float(_load().oracle_fp16_bits_to_f32(c_uint16(h)))


def f64_to_bf16_bits(x: float) -> int:
    return int(_load().oracle_f64_to_bf16_bits(c_double(x)))


def gelu_erf(y: float) -> float:
    return float(_load().oracle_gelu_erf(c_double(y)))


# ------------------------------------------------------------------------ O1
def quant_int8_rows(A):
    """O1: per-row absmax/127 int8 quantisation.  A: fp32 [R,C] (bf16 inputs are
    passed already widened).  Returns (q int8 [R,C], s fp32 [R])."""
    A = _c(A, np.float32)
    R, C = A.shape
    q = np.empty((R, C), np.int8)
    s = np.empty((R,), np.float32)
    _load().oracle_quant_int8_rows(_p(A, c_float), R, C, _p(q, c_int8), _p(s, c_float))
    return q, s


# ------------------------------------------------------------------------ O2
def quant_int4_groups(W, group: int = 32):
    """O2: returns (codes int8 [N,K], sg_bits uint16 [N,K/G], packed uint8 [N,K/2])."""
    W = _c(W, np.float32)
    N, K = W.shape
    assert K % group == 0 and K % 2 == 0
    codes = np.empty((N, K), np.int8)
    sg = np.empty((N, K // group), np.uint16)
    packed = np.empty((N, K // 2), np.uint8)
    _load().oracle_quant_int4_groups(_p(W, c_float), N, K, group, _p(codes, c_int8),
                                     _p(sg, c_uint16), _p(packed, c_uint8))
    return codes, sg, packed


def unpack_int4(packed, K: int):
    packed = _c(packed, np.uint8)
    N = packed.shape[0]
    codes = np.empty((N, K), np.int8)
    _load().oracle_unpack_int4(_p(packed, c_uint8), N, K, _p(codes, c_int8))
    return codes


def dequant_int4(codes, sg_bits, variant: int = 0, group: int = 32):
    assert variant in (0, 1), "the oracle holds the definitions only (tests/kernel_models.py has the operand-format models)"
    codes = _c(codes, np.int8)
    sg_bits = _c(sg_bits, np.uint16)
    N, K = codes.shape
    out = np.empty((N, K), np.float64)
    _load().oracle_dequant_int4(_p(codes, c_int8), _p(sg_bits, c_uint16), variant, N, K, group,
                                _p(out, c_double))
    return out


# ------------------------------------------------------------------------ O3
def gemm_i8(Xq, Wq):
    """Exact int8 GEMM acc[m,n] = sum_k Xq[m,k]*Wq[n,k] (int64).  Asserts int32 fit."""
    Xq = _c(Xq, np.int8)
    Wq = _c(Wq, np.int8)
    M, K = Xq.shape
    N, K2 = Wq.shape
    assert K == K2
    acc = np.empty((M, N), np.int64)
    ovf = _load().oracle_gemm_i8(_p(Xq, c_int8), _p(Wq, c_int8), M, N, K, _p(acc, c_int64))
    assert ovf == 0, "int8 GEMM accumulator does not fit int32"
    return acc


def epilogue_w8a8(acc, sx, sw, bias=None, act: int = ACT_NONE):
    """y = acc*sx[m]*sw[n] + b[n] (+GELU) in fp64."""
    acc = _c(acc, np.int64)
    sx = _c(sx, np.float32)
    sw = _c(sw, np.float32)
    M, N = acc.shape
    y = np.empty((M, N), np.float64)
    b = None if bias is None else _c(bias, np.float64)
    _load().oracle_epilogue_w8a8(_p(acc, c_int64), _p(sx, c_float), _p(sw, c_float),
                                 None if b is None else _p(b, c_double), act, M, N,
                                 _p(y, c_double))
    return y


def linear_w8a8(X, Wq, sw, bias=None, act: int = ACT_NONE):
    """Whole W8A8 linear from fp32 X (O1 on X, then O3).  Returns dict with
    xq, sx, acc (int64), y (fp64)."""
    xq, sx = quant_int8_rows(X)
    acc = gemm_i8(xq, Wq)
    y = epilogue_w8a8(acc, sx, sw, bias, act)
    return {"xq": xq, "sx": sx, "acc": acc, "y": y}


# ------------------------------------------------------------------------ O4
def linear_w4a16(X, codes, sg_bits, bias=None, act: int = ACT_NONE, variant: int = 0,
                 group: int = 32):
    """O4: y fp64 [M,N].  X fp32 holding bf16 values; codes int8 [N,K].  variant 0: w^ = bf16_rne(q sg); 1: w^ = q sg."""
    assert variant in (0, 1), "the oracle holds the definitions only (tests/kernel_models.py has the operand-format models)"
    X = _c(X, np.float32)
    codes = _c(codes, np.int8)
    sg_bits = _c(sg_bits, np.uint16)
    M, K = X.shape
    N = codes.shape[0]
    y = np.empty((M, N), np.float64)
    b = None if bias is None else _c(bias, np.float64)
    _load().oracle_linear_w4a16(_p(X, c_float), _p(codes, c_int8), _p(sg_bits, c_uint16),
                                None if b is None else _p(b, c_double), act, variant, M, N, K,
                                group, _p(y, c_double))
    return y


# ------------------------------------------------------------------------ O6
def linear_w8a16(X, Wq, sw, bias=None, act: int = ACT_NONE, variant: int = 0):
    """O6 (q8 weight-only): y fp64 [M,N].  X fp32 holding bf16 values; Wq int8 [N,K]; sw fp32 [N]."""
    X = _c(X, np.float32)
    Wq = _c(Wq, np.int8)
    sw = _c(sw, np.float32)
    M, K = X.shape
    N = Wq.shape[0]
    y = np.empty((M, N), np.float64)
    b = None if bias is None else _c(bias, np.float64)
    _load().oracle_linear_w8a16(_p(X, c_float), _p(Wq, c_int8), _p(sw, c_float),
                                None if b is None else _p(b, c_double), act, variant, M, N, K, _p(y, c_double))
    return y


# ------------------------------------------------------------------------ O7
STEER_ADD, STEER_PROJECT = 0, 1


def steer(H, d, strength: float, hbar_norm: float = 1.0, op: int = STEER_ADD):
    """O7: eq. 2 additive injection (op 0) or per-token projection (op 1), fp64 out [M,D]."""
    H = _c(H, np.float32)
    d = _c(d, np.float32)
    M, D = H.shape
    out = np.empty((M, D), np.float64)
    _load().oracle_steer(_p(H, c_float), M, D, _p(d, c_float), float(strength), float(hbar_norm), op, _p(out, c_double))
    return out


# ------------------------------------------------------------------------ O8
NORM_LAYER, NORM_RMS = 0, 1


def norm_rows(X, gamma, beta=None, kind: int = NORM_LAYER, eps: float = 1e-5):
    """O8: LayerNorm (kind 0) / RMSNorm (kind 1) over the last axis, fp64 out [M,K]."""
    X = _c(X, np.float32)
    gamma = _c(gamma, np.float32)
    b = None if beta is None else _c(beta, np.float32)
    M, K = X.shape
    out = np.empty((M, K), np.float64)
    _load().oracle_norm_rows(_p(X, c_float), M, K, _p(gamma, c_float), None if b is None else _p(b, c_float), kind,
                             float(eps), _p(out, c_double))
    return out


def norm_quant_int8(X, gamma, beta=None, kind: int = NORM_LAYER, eps: float = 1e-5, dtype: int = 1):
    """O8 then O1: n = round_dtype(norm(X)) (the tensor an unfused norm kernel stores), (q, s) = O1(n)."""
    n = round_out(norm_rows(X, gamma, beta, kind, eps), dtype)
    q, s = quant_int8_rows(n)
    return n, q, s


# ------------------------------------------------------------------------ O9
def attention(QKV, B: int, S: int, H: int, Dh: int, scale: float | None = None):
    """O9: full softmax(q k^T * scale) v per (sequence, head), fp64 out [B*S, H*Dh]."""
    QKV = _c(QKV, np.float32)
    assert QKV.shape == (B * S, 3 * H * Dh)
    if scale is None:
        scale = 1.0 / np.sqrt(Dh)
    O = np.empty((B * S, H * Dh), np.float64)
    _load().oracle_attention(_p(QKV, c_float), B, S, H, Dh, float(scale), _p(O, c_double))
    return O


# ---------------------------------------------------------------- output cast
def round_out(y, dtype: int):
    """One rounding of fp64 y to fp32 (dtype 0) or bf16 (dtype 1, widened to fp32)."""
    y = _c(y, np.float64)
    out = np.empty(y.shape, np.float32)
    _load().oracle_round_out(_p(y, c_double), y.size, dtype, _p(out, c_float))
    return out
