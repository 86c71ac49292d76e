"""Models of a KERNEL'S OPERAND FORMAT -- test-side diagnostics, not definitions (R12b / R12c).

The small-M weight-streaming kernel (csrc/w4a16_stream.cu) feeds the tensor core fp16 operands.  The acceptance
gate of that path is north_star's: <= 2e-2 against the oracle's definitions (O4 variants 0 and 1), applied on every
stream-kernel test.  The two functions here only explain the residual: they restate what the kernel's operands
are, so a result that passes the gate can also be compared bit-closely with "the definition evaluated on those
operands".  They were variants 2 and 3 of oracle_linear_w4a16 until round 3 (note (a): a model of the
kernel belongs in tests/, oracle/ holds definitions only).  numpy's float16 is the rounding used; the oracle's own
fp16 conversions are pinned against it over all 65 536 patterns (tests/test_oracle_quant.py), and the pins of these
models are in tests/test_oracle_linear.py.

  fp16_operand  (R12b):  w^ = fp16_rn(q * sg)
  offset_binary (R12c):  w^ = fp16_rn((q + 8) * sg) - 8 * sg   -- the unsigned code is scaled and rounded to fp16,
                         the zero point is subtracted exactly (by the tensor core, on group sums of x)
"""
import numpy as np
from scipy.special import erf

FP16_OPERAND, OFFSET_BINARY = "fp16_operand", "offset_binary"


def dequant_int4(codes: np.ndarray, sg_bits: np.ndarray, model: str, group: int = 32) -> np.ndarray:
    """fp64 [N, K] weights as the stream kernel's tensor-core operand represents them."""
    s = np.repeat(np.ascontiguousarray(sg_bits, dtype=np.uint16).view(np.float16).astype(np.float32), group, axis=1)
    q = codes.astype(np.float32)
    if model == FP16_OPERAND:
        return (q * s).astype(np.float16).astype(np.float64)          # the fp32 product is exact (3 x 11 bits)
    if model == OFFSET_BINARY:
        return ((q + np.float32(8.0)) * s).astype(np.float16).astype(np.float64) - 8.0 * s.astype(np.float64)
    raise ValueError(model)


def linear_w4a16(X: np.ndarray, codes: np.ndarray, sg_bits: np.ndarray, bias, act: int, model: str) -> np.ndarray:
    """y = x w^T + b (+ GELU) in fp64 on the modelled operands.  X: fp32 holding bf16 values."""
    y = X.astype(np.float64) @ dequant_int4(codes, sg_bits, model).T
    if bias is not None:
        y = y + np.asarray(bias, dtype=np.float64)
    if act == 1:
        y = 0.5 * y * (1.0 + erf(y / np.sqrt(2.0)))
    return y
