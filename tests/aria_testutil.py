"""Helpers shared by the GPU parity tests: move seeded host arrays to the device, bring results
back, compare in the norms DESIGN.md states.  No method arithmetic here."""
import numpy as np
import torch


def dev_bf16(bits: np.ndarray) -> torch.Tensor:
    """bf16 bit patterns (uint16 numpy) -> cuda bfloat16 tensor with the same bits."""
    return torch.from_numpy(bits.view(np.int16).copy()).cuda().view(torch.bfloat16)


def dev_f32(x: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32)).cuda()


def dev_i8(x: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(x, dtype=np.int8)).cuda()


def host_f32(t: torch.Tensor) -> np.ndarray:
    """Device tensor (fp32 or bf16) -> fp32 numpy (bf16 widened exactly)."""
    return t.detach().float().cpu().numpy()


def host_bits16(t: torch.Tensor) -> np.ndarray:
    return t.detach().view(torch.int16).cpu().numpy().view(np.uint16)


def rel_err(got: np.ndarray, ref: np.ndarray) -> float:
    """north_star norm (reading R10): max |got - ref| / max |ref|."""
    return float(np.abs(got.astype(np.float64) - ref.astype(np.float64)).max() / np.abs(ref).max())


def bf16_ulp_diff(got_bits: np.ndarray, ref_bits: np.ndarray) -> np.ndarray:
    """Distance in bf16 ulps between two bf16 bit arrays (sign-magnitude -> ordered ints)."""
    def key(b):
        b = b.astype(np.int32)
        return np.where(b & 0x8000, -(b & 0x7FFF), b & 0x7FFF)
    return np.abs(key(got_bits) - key(ref_bits))


def check_bf16_out(got_bits: np.ndarray, ref64: np.ndarray, ref_bf16_bits: np.ndarray, eps_rel: float,
                   max_mismatch: float):
    """bf16 output gate (reading R9).  The kernel rounds an fp32 value that is within
    eps = eps_rel * max|ref| of the fp64 reference, so (a) every element lies within
    eps + half a bf16 ulp (<= 2^-8 |ref| + eps) of the reference, and (b) all but a small
    fraction (elements whose fp32 noise straddles a rounding boundary) equal bf16_rne(ref)
    bit for bit.  Returns the mismatch fraction."""
    got = (got_bits.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    eps = eps_rel * np.abs(ref64).max()
    bound = 2.0 ** -8 * np.abs(ref64) + eps + 2.0 ** -133
    assert np.all(np.abs(got - ref64) <= bound), float((np.abs(got - ref64) - bound).max())
    mism = float((got_bits != ref_bf16_bits).mean())
    assert mism <= max_mismatch, mism
    return mism
