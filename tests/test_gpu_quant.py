"""GPU parity, S0 + S1: codes and scales must be BIT-EXACT against the oracle (north_star)."""
import numpy as np
import pytest
import torch

from paper_2607_08526_b200 import inputs
from aria_testutil import dev_bf16, dev_f32, host_bits16

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def aria():
    from paper_2607_08526_b200 import binding
    binding.lib()
    return binding


def _check_i8(aria, oracle, x_dev, x_host_f32, what):
    q, s = what(x_dev)
    torch.cuda.synchronize()
    qo, so = oracle.quant_int8_rows(x_host_f32)
    assert np.array_equal(s.cpu().numpy().view(np.uint32), so.view(np.uint32)), "scales differ"
    assert np.array_equal(q.cpu().numpy(), qo), "codes differ"


def test_act_int8_c1_fp32(aria, oracle):
    c = inputs.c1()
    _check_i8(aria, oracle, dev_f32(c["X"]), c["X"], aria.aria_quantize_act_int8)
    _check_i8(aria, oracle, dev_f32(c["W"]), c["W"], aria.aria_quantize_weights_int8)


@pytest.mark.parametrize("M,K", [(512, 1536), (200, 6144), (3, 32), (1, 8192 + 64), (37, 9984)])
def test_act_int8_bf16_shapes(aria, oracle, M, K):
    bits, x = inputs.normal_bf16((M, K), 1.0, 50, M * 100003 + K)
    _check_i8(aria, oracle, dev_bf16(bits), x, aria.aria_quantize_act_int8)


def test_act_int8_outliers_zero_rows_and_ties(aria, oracle):
    c = inputs.c3(M=256)
    x = c["X"].copy()
    x[5] = 0.0                                    # all-zero row -> scale 1, codes 0
    x[6] = 0.0
    x[6, 7] = -3.0                                # single non-zero
    x[7, :256] = (np.arange(256) - 128 + 0.5)     # exact .5 ties at scale 1 ...
    x[7, 256:] = 0
    x[7, 300] = 127.0                             # ... because absmax is exactly 127
    bits = inputs.bf16_bits(x)
    x = inputs.bf16_as_f32(bits)
    _check_i8(aria, oracle, dev_bf16(bits), x, aria.aria_quantize_act_int8)


def test_weights_int8_bf16_and_fp32(aria, oracle):
    W = inputs.normal_f32((768, 1536), 0.02, 51, 0)
    _check_i8(aria, oracle, dev_f32(W), W, aria.aria_quantize_weights_int8)
    bits = inputs.bf16_bits(W)
    _check_i8(aria, oracle, dev_bf16(bits), inputs.bf16_as_f32(bits), aria.aria_quantize_weights_int8)


@pytest.mark.parametrize("N,K", [(512, 1536), (136, 6144), (8, 32)])
def test_weights_int4(aria, oracle, N, K):
    W = inputs.normal_f32((N, K), 0.02, 52, N + K)
    W[0, :32] = 0.0                               # all-zero group
    if K >= 64:
        W[1, 32:64] *= np.float32(1e-5)           # fp16-subnormal scale
    codes, sg, packed = oracle.quant_int4_groups(W)
    q4, s = aria.aria_quantize_weights_int4(dev_f32(W))
    torch.cuda.synchronize()
    assert np.array_equal(host_bits16(s), sg), "group scales differ"
    assert np.array_equal(q4.cpu().numpy(), packed), "packed codes differ"
    bits = inputs.bf16_bits(W)
    codes, sg, packed = oracle.quant_int4_groups(inputs.bf16_as_f32(bits))
    q4, s = aria.aria_quantize_weights_int4(dev_bf16(bits))
    torch.cuda.synchronize()
    assert np.array_equal(host_bits16(s), sg) and np.array_equal(q4.cpu().numpy(), packed)


@pytest.mark.parametrize("dtype,M,K", [("bf16", 64, 1536), ("bf16", 40, 6144), ("bf16", 9, 9984), ("f32", 33, 1536),
                                       ("f32", 5, 6144)])
def test_round_act_with_a_too_small_absmax_saturates_instead_of_wrapping(aria, oracle, dtype, M, K):
    """aria_round_act_int8 takes the row maximum from the caller.  With a maximum BELOW the row's own
    (a stale buffer) the division-free rounding used to wrap (x/s = 130 -> code -126); aria.h promises the
    clamp.  Expected value without retyping the formula: quantising with absmax a' saturates exactly the
    elements above a', so it equals the oracle's S1 of the row clipped to +-a' (a' is a value of the row,
    hence the clipped row's own maximum).  Rows with a correct maximum stay bit-identical to S1, a NaN
    maximum means scale 1 with saturation, and clear=1 still zeroes the buffer.  All row-kernel variants."""
    if dtype == "bf16":
        bits, x = inputs.normal_bf16((M, K), 1.0, 52, M + K)
        X = dev_bf16(bits)
    else:
        x = inputs.normal_f32((M, K), 1.0, 52, M + K)
        X = dev_f32(x)
    ax = np.abs(x)
    amax = ax.max(axis=1).astype(np.float32)
    small = np.sort(ax, axis=1)[:, -K // 16].astype(np.float32)   # 1/16 of each row lies above it
    given = amax.copy()
    given[0::2] = small[0::2]                                     # even rows: too small; odd rows: correct
    clipped = np.clip(x, -given[:, None], given[:, None])
    qo, so = oracle.quant_int8_rows(clipped)
    buf = dev_f32(given)
    q, s = aria.aria_round_act_int8(X, buf, clear=True)
    torch.cuda.synchronize()
    assert np.array_equal(s.cpu().numpy().view(np.uint32), so.view(np.uint32))
    assert np.array_equal(q.cpu().numpy(), qo)
    assert int((q.cpu().numpy()[0::2] == 127).sum() + (q.cpu().numpy()[0::2] == -127).sum()) >= (M + 1) // 2 * (K // 16)
    assert not buf.any()                                          # cleared after it was read
    # NaN maximum: scale 1, codes clamp(rint(x), +-127) -- x scaled up so that saturation matters
    big = (x * np.float32(64.0)).astype(np.float32)
    Xb = dev_bf16(inputs.bf16_bits(big)) if dtype == "bf16" else dev_f32(big)
    q, s = aria.aria_round_act_int8(Xb, torch.full((M,), float("nan"), device="cuda"))
    torch.cuda.synchronize()
    assert np.all(s.cpu().numpy() == 1.0)
    assert np.array_equal(q.cpu().numpy(), np.clip(np.rint(big), -127, 127).astype(np.int8))
