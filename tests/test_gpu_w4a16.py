"""GPU parity, S4 (W4A16): packed codes / scales bit-exact (test_gpu_quant), output within 2e-2
of the oracle in the north_star norm -- against BOTH oracle variants (w^ rounded to bf16, and
exact q*sg; reading R12).  The kernel dequantises exactly, so the fp32 output is also held to a
much tighter bound against variant 0."""
import numpy as np
import pytest
import torch

from paper_2607_08526_b200 import inputs
from aria_testutil import check_bf16_out, dev_bf16, dev_f32, host_bits16, host_f32, rel_err

pytestmark = pytest.mark.gpu
TOL = 2e-2              # north_star: bf16 W4A16 output
TOL_F32_V0 = 2e-5       # fp32 output vs variant 0: only fp32 accumulation order differs


@pytest.fixture(scope="module")
def aria():
    from paper_2607_08526_b200 import binding
    binding.lib()
    return binding


def _case(aria, oracle, M, K, N, bias=True, act=0, seed=70):
    bits, x = inputs.normal_bf16((M, K), 1.0, seed, M * 13 + K * 7 + N)
    W = inputs.normal_f32((N, K), 0.02, seed, M * 13 + K * 7 + N + 1)
    bb, bf = inputs.normal_bf16((N,), 0.01, seed, M * 13 + K * 7 + N + 2)
    codes, sg, packed = oracle.quant_int4_groups(W)
    q4, s = aria.aria_quantize_weights_int4(dev_f32(W))
    assert np.array_equal(q4.cpu().numpy(), packed) and np.array_equal(host_bits16(s), sg)
    b64 = bf.astype(np.float64) if bias else None
    ref0 = oracle.linear_w4a16(x, codes, sg, b64, act, variant=0)
    ref1 = oracle.linear_w4a16(x, codes, sg, b64, act, variant=1)
    X = dev_bf16(bits)
    bd = dev_bf16(bb) if bias else None
    y32 = aria.aria_linear_w4a16(X, q4, s, bd, act, aria.F32)
    y16 = aria.aria_linear_w4a16(X, q4, s, bd, act, aria.BF16)
    torch.cuda.synchronize()
    e0, e1 = rel_err(host_f32(y32), ref0), rel_err(host_f32(y32), ref1)
    assert e0 <= TOL_F32_V0, e0
    assert e1 <= TOL, e1
    assert rel_err(host_f32(y16), ref0) <= TOL and rel_err(host_f32(y16), ref1) <= TOL
    check_bf16_out(host_bits16(y16), ref0, inputs.bf16_bits(oracle.round_out(ref0, oracle.OUT_BF16)),
                   TOL_F32_V0, 1e-2)


def test_single_tile_structured(aria, oracle):
    # sg = 1 everywhere, small-integer X: result is an exact integer, any layout slip shows
    M, K, N = 32, 128, 128
    rng = np.random.default_rng(71)
    W = rng.integers(-7, 8, size=(N, K)).astype(np.float32)
    W[:, 0::32] = 7.0
    x = rng.integers(-4, 5, size=(M, K)).astype(np.float32)
    codes, sg, packed = oracle.quant_int4_groups(W)
    assert np.all(sg == 0x3C00)
    q4, s = aria.aria_quantize_weights_int4(dev_f32(W))
    y = aria.aria_linear_w4a16(dev_bf16(inputs.bf16_bits(x)), q4, s, None, 0, aria.F32)
    assert np.array_equal(host_f32(y).astype(np.int64), x.astype(np.int64) @ W.astype(np.int64).T)


@pytest.mark.parametrize("M", [32, 512])
@pytest.mark.parametrize("K,N", [(1536, 4608), (1536, 6144), (6144, 1536)])
def test_c4_shapes(aria, oracle, M, K, N):
    # C4's M=4096 cases are checked on sampled rows in test_gpu_stack.py (oracle time)
    _case(aria, oracle, M, K, N)


@pytest.mark.parametrize("M,K,N", [(1, 32, 8), (17, 96, 40), (33, 160, 136), (64, 256, 128), (100, 1536, 264),
                                   (129, 192, 128), (300, 416, 392), (2000, 256, 1536)])  # last: TT = 192 tiles, ragged token tail
def test_ragged_shapes(aria, oracle, M, K, N):
    _case(aria, oracle, M, K, N, bias=(M % 2 == 1))


def test_gelu_epilogue(aria, oracle):
    _case(aria, oracle, 64, 512, 256, act=1)


def test_split_k_is_deterministic(aria, oracle):
    M, K, N = 32, 6144, 1536
    bits, x = inputs.normal_bf16((M, K), 1.0, 72, 0)
    W = inputs.normal_f32((N, K), 0.02, 72, 1)
    q4, s = aria.aria_quantize_weights_int4(dev_f32(W))
    X = dev_bf16(bits)
    ws = aria.workspace(aria.aria_workspace_bytes(M, K, N, aria.W4A16))
    ys = [host_bits16(aria.aria_linear_w4a16(X, q4, s, None, 0, aria.BF16, ws=ws)) for _ in range(5)]
    torch.cuda.synchronize()
    for y in ys[1:]:
        assert np.array_equal(y, ys[0])
