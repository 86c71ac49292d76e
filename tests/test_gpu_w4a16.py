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


def _edge_case(aria, oracle, M, K, N, x, W, seed):
    bits = inputs.bf16_bits(x)
    xb = inputs.bf16_as_f32(bits)
    codes, sg, packed = oracle.quant_int4_groups(W)
    q4, s = aria.aria_quantize_weights_int4(dev_f32(W))
    assert np.array_equal(q4.cpu().numpy(), packed) and np.array_equal(host_bits16(s), sg)
    bb, bf = inputs.normal_bf16((N,), 0.01, seed, 9)
    b64 = bf.astype(np.float64)
    ref0 = oracle.linear_w4a16(xb, codes, sg, b64, 0, variant=0)
    ref1 = oracle.linear_w4a16(xb, codes, sg, b64, 0, variant=1)
    ws = aria.workspace(aria.aria_workspace_bytes(M, K, N, aria.W4A16))
    y32 = aria.aria_linear_w4a16(dev_bf16(bits), q4, s, dev_bf16(bb), 0, aria.F32, ws=ws)
    y16 = aria.aria_linear_w4a16(dev_bf16(bits), q4, s, dev_bf16(bb), 0, aria.BF16, ws=ws)
    torch.cuda.synchronize()
    assert rel_err(host_f32(y32), ref0) <= TOL_F32_V0
    for r in (ref0, ref1):
        assert rel_err(host_f32(y16), r) <= TOL
    return sg


@pytest.mark.parametrize("M", [32, 300])
def test_edge_groups_and_outlier_activations(aria, oracle, M):
    """S4 edge cases through the GEMM itself: an all-zero group, a group with an
    fp16-SUBNORMAL scale, a group with a scale far above 64, C3-style x20 outlier channels in X."""
    K, N = 1536, 264
    W = inputs.normal_f32((N, K), 0.02, 73, 1)
    W[:, 32:64] = 0.0
    W[:, 96:128] = inputs.normal_f32((N, 32), 1.0, 73, 2) * np.float32(7e-6)
    W[:, 160:192] = inputs.normal_f32((N, 32), 1.0, 73, 3) * np.float32(200.0)
    x = inputs.normal_f32((M, K), 1.0, 73, 0)
    x[:, inputs.outlier_channels(K, 73, 5)] *= np.float32(20.0)
    sg = _edge_case(aria, oracle, M, K, N, x, W, 73)
    assert np.any(sg == 0) and np.any((sg != 0) & ((sg & 0x7C00) == 0)) and np.max(sg & 0x7FFF) > 0x53FF


@pytest.mark.parametrize("scale", [1.0e5 / 4.0, 2.0 ** -20])
def test_activations_beyond_fp16_range_and_far_below_it(aria, oracle, scale):
    """bf16 activations above 65504 and a tensor far below 2^-14: the bf16 GEMM takes both as they are."""
    M, K, N = 64, 512, 136
    x = inputs.normal_f32((M, K), 1.0, 74, 0) * np.float32(scale)
    W = inputs.normal_f32((N, K), 0.02, 74, 1)
    if scale > 1:
        assert np.abs(x).max() > 65504.0
    _edge_case(aria, oracle, M, K, N, x, W, 74)


def test_every_token_tile_variant_is_reached(aria, oracle):
    """The launcher's plan (aria_w4a16_tile_plan) reaches every compiled token tile TT and split-K; each of
    these shapes runs the variant named beside it (asserted on the host plan, computed on the device)."""
    import torch as _t
    sms = _t.cuda.get_device_properties(0).multi_processor_count
    want = {32: (32, 256, 1536), 64: (64, 18944, 256), 128: (512, 1536, 6144), 192: (2000, 1536, 256), 256: (1024, 4608, 256)}
    for tt, (M, N, K) in want.items():
        assert aria.aria_w4a16_tile_plan(M, N, K, sms)[0] == tt, (tt, aria.aria_w4a16_tile_plan(M, N, K, sms))
        _case(aria, oracle, M, K, N, seed=75)
    assert aria.aria_w4a16_tile_plan(512, 1536, 6144, sms)[1] > 1      # and split-K
