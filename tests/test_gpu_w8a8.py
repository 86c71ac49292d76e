"""GPU parity, S2 + S3 (W8A8): int32 accumulators bit-exact; fp32 output within 1e-3 of the
oracle in the north_star norm (reading R10); bf16 output == bf16(oracle) up to 1 ulp on a
small fraction (reading R9)."""
import numpy as np
import pytest
import torch

from paper_2607_08526_b200 import inputs
from aria_testutil import check_bf16_out, dev_bf16, dev_f32, dev_i8, host_bits16, host_f32, rel_err

pytestmark = pytest.mark.gpu
TOL_F32 = 1e-3          # north_star: max relative error (vs output magnitude) on the fp32 output


@pytest.fixture(scope="module")
def aria():
    from paper_2607_08526_b200 import binding
    binding.lib()
    return binding


def test_acc_structured_single_tile(aria, oracle):
    # index-coded operands localise any layout / descriptor mistake
    M, N, K = 128, 64, 128
    Xq = np.zeros((M, K), np.int8)
    Xq[np.arange(M), np.arange(M) % K] = 1                       # one-hot rows
    Wq = ((np.arange(N)[:, None] * 7 + np.arange(K)[None, :] * 3) % 251 - 125).astype(np.int8)
    acc = aria.aria_gemm_i8_i32(dev_i8(Xq), dev_i8(Wq)).cpu().numpy()
    assert np.array_equal(acc.astype(np.int64), oracle.gemm_i8(Xq, Wq))


@pytest.mark.parametrize("M,N,K", [(128, 256, 256), (64, 256, 256), (512, 1536, 1536), (300, 392, 416),
                                   (1, 8, 32), (129, 264, 6144), (1000, 4608, 1536)])
def test_acc_bit_exact(aria, oracle, M, N, K):
    rng = np.random.default_rng([60, M, N, K])
    Xq = rng.integers(-127, 128, size=(M, K), dtype=np.int8)
    Wq = rng.integers(-127, 128, size=(N, K), dtype=np.int8)
    acc = aria.aria_gemm_i8_i32(dev_i8(Xq), dev_i8(Wq)).cpu().numpy()
    ref = oracle.gemm_i8(Xq, Wq)
    assert np.array_equal(acc.astype(np.int64), ref)


# (M, N) -> (BN, CTAS) on 148 SMs (tests/test_abi.py pins these on the host); K small keeps the oracle quick
TILE_VARIANT_SHAPES = {(64, 1): (64, 256), (128, 1): (128, 18944), (192, 1): (128, 28416), (256, 1): (100, 37888),
                       (128, 2): (512, 1536), (192, 2): (2048, 1536), (256, 2): (1000, 4608)}


@pytest.mark.parametrize("variant", sorted(TILE_VARIANT_SHAPES))
def test_acc_bit_exact_in_every_tile_variant(aria, oracle, variant):
    """Every compiled (BN, CTAS) instantiation of the W8A8 GEMM, reached through the launcher's own plan
    (the CTAS = 1 / BN >= 128 variants had no test)."""
    M, N = TILE_VARIANT_SHAPES[variant]
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    assert aria.aria_w8a8_tile_plan(M, N, sms) == variant
    K = 160
    rng = np.random.default_rng([63, M, N])
    Xq = rng.integers(-127, 128, size=(M, K), dtype=np.int8)
    Wq = rng.integers(-127, 128, size=(N, K), dtype=np.int8)
    acc = aria.aria_gemm_i8_i32(dev_i8(Xq), dev_i8(Wq)).cpu().numpy()
    assert np.array_equal(acc.astype(np.int64), oracle.gemm_i8(Xq, Wq))


@pytest.mark.parametrize("M,N,K", [(4096, 6144, 1536), (4096, 1536, 6144)])
def test_acc_bit_exact_full_size_multi_wave(aria, oracle, M, N, K):
    """C3's GEMMs at full size: 2-6 waves of the persistent tile loop with both TMEM accumulators in
    flight, raw int32 output.  64 sampled rows (first / last row of the first / last tile included) x all
    N columns against the oracle; a row of acc depends only on its own row of Xq."""
    rng = np.random.default_rng([64, M, N, K])
    Xq = rng.integers(-127, 128, size=(M, K), dtype=np.int8)
    Wq = rng.integers(-127, 128, size=(N, K), dtype=np.int8)
    acc = aria.aria_gemm_i8_i32(dev_i8(Xq), dev_i8(Wq))
    torch.cuda.synchronize()
    rows = np.sort(np.random.default_rng(65).choice(M, size=64, replace=False))
    rows[:4] = (0, 127, 128, 255)
    rows[-2:] = (M - 256, M - 1)
    rows = np.unique(rows)
    ref = oracle.gemm_i8(Xq[rows], Wq)
    assert np.array_equal(acc[torch.from_numpy(rows).cuda()].cpu().numpy().astype(np.int64), ref)
    # and a cheap whole-matrix property: column sums of acc equal (column sums of Xq) . Wq^T exactly
    colsum = acc.to(torch.int64).sum(dim=0).cpu().numpy()
    assert np.array_equal(colsum, Xq.astype(np.int64).sum(axis=0) @ Wq.astype(np.int64).T)


def test_acc_extreme_values(aria, oracle):
    K = 6144
    Xq = np.full((128, K), 127, np.int8)
    Wq = np.full((64, K), 127, np.int8)
    Wq[1::2] = -127
    acc = aria.aria_gemm_i8_i32(dev_i8(Xq), dev_i8(Wq)).cpu().numpy()
    assert np.all(acc[:, 0::2] == 99096576) and np.all(acc[:, 1::2] == -99096576)


def _linear_case(aria, oracle, Xdev, Xf32, W, bias_dev, bias_f64, act, yt_list):
    wq_d, sw_d = aria.aria_quantize_weights_int8(dev_f32(W))
    wq, sw = oracle.quant_int8_rows(W)
    assert np.array_equal(wq_d.cpu().numpy(), wq)
    ref = oracle.linear_w8a8(Xf32, wq, sw, bias_f64, act)["y"]
    out = {}
    for yt in yt_list:
        y = aria.aria_linear_w8a8(Xdev, wq_d, sw_d, bias_dev, act, yt)
        torch.cuda.synchronize()
        if yt == aria.F32:
            e = rel_err(host_f32(y), ref)
            assert e <= TOL_F32, e
            out["f32_err"] = e
        else:
            ref_bits = inputs.bf16_bits(oracle.round_out(ref, oracle.OUT_BF16))
            out["bf16_mismatch"] = check_bf16_out(host_bits16(y), ref, ref_bits, 1e-5,
                                                      2e-2 if act else 5e-3)  # erff noise + (-0 vs -1e-14) tails
    return out


def test_c1_tiny_fp32(aria, oracle):
    c = inputs.c1()
    _linear_case(aria, oracle, dev_f32(c["X"]), c["X"], c["W"], dev_f32(c["b"]), c["b"].astype(np.float64),
                 aria.ACT_NONE, [aria.F32])


def test_c2_attention_projections(aria, oracle):
    c = inputs.c2()
    X = dev_bf16(c["X_bits"])
    for Wn, bn in (("Wqkv", "bqkv"), ("Wout", "bout")):
        bb, bf = c[bn]
        _linear_case(aria, oracle, X, c["X"], c[Wn], dev_bf16(bb), bf.astype(np.float64), aria.ACT_NONE,
                     [aria.F32, aria.BF16])


def test_c3_mlp_outliers_teacher_forced(aria, oracle):
    # reduced M (oracle finishes in seconds); full-size rows are sampled in test_gpu_stack.py
    c = inputs.c3(M=384)
    X = dev_bf16(c["X_bits"])
    bu_b, bu = c["bup"]
    bd_b, bd = c["bdown"]
    _linear_case(aria, oracle, X, c["X"], c["Wup"], dev_bf16(bu_b), bu.astype(np.float64), aria.ACT_GELU_ERF,
                 [aria.F32, aria.BF16])
    # teacher forcing (reading O5): the down-projection's oracle takes the GPU's own bf16 H
    wq_d, sw_d = aria.aria_quantize_weights_int8(dev_f32(c["Wup"]))
    H = aria.aria_linear_w8a8(X, wq_d, sw_d, dev_bf16(bu_b), aria.ACT_GELU_ERF, aria.BF16)
    torch.cuda.synchronize()
    Hf = host_f32(H)
    hq_d, hs_d = aria.aria_quantize_act_int8(H)
    hq, hs = oracle.quant_int8_rows(Hf)
    assert np.array_equal(hq_d.cpu().numpy(), hq) and np.array_equal(hs_d.cpu().numpy(), hs)
    _linear_case(aria, oracle, H, Hf, c["Wdown"], dev_bf16(bd_b), bd.astype(np.float64), aria.ACT_NONE,
                 [aria.F32, aria.BF16])


def test_no_bias_and_ragged_shapes(aria, oracle):
    for (M, K, N) in [(77, 160, 72), (130, 1536, 200), (5, 32, 8)]:
        bits, x = inputs.normal_bf16((M, K), 1.0, 61, M + K + N)
        W = inputs.normal_f32((N, K), 0.02, 61, M + K + N + 1)
        _linear_case(aria, oracle, dev_bf16(bits), x, W, None, None, aria.ACT_NONE, [aria.F32, aria.BF16])


def test_zero_input_gives_bias(aria, oracle):
    M, K, N = 64, 256, 128
    X = torch.zeros((M, K), dtype=torch.bfloat16, device="cuda")
    W = inputs.normal_f32((N, K), 0.02, 62, 0)
    b = inputs.normal_f32((N,), 0.01, 62, 1)
    wq_d, sw_d = aria.aria_quantize_weights_int8(dev_f32(W))
    y = aria.aria_linear_w8a8(X, wq_d, sw_d, dev_f32(b), aria.ACT_NONE, aria.F32)
    assert np.array_equal(host_f32(y), np.broadcast_to(b, (M, N)))


def test_prequantised_entry_point_matches_fused_call(aria, oracle):
    c = inputs.c2(M=256)
    X = dev_bf16(c["X_bits"])
    wq_d, sw_d = aria.aria_quantize_weights_int8(dev_f32(c["Wout"]))
    b = dev_bf16(c["bout"][0])
    y1 = aria.aria_linear_w8a8(X, wq_d, sw_d, b, aria.ACT_NONE, aria.F32)
    xq, sx = aria.aria_quantize_act_int8(X)
    y2 = aria.aria_linear_w8a8_q(xq, sx, wq_d, sw_d, b, aria.ACT_NONE, aria.F32)
    assert torch.equal(y1, y2)


@pytest.mark.parametrize("io", ["bf16", "f32"])
def test_fused_absmax_chain_codes_and_scales_bit_exact(aria, oracle, io):
    """Fused S1: a -> b -> c chained (in == NULL twice).  Layers a and b reduce the per-token absmax of
    what they store in their own epilogues; the S1 passes of b and c take it from there.  Teacher-forced
    (SURVEY O5): the codes and scales the oracle derives from the GPU's own stored output must reproduce
    every next layer's output -- checked through aria_linear_w8a8_q fed with the ORACLE's codes, which
    must equal the chain's output bit for bit -- and the eager chain equals per-layer calls."""
    M, dims = 300, (416, 1536, 288, 136)
    dt = torch.bfloat16 if io == "bf16" else torch.float32
    code = aria.BF16 if io == "bf16" else aria.F32
    bits, x = inputs.normal_bf16((M, dims[0]), 1.0, 66, 0)
    X = dev_bf16(bits) if io == "bf16" else dev_f32(x)
    specs = []
    for i in range(3):
        W = inputs.normal_f32((dims[i + 1], dims[i]), 0.05, 66, 10 + i)
        wq, sw = aria.aria_quantize_weights_int8(dev_f32(W))
        bb, bf = inputs.normal_bf16((dims[i + 1],), 0.01, 66, 20 + i)
        specs.append({"K": dims[i], "N": dims[i + 1], "act": aria.ACT_GELU_ERF if i == 0 else aria.ACT_NONE,
                      "in": X if i == 0 else None, "wq": wq, "w_scale": sw,
                      "bias": dev_bf16(bb) if io == "bf16" else dev_f32(bf),
                      "out": torch.zeros((M, dims[i + 1]), dtype=dt, device="cuda")})
    layers = aria.make_layers(specs)
    ws = aria.workspace(aria.aria_workspace_bytes(M, max(dims), max(dims), aria.W8A8))
    for _ in range(2):                                   # twice: the absmax buffers are re-zeroed in-chain
        for s in specs:
            s["out"].zero_()
        aria.aria_denoiser_linears(layers, M, aria.W8A8, code, ws)
        torch.cuda.synchronize()
        prev = X
        for s in specs:
            xin = host_f32(prev)
            xq, sx = oracle.quant_int8_rows(xin)                     # the definition, on the GPU's own input
            y = aria.aria_linear_w8a8_q(dev_i8(xq), dev_f32(sx), s["wq"], s["w_scale"], s["bias"], s["act"], code)
            assert torch.equal(y, s["out"]), s["N"]
            y2 = aria.aria_linear_w8a8(prev, s["wq"], s["w_scale"], s["bias"], s["act"], code)
            assert torch.equal(y2, s["out"])
            prev = s["out"]
