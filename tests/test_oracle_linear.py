"""Pins for the oracle's linears: O3 (int8 GEMM + rescale/bias/GELU epilogue) and
O4 (W4A16), plus the output cast.  Hand-worked H1/H2, closed forms, numpy
int64 / fp64 matmul as the library routine, math.erf, textbook X W^T + b on
grids with no quantisation error."""
import json
import math
import os

import kernel_models
import ml_dtypes
import numpy as np

from paper_2607_08526_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _gold(name):
    with open(os.path.join(GOLD, name)) as f:
        return json.load(f)


# ------------------------------------------------------------------ O3: GEMM
def test_o3_hand_example_h1(oracle):
    g = _gold("h1_w8a8.json")
    X = np.array(g["X"], np.float32)
    W = np.array(g["W"], np.float32)
    b = np.array(g["b"], np.float64)
    wq, sw = oracle.quant_int8_rows(W)
    r = oracle.linear_w8a8(X, wq, sw, b)
    assert np.array_equal(r["acc"], np.array(g["acc"], np.int64))
    assert np.array_equal(r["y"][:, :3], np.array(g["y_cols012"], np.float64))
    assert np.allclose(r["y"][:, 3], np.array(g["y_col3_approx"]), rtol=2e-9, atol=0)
    assert np.array_equal(oracle.round_out(r["y"], oracle.OUT_F32)[:, 3],
                          np.array(g["y_col3_fp32"], np.float32))


def test_o3_closed_forms(oracle):
    K = 6144
    acc = oracle.gemm_i8(np.full((3, K), 127, np.int8), np.full((5, K), 127, np.int8))
    assert np.all(acc == K * 16129) and K * 16129 == 99096576
    acc = oracle.gemm_i8(np.full((2, K), -127, np.int8), np.full((2, K), 127, np.int8))
    assert np.all(acc == -99096576)
    rng = np.random.default_rng(3)
    Wq = rng.integers(-127, 128, size=(40, 96), dtype=np.int8)      # N=40, K=96
    # one-hot rows of X pick out columns of Wq (catches a transposed operand)
    Xq = np.zeros((96, 96), np.int8)
    Xq[np.arange(96), np.arange(96)] = 1
    assert np.array_equal(oracle.gemm_i8(Xq, Wq), Wq.T.astype(np.int64))
    # identity Wq returns Xq
    Xr = rng.integers(-127, 128, size=(17, 96), dtype=np.int8)
    assert np.array_equal(oracle.gemm_i8(Xr, np.eye(96, dtype=np.int8)), Xr.astype(np.int64))


def test_o3_gemm_matches_numpy_int64_matmul(oracle):
    rng = np.random.default_rng(4)
    Xq = rng.integers(-127, 128, size=(37, 200), dtype=np.int8)
    Wq = rng.integers(-127, 128, size=(53, 200), dtype=np.int8)
    ref = Xq.astype(np.int64) @ Wq.astype(np.int64).T
    assert np.array_equal(oracle.gemm_i8(Xq, Wq), ref)


# -------------------------------------------------------------- O3: epilogue
def test_o3_epilogue_special_cases(oracle):
    rng = np.random.default_rng(6)
    acc = rng.integers(-10 ** 8, 10 ** 8, size=(9, 13)).astype(np.int64)
    one_m, one_n = np.ones(9, np.float32), np.ones(13, np.float32)
    assert np.array_equal(oracle.epilogue_w8a8(acc, one_m, one_n), acc.astype(np.float64))
    sx = rng.random(9).astype(np.float32) + 0.5
    sw = rng.random(13).astype(np.float32) * 0.01
    b = rng.standard_normal(13)
    y = oracle.epilogue_w8a8(acc, sx, sw, b)
    ref = acc.astype(np.float64) * sx.astype(np.float64)[:, None] * sw.astype(np.float64)[None, :] + b
    assert np.allclose(y, ref, rtol=1e-15, atol=0)
    # row scale belongs to rows, column scale and bias to columns (non-square on purpose)
    y2 = oracle.epilogue_w8a8(acc, sx * 2, sw, b)
    assert np.allclose(y2 - b, 2 * (y - b), rtol=1e-14)
    yg = oracle.epilogue_w8a8(acc, sx, sw * np.float32(1e-6), b, act=oracle.ACT_GELU_ERF)
    v = acc.astype(np.float64) * sx.astype(np.float64)[:, None] * (sw * np.float32(1e-6)).astype(np.float64)[None, :] + b
    ref_g = np.array([[0.5 * t * (1 + math.erf(t / math.sqrt(2))) for t in row] for row in v])
    assert np.allclose(yg, ref_g, rtol=1e-14, atol=1e-300)


def test_gelu_pins(oracle):
    assert oracle.gelu_erf(0.0) == 0.0
    for x in [0.1, 0.5, 1.0, 2.5, 4.0, 7.0]:
        assert abs((oracle.gelu_erf(x) - oracle.gelu_erf(-x)) - x) <= 1e-15 * max(1, x)
        assert abs(oracle.gelu_erf(x) - 0.5 * x * (1 + math.erf(x / math.sqrt(2)))) <= 1e-15 * x
    for x in [6.0, 8.0, 20.0]:
        assert np.float32(oracle.gelu_erf(x)) == np.float32(x)
        assert abs(oracle.gelu_erf(-x)) < 1e-8
    # textbook value: gelu(1) = Phi(1) = 0.8413447460685429...
    assert abs(oracle.gelu_erf(1.0) - 0.8413447460685429) < 1e-15


def test_w8a8_equals_textbook_linear_on_exact_grid(oracle):
    # X rows and W rows already on their int8 grids with power-of-two scales =>
    # quantisation is lossless and the W8A8 result is the plain fp64 X W^T + b.
    rng = np.random.default_rng(8)
    M, K, N = 19, 160, 23
    xi = rng.integers(-127, 128, size=(M, K))
    wi = rng.integers(-127, 128, size=(N, K))
    xi[:, 0] = 127
    wi[:, 1] = -127
    sx = 2.0 ** rng.integers(-6, 3, size=M)
    sw = 2.0 ** rng.integers(-12, -4, size=N)
    X = (xi * sx[:, None]).astype(np.float32)
    W = (wi * sw[:, None]).astype(np.float32)
    b = rng.standard_normal(N)
    wq, sws = oracle.quant_int8_rows(W)
    assert np.array_equal(wq, wi.astype(np.int8)) and np.array_equal(sws, sw.astype(np.float32))
    r = oracle.linear_w8a8(X, wq, sws, b)
    assert np.array_equal(r["xq"], xi.astype(np.int8)) and np.array_equal(r["sx"], sx.astype(np.float32))
    ref = X.astype(np.float64) @ W.astype(np.float64).T + b
    assert np.allclose(r["y"], ref, rtol=1e-13, atol=1e-13)


def test_w8a8_quantisation_noise_level(oracle):
    # sanity, not a definition: on C2-like data the W8A8 output is ~39 dB SQNR
    # from the unquantised product -- catches gross scale mistakes
    X = inputs.bf16_as_f32(inputs.bf16_bits(inputs.normal_f32((64, 1536), 1.0, 77, 0)))
    W = inputs.normal_f32((256, 1536), 0.02, 77, 1)
    wq, sw = oracle.quant_int8_rows(W)
    y = oracle.linear_w8a8(X, wq, sw)["y"]
    ref = X.astype(np.float64) @ W.astype(np.float64).T
    sqnr = 10 * np.log10((ref ** 2).sum() / ((y - ref) ** 2).sum())
    assert 35 < sqnr < 45


# ------------------------------------------------------------------ O4
def test_o4_hand_example_h2(oracle):
    g = _gold("h2_int4.json")
    x = np.zeros((1, 32), np.float32)
    x[0, :4] = g["x4"]
    for case in g["cases"]:
        w = np.zeros((1, 32), np.float32)
        w[0, :4] = case["w4"]
        codes, sg, _ = oracle.quant_int4_groups(w)
        assert oracle.linear_w4a16(x, codes, sg, variant=0)[0, 0] == case["y_bf16w"]
        assert oracle.linear_w4a16(x, codes, sg, variant=1)[0, 0] == case["y_exactw"]


def test_o4_integer_special_case(oracle):
    # sg = 1, codes in [-7,7], x small integers => exact integer result
    rng = np.random.default_rng(9)
    M, K, N = 11, 96, 14
    codes = rng.integers(-7, 8, size=(N, K)).astype(np.int8)
    sg = np.full((N, K // 32), 0x3C00, np.uint16)
    x = rng.integers(-8, 9, size=(M, K)).astype(np.float32)
    b = rng.integers(-5, 6, size=N).astype(np.float64)
    y = oracle.linear_w4a16(x, codes, sg, b)
    assert np.array_equal(y, x.astype(np.int64) @ codes.astype(np.int64).T + b)


def test_o4_reduces_to_numpy_matmul(oracle):
    X = inputs.bf16_as_f32(inputs.bf16_bits(inputs.normal_f32((21, 256), 1.0, 78, 0)))
    W = inputs.normal_f32((40, 256), 0.02, 78, 1)
    b = inputs.normal_f32((40,), 0.01, 78, 2).astype(np.float64)
    codes, sg, packed = oracle.quant_int4_groups(W)
    for variant in (0, 1):
        # independent dequantisation: numpy fp16 decode, exact product, ml_dtypes bf16 rounding (variant 0)
        s = np.repeat(sg.view(np.float16).astype(np.float32), 32, axis=1)
        prod = codes.astype(np.float32) * s
        what = prod.astype(ml_dtypes.bfloat16).astype(np.float64) if variant == 0 else prod.astype(np.float64)
        assert np.array_equal(oracle.dequant_int4(codes, sg, variant), what)
        ref = X.astype(np.float64) @ what.T + b
        y = oracle.linear_w4a16(X, codes, sg, b, variant=variant)
        assert np.allclose(y, ref, rtol=1e-12, atol=1e-12)
    # the two variants differ by bf16 rounding of w^ only: relative 2^-9 per weight
    y0 = oracle.linear_w4a16(X, codes, sg, variant=0)
    y1 = oracle.linear_w4a16(X, codes, sg, variant=1)
    assert 0 < np.abs(y0 - y1).max() < 2e-2 * np.abs(y1).max()
    # the operand-format models of the stream kernel (tests/kernel_models.py; diagnostics, not definitions):
    # fp16 rounding of w^ (11 significant bits) sits 8x closer to the exact product than bf16 rounding
    y2 = kernel_models.linear_w4a16(X, codes, sg, None, 0, kernel_models.FP16_OPERAND)
    assert 0 < np.abs(y2 - y1).max() < 0.25 * np.abs(y0 - y1).max()
    # offset-binary fp16 rounding acts on u*sg (up to 15*sg): at most ~2x the error of the fp16-operand model
    y3 = kernel_models.linear_w4a16(X, codes, sg, None, 0, kernel_models.OFFSET_BINARY)
    assert 0 < np.abs(y3 - y1).max() < 0.5 * np.abs(y0 - y1).max()
    # and the models rebuilt from the oracle's own (pinned) scalar fp16 conversions, element by element
    sf = [[oracle.fp16_bits_to_f32(int(v)) for v in row] for row in sg]
    for model, f in ((kernel_models.FP16_OPERAND, lambda q, s_: oracle.fp16_bits_to_f32(oracle.f32_to_fp16_bits(float(np.float32(q) * np.float32(s_))))),
                     (kernel_models.OFFSET_BINARY, lambda q, s_: oracle.fp16_bits_to_f32(oracle.f32_to_fp16_bits(float(np.float32(q + 8) * np.float32(s_)))) - 8.0 * s_)):
        w = kernel_models.dequant_int4(codes, sg, model)
        for n in range(0, codes.shape[0], 7):
            for k in range(0, codes.shape[1], 5):
                assert w[n, k] == f(int(codes[n, k]), sf[n][k // 32])


def test_offset_binary_model_hand_values():
    # H2(iii) group (tests/golden/h2_int4.json): sg = 0x297C = 0.0428466796875, codes [2,-5,7,-1].
    # u*sg = [10, 3, 15, 7]*sg = [0.428466796875, 0.1285400390625, 0.6427001953125, 0.2999267578125];
    # fp16 spacing is 2^-12 in [0.25,0.5), 2^-13 in [0.125,0.25), 2^-11 in [0.5,1):
    #   0.428466796875 = 1755*2^-12 exact; 0.1285400390625 = 1053*2^-13 exact;
    #   0.6427001953125 = 1316.25*2^-11 -> 1316*2^-11 = 0.642578125; 0.2999267578125 = 1228.5*2^-12 -> tie to even 1228*2^-12 = 0.2998046875
    sg = np.zeros((1, 1), np.uint16); sg[0, 0] = 0x297C
    codes = np.zeros((1, 32), np.int8); codes[0, :4] = [2, -5, 7, -1]
    w = kernel_models.dequant_int4(codes, sg, kernel_models.OFFSET_BINARY)[0]
    s = 0.0428466796875
    assert w[0] == 0.428466796875 - 8 * s and w[1] == 0.1285400390625 - 8 * s
    assert w[2] == 0.642578125 - 8 * s and w[3] == 0.2998046875 - 8 * s
    assert np.all(w[4:] == np.float64(np.float16(8 * s)) - 8 * s)     # code 0 -> fp16(8 sg) - 8 sg = 0 (8 sg is exact)
    assert np.all(w[4:] == 0.0)


def test_o4_quantisation_noise_level(oracle):
    # sanity: ~20 dB SQNR for int4-g32 on N(0,0.02) weights
    X = inputs.bf16_as_f32(inputs.bf16_bits(inputs.normal_f32((32, 1536), 1.0, 79, 0)))
    W = inputs.normal_f32((128, 1536), 0.02, 79, 1)
    codes, sg, _ = oracle.quant_int4_groups(W)
    y = oracle.linear_w4a16(X, codes, sg)
    ref = X.astype(np.float64) @ W.astype(np.float64).T
    sqnr = 10 * np.log10((ref ** 2).sum() / ((y - ref) ** 2).sum())
    assert 17 < sqnr < 24


# ------------------------------------------------------------------ output cast
def test_round_out(oracle):
    rng = np.random.default_rng(10)
    y = rng.standard_normal(5000) * 100
    assert np.array_equal(oracle.round_out(y, oracle.OUT_F32), y.astype(np.float32))
    y32 = y.astype(np.float32)
    ref = y32.astype(ml_dtypes.bfloat16).astype(np.float32)
    assert np.array_equal(oracle.round_out(y32.astype(np.float64), oracle.OUT_BF16), ref)
    assert oracle.round_out(np.array([1.0 + 2.0 ** -8 + 2.0 ** -30]), oracle.OUT_BF16)[0] == np.float32(1.0078125)
