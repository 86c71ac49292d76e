"""Pins for the oracle's quantisers O1 (int8 rows) and O2 (int4 groups).

None of these re-types the oracle's formula: they check it against hand-worked
numbers (tests/golden), a brute-force nearest-code
search in fp64, algebraic invariants, and library conversions (numpy float16,
ml_dtypes bfloat16).
"""
import json
import os

import ml_dtypes
import numpy as np
import pytest

from paper_2607_08526_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _gold(name):
    with open(os.path.join(GOLD, name)) as f:
        return json.load(f)


# ------------------------------------------------------------------ conversions
def test_fp16_conversion_matches_numpy_all_patterns(oracle):
    # every fp16 bit pattern widens to the value numpy gives (exact both ways)
    bits = np.arange(65536, dtype=np.uint16)
    ref = bits.view(np.float16).astype(np.float32)
    got = np.array([oracle.fp16_bits_to_f32(int(b)) for b in bits], dtype=np.float32)
    fin = np.isfinite(ref)
    assert np.array_equal(got[fin], ref[fin])
    assert np.array_equal(np.isnan(got), np.isnan(ref))
    # and rounds back to itself
    back = np.array([oracle.f32_to_fp16_bits(float(v)) for v in ref[fin]], dtype=np.uint16)
    assert np.array_equal(back, bits[fin])


def test_fp32_to_fp16_rne_matches_numpy(oracle):
    rng = np.random.default_rng(11)
    x = np.concatenate([
        rng.standard_normal(20000).astype(np.float32) * 0.01,
        rng.standard_normal(5000).astype(np.float32) * 1e-6,       # fp16 subnormal range
        rng.standard_normal(2000).astype(np.float32) * 3e4,        # near overflow
        # exact ties between adjacent fp16 values, normal and subnormal
        (np.arange(1, 2000, dtype=np.float32) + 0.5) * np.float32(2.0 ** -24),
        (np.float32(1.0) + (np.arange(0, 2000, dtype=np.float32) + 0.5) * np.float32(2.0 ** -10)),
        np.array([0.0, -0.0, 65504.0, 65519.9, 65520.0, 1e9, -1e9, 2.0 ** -25, 2.0 ** -24 * 1.5],
                 dtype=np.float32)])
    with np.errstate(over="ignore"):
        ref = x.astype(np.float16).view(np.uint16)
    got = np.array([oracle.f32_to_fp16_bits(float(v)) for v in x], dtype=np.uint16)
    assert np.array_equal(got, ref)


def test_f64_to_bf16_matches_ml_dtypes_on_fp32_inputs(oracle):
    # On values that are exactly fp32, one rounding from double == fp32->bf16 RNE
    rng = np.random.default_rng(12)
    x = np.concatenate([rng.standard_normal(20000).astype(np.float32) * 50,
                        rng.standard_normal(2000).astype(np.float32) * 1e-39,
                        np.array([0.0, -0.0, 1.0, 1.00390625, 1.01171875, 3.3895314e38, 3.4e38],
                                 dtype=np.float32)])
    ref = x.astype(ml_dtypes.bfloat16).view(np.uint16)
    got = np.array([oracle.f64_to_bf16_bits(float(v)) for v in x], dtype=np.uint16)
    assert np.array_equal(got, ref)


def test_f64_to_bf16_single_rounding(oracle):
    # 1 + 2^-8 + 2^-30: above the tie -> rounds up with one rounding; a detour
    # through fp32 would first land ON the tie (1+2^-8) and then round to even (down).
    x = 1.0 + 2.0 ** -8 + 2.0 ** -30
    assert oracle.f64_to_bf16_bits(x) == 0x3F81
    assert oracle.f64_to_bf16_bits(1.0 + 2.0 ** -8) == 0x3F80          # exact tie -> even
    assert oracle.f64_to_bf16_bits(1.0 + 3 * 2.0 ** -8) == 0x3F82      # tie -> even (up)


# ------------------------------------------------------------------ O1
def test_o1_hand_example_h1(oracle):
    g = _gold("h1_w8a8.json")
    X = np.array(g["X"], np.float32)
    W = np.array(g["W"], np.float32)
    xq, sx = oracle.quant_int8_rows(X)
    wq, sw = oracle.quant_int8_rows(W)
    assert np.array_equal(xq, np.array(g["Xq"], np.int8))
    assert np.array_equal(sx, np.array(g["sx"], np.float32))
    assert np.array_equal(wq, np.array(g["Wq"], np.int8))
    assert np.array_equal(sw[:3], np.array(g["sw_exact"], np.float32))
    assert sw[3:].view(np.uint32)[0] == int(g["sw3_bits"], 16)


def test_o1_brute_force_all_bf16_patterns(oracle):
    # One fixed absmax (3.0): every finite bf16 value |x| <= 3 is a row element.
    # q must be the nearest code to x/s (s = fl32(3/127)); exact ties in real
    # arithmetic go to the even code.  The search is done in exact rational-free
    # fp64 (x and s are fp32, so x - c*s is exact in fp64 up to 1 ulp of fp64).
    bits = np.arange(65536, dtype=np.uint16)
    vals = inputs.bf16_as_f32(bits)
    keep = np.isfinite(vals) & (np.abs(vals) <= 3.0)
    vals = vals[keep]
    row = np.concatenate([[np.float32(3.0)], vals]).astype(np.float32)[None, :]
    q, s = oracle.quant_int8_rows(row)
    s64 = float(s[0])
    assert s[0] == np.float32(3.0) / np.float32(127.0)
    codes = np.arange(-127, 128, dtype=np.float64)
    x64 = row[0].astype(np.float64)
    err = np.abs(x64[:, None] - codes[None, :] * s64)          # [n, 255]
    best = err.min(axis=1)
    qi = q[0].astype(np.int64)
    got_err = np.abs(x64 - qi * s64)
    # the chosen code is a nearest code up to the fp32 rounding of x/s
    # (|x/s| <= 127 -> abs rounding error <= 2^-18; see DESIGN.md tolerance note)
    assert np.all(got_err <= best + s64 * 2.0 ** -17)
    # where the nearest code is unambiguous by a margin, it must be exactly it
    order = np.sort(err, axis=1)
    clear = (order[:, 1] - order[:, 0]) > s64 * 2.0 ** -16
    assert clear.mean() > 0.99
    assert np.array_equal(qi[clear], codes[np.argmin(err, axis=1)][clear].astype(np.int64))
    assert q[0, 0] == 127


def test_o1_ties_go_to_even(oracle):
    # scale exactly 1 (absmax 127): x = k + 0.5 must round to the even neighbour
    ks = np.arange(-126, 126)
    row = np.concatenate([[127.0], ks + 0.5]).astype(np.float32)[None, :]
    q, s = oracle.quant_int8_rows(row)
    assert s[0] == 1.0
    lo = np.floor(ks + 0.5).astype(np.int64)
    expect = np.where(lo % 2 == 0, lo, lo + 1)
    assert np.array_equal(q[0, 1:].astype(np.int64), expect)


@pytest.mark.parametrize("bf16", [False, True])
@pytest.mark.parametrize("outliers", [False, True])
def test_o1_invariants(oracle, bf16, outliers):
    rng = np.random.default_rng(5)
    A = rng.standard_normal((64, 1536)).astype(np.float32)
    if outliers:
        A[:, rng.choice(1536, 15, replace=False)] *= 20
    if bf16:
        A = inputs.bf16_as_f32(inputs.bf16_bits(A))
    A[7] = 0.0                                            # all-zero row (reading R3)
    q, s = oracle.quant_int8_rows(A)
    qi = q.astype(np.int64)
    assert np.abs(qi).max() <= 127
    # absmax element maps to +-127; zero row -> scale 1, codes 0
    am = np.abs(A).argmax(axis=1)
    r = np.arange(A.shape[0])
    nz = np.abs(A).max(axis=1) > 0
    assert np.all(np.abs(qi[r, am])[nz] == 127)
    assert s[7] == 1.0 and not qi[7].any()
    # dequantisation error <= s/2 (1 + 2^-10), evaluated in fp64
    err = np.abs(A.astype(np.float64) - qi * s.astype(np.float64)[:, None])
    assert np.all(err <= 0.5 * s.astype(np.float64)[:, None] * (1 + 2.0 ** -10))
    # sign symmetry
    q2, s2 = oracle.quant_int8_rows(-A)
    assert np.array_equal(q2, -q) and np.array_equal(s2, s)
    # power-of-two scale equivariance
    q3, s3 = oracle.quant_int8_rows(A * np.float32(8.0))
    assert np.array_equal(q3, q) and np.array_equal(s3[nz], (s * np.float32(8.0))[nz])
    # idempotence on the dequantised grid
    D = (qi * s.astype(np.float64)[:, None]).astype(np.float32)
    q4, _ = oracle.quant_int8_rows(D)
    assert np.array_equal(q4, q)


# ------------------------------------------------------------------ O2
def _group(first4):
    w = np.zeros((1, 32), np.float32)
    w[0, :4] = first4
    return w


def test_o2_hand_example_h2(oracle):
    g = _gold("h2_int4.json")
    for case in g["cases"]:
        codes, sg, packed = oracle.quant_int4_groups(_group(case["w4"]))
        assert int(sg[0, 0]) == int(case["sg_bits"], 16)
        assert oracle.fp16_bits_to_f32(int(sg[0, 0])) == case["sg"]
        assert codes[0, :4].tolist() == case["codes4"]
        assert not codes[0, 4:].any()
        assert [int(b) for b in packed[0, :2]] == [int(b, 16) for b in case["bytes2"]]
        assert not packed[0, 2:].any()
        if "what_bf16" in case:
            what = oracle.dequant_int4(codes, sg, variant=0)
            assert what[0, :4].tolist() == case["what_bf16"]


def test_o2_pack_roundtrip_all_pairs(oracle):
    # all 15 x 15 code pairs through pack -> unpack; byte value from the format definition
    pairs = [(a, b) for a in range(-7, 8) for b in range(-7, 8)]
    K = 2 * len(pairs)
    K_pad = (K + 31) // 32 * 32
    codes = np.zeros((1, K_pad), np.int8)
    codes[0, :K] = np.array(pairs, np.int8).reshape(-1)
    # build weights that quantise exactly to these codes: w = code * 1.0 with a 7 in each group
    W = codes.astype(np.float32).copy()
    for g0 in range(0, K_pad, 32):
        if np.abs(W[0, g0:g0 + 32]).max() < 7:
            W[0, g0 + 31] = 7.0
    c2, sg, packed = oracle.quant_int4_groups(W)
    assert np.all(sg == 0x3C00)                       # every group scale is exactly 1.0
    assert np.array_equal(c2[0, :K], codes[0, :K])
    for j, (a, b) in enumerate(pairs):
        assert int(packed[0, j]) == ((a & 0xF) | ((b & 0xF) << 4))
    assert np.array_equal(oracle.unpack_int4(packed, K_pad), c2)
    assert not np.any((packed & 0xF) == 8) and not np.any((packed >> 4) == 8)   # -8 never produced


def test_o2_invariants_and_nearest_code(oracle):
    W = inputs.normal_f32((64, 1536), 0.02, 99, 0)
    W[3, 64:96] = 0.0                                  # all-zero group (reading R3)
    W[5, 0:32] *= np.float32(1e-5)                     # fp16-subnormal scale group
    codes, sg_bits, packed = oracle.quant_int4_groups(W)
    ci = codes.astype(np.int64)
    assert np.abs(ci).max() <= 7
    sg = sg_bits.view(np.float16).astype(np.float64)   # numpy's fp16 decoding, not the oracle's
    a = np.abs(W.reshape(64, -1, 32)).max(axis=2)
    # the scale is fp16_rne(fl32(a/7)) -- numpy conversion as the independent reference
    assert np.array_equal((a / np.float32(7.0)).astype(np.float16).view(np.uint16), sg_bits)
    assert sg_bits[3, 2] == 0 and not ci[3, 64:96].any()
    # absmax element -> +-7 for groups whose scale is in the fp16 normal range
    Wg = W.reshape(64, -1, 32).astype(np.float64)
    cg = ci.reshape(64, -1, 32)
    normal = (a / 7.0) >= 2.0 ** -14
    am = np.abs(Wg).argmax(axis=2)
    top = np.take_along_axis(np.abs(cg), am[..., None], axis=2)[..., 0]
    assert np.all(top[normal] == 7)
    # nearest code w.r.t. the fp16 scale: error <= sg/2 (1+2^-10) unless clamped at +-7
    err = np.abs(Wg - cg * sg[..., None])
    unclamped = np.abs(Wg) <= 7 * sg[..., None]
    bound = 0.5 * sg[..., None] * (1 + 2.0 ** -10)
    assert np.all((err <= bound) | ~unclamped)
    # clamped elements (fp16 rounding made 7*sg < |w|) stay within one fp16 ulp of the scale
    assert np.all(err[~unclamped] <= 7 * sg[..., None].repeat(32, 2)[~unclamped] * 2.0 ** -10)
    # sign symmetry and power-of-two equivariance
    c2, s2, _ = oracle.quant_int4_groups(-W)
    assert np.array_equal(c2, -codes) and np.array_equal(s2, sg_bits)
    c3, s3, _ = oracle.quant_int4_groups(W * np.float32(4.0))
    big = normal & (a * 4 / 7.0 < 6e4)
    assert np.array_equal(c3.reshape(64, -1, 32)[big], codes.reshape(64, -1, 32)[big])
    assert np.array_equal(s3.view(np.float16)[big].astype(np.float32),
                          sg_bits.view(np.float16)[big].astype(np.float32) * 4)
