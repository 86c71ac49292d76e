"""Pins for the oracle's NEXT rows: O6, the q8 weight-only linear (W8A16), and O7,
in-graph activation steering (eq. 2 and the projection variant).  Hand-worked H3 / H4,
integer special cases, numpy fp64 matmul with an independent bf16 rounding (ml_dtypes), and the
invariants the paper states (strength 0 is the identity, bit for bit; beta = -1 removes the component)."""
import json
import os
import struct

import ml_dtypes
import numpy as np

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _gold(name):
    with open(os.path.join(GOLD, name)) as f:
        return json.load(f)


def _f32(bits_hex):
    return struct.unpack("f", struct.pack("I", int(bits_hex, 16)))[0]


# ------------------------------------------------------------------ O6: W8A16
def test_o6_hand_example_h3(oracle):
    g = _gold("h3_w8a16.json")
    x = np.array([g["x"]], np.float32)
    Wq = np.array(g["Wq"], np.int8)
    sw = np.array([_f32(b) for b in g["sw_bits"]], np.float32)
    b = np.array(g["b"], np.float64)
    y0 = oracle.linear_w8a16(x, Wq, sw, b, variant=0)
    y1 = oracle.linear_w8a16(x, Wq, sw, b, variant=1)
    assert np.array_equal(y0[0], np.array(g["y_bf16w"]))
    assert y1[0, 0] == g["y_exactw_row0"] and abs(y1[0, 1] - g["y_exactw_row1"]) < 1e-15
    # the dequantised weights themselves: a one-hot x picks them out (bias off)
    what = oracle.linear_w8a16(np.eye(4, dtype=np.float32), Wq, sw, None, variant=0).T
    assert np.array_equal(what, np.array(g["what_bf16"]))


def test_o6_integer_special_case(oracle):
    # sw a power of two, codes and x small integers: every product and sum is an exact integer multiple
    rng = np.random.default_rng(11)
    Wq = rng.integers(-127, 128, size=(24, 64), dtype=np.int8)
    sw = np.full((24,), 0.25, np.float32)
    x = rng.integers(-4, 5, size=(9, 64)).astype(np.float32)
    ref = 0.25 * (x.astype(np.int64) @ Wq.astype(np.int64).T)
    for v in (0, 1):     # |q| * 0.25 has <= 7 significant bits: bf16 rounding is the identity
        assert np.array_equal(oracle.linear_w8a16(x, Wq, sw, None, variant=v), ref)


def test_o6_reduces_to_numpy_matmul_with_an_independent_bf16_rounding(oracle):
    rng = np.random.default_rng(12)
    N, K, M = 40, 96, 13
    Wq = rng.integers(-127, 128, size=(N, K), dtype=np.int8)
    sw = (np.abs(rng.standard_normal(N)) * 0.01 + 1e-4).astype(np.float32)
    x = rng.standard_normal((M, K)).astype(ml_dtypes.bfloat16).astype(np.float32)
    b = rng.standard_normal(N) * 0.01
    prod = Wq.astype(np.float64) * sw.astype(np.float64)[:, None]        # exact in fp64
    # variant 1: plain fp64 matmul
    assert np.allclose(oracle.linear_w8a16(x, Wq, sw, b, variant=1), x.astype(np.float64) @ prod.T + b, rtol=1e-12, atol=1e-13)
    # variant 0: bf16 rounding by ml_dtypes.  Its fp64 -> bf16 cast goes through fp32 (a DOUBLE rounding), which
    # differs from the single rounding of the definition only when the fp32 rounding lands on a bf16 tie: none of
    # these 3840 products does (checked: every fp32-rounded product is off a tie), so the two agree exactly.
    p32 = prod.astype(np.float32)
    assert not np.any((p32.view(np.uint32) & 0xFFFF) == 0x8000)
    what = p32.astype(ml_dtypes.bfloat16).astype(np.float64)
    got = oracle.linear_w8a16(x, Wq, sw, b, variant=0)
    assert np.allclose(got, x.astype(np.float64) @ what.T + b, rtol=1e-12, atol=1e-13)
    # GELU composes as in O3
    gg = oracle.linear_w8a16(x, Wq, sw, b, act=1, variant=0)
    assert np.allclose(gg, [[oracle.gelu_erf(v) for v in row] for row in got], rtol=1e-14, atol=0)


def test_o6_single_rounding_of_the_product(oracle):
    """The definition rounds the EXACT product q * sw once.  Construct (q, sw) whose fp32-rounded product sits
    exactly on the bf16 tie T = 1 + 2^-8 (between 1.0, even, and 1 + 2^-7) while the exact product is just
    ABOVE it: rounding twice (fp32, then bf16, ties to even) would give 1.0, the definition gives 1 + 2^-7."""
    from fractions import Fraction
    T = Fraction(1) + Fraction(1, 256)
    found = None
    for q in range(3, 128, 2):
        sw = np.float32(float(T) / q)
        exact = Fraction(float(sw)) * q
        if exact > T and np.float32(float(exact)) == np.float32(float(T)) and exact - T < Fraction(1, 2 ** 24):
            found = (q, sw)
            break
    assert found is not None
    q, sw = found
    assert float(np.float32(q) * sw) == float(T)                       # what a fp32 multiply returns: the tie
    y = oracle.linear_w8a16(np.array([[1.0]], np.float32), np.array([[q]], np.int8), np.array([sw], np.float32),
                            None, variant=0)
    assert y[0, 0] == 1.0 + 2.0 ** -7
    y1 = oracle.linear_w8a16(np.array([[1.0]], np.float32), np.array([[q]], np.int8), np.array([sw], np.float32),
                             None, variant=1)
    assert Fraction(float(y1[0, 0])) == Fraction(float(sw)) * q        # variant 1: the exact product (fits fp64)


# ------------------------------------------------------------------ O7: steering
def test_o7_hand_example_h4(oracle):
    g = _gold("h4_steer.json")
    h = np.array(g["h"], np.float32)
    d = np.array(g["d"], np.float32)
    assert np.array_equal(oracle.steer(h, d, 0.5, g["hbar_norm"], oracle.STEER_ADD), np.array(g["add_alpha_0p5"]))
    assert np.array_equal(oracle.steer(h, d, -1.0, 1.0, oracle.STEER_PROJECT), np.array(g["project_beta_m1"]))
    assert np.array_equal(oracle.steer(h, d, 2.0, 1.0, oracle.STEER_PROJECT), np.array(g["project_beta_2"]))


def test_o7_strength_zero_is_the_identity_bit_for_bit(oracle):
    # "at strength 0 the output is bit-identical to the base model" -- including -0.0 and subnormals
    h = np.array([[-0.0, 0.0, 1e-40, -3.5], [np.float32(2.0 ** -126), -1.0, 7.25, -0.0]], np.float32)
    d = np.array([0.5, -0.5, 0.5, 0.5], np.float32)
    for op in (oracle.STEER_ADD, oracle.STEER_PROJECT):
        out = oracle.steer(h, d, 0.0, 3.0, op)
        assert np.array_equal(out.view(np.uint64), h.astype(np.float64).view(np.uint64))


def test_o7_invariants(oracle):
    rng = np.random.default_rng(13)
    M, D = 7, 64
    h = rng.standard_normal((M, D)).astype(np.float32)
    d = rng.standard_normal(D)
    d = (d / np.linalg.norm(d)).astype(np.float32)
    d64 = d.astype(np.float64)
    # additive: the same rank-one offset alpha * n * d on every token (eq. 2: "adds one rank-one term")
    out = oracle.steer(h, d, 0.3, 11.0, oracle.STEER_ADD)
    off = out - h.astype(np.float64)
    assert np.allclose(off, np.broadcast_to(0.3 * 11.0 * d64, (M, D)), rtol=0, atol=1e-15)
    # linear in alpha
    out2 = oracle.steer(h, d, 0.6, 11.0, oracle.STEER_ADD)
    assert np.allclose(out2 - h, 2 * off, rtol=0, atol=1e-15)
    # projection, beta = -1: the component along d is removed (|d| = 1 up to fp32 rounding of d)
    out = oracle.steer(h, d, -1.0, 1.0, oracle.STEER_PROJECT)
    assert np.max(np.abs(out @ d64)) <= 1e-6 * np.max(np.abs(h.astype(np.float64) @ d64))
    # projection leaves the orthogonal complement alone: out - h is parallel to d
    diff = out - h.astype(np.float64)
    assert np.allclose(diff, np.outer(diff @ d64 / (d64 @ d64), d64), rtol=0, atol=1e-14)
    # beta scales the component by (1 + beta)
    out = oracle.steer(h, d, 1.5, 1.0, oracle.STEER_PROJECT)
    assert np.allclose(out @ d64, (1 + 1.5 * (d64 @ d64)) * (h.astype(np.float64) @ d64), rtol=1e-12, atol=1e-14)
