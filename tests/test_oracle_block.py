"""Pins for the oracle's NEXT-2 row: O8, the normalisation whose output S1 quantises, and O9,
full multi-head self-attention between QKV and the out-projection.  Hand-worked H5 / H6,
closed forms and invariants that a dropped term, a wrong axis, a transposed operand or a missing scale would
break, and torch's fp64 layer_norm / scaled_dot_product_attention as the library routine."""
import json
import math
import os

import numpy as np
import torch

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _gold(name):
    with open(os.path.join(GOLD, name)) as f:
        return json.load(f)


# ------------------------------------------------------------------ O8: norm (-> S1)
def test_o8_hand_example_h5(oracle):
    g = _gold("h5_norm.json")
    x = np.array([g["x_ln"]], np.float32)
    one = np.ones(4, np.float32)
    assert np.allclose(oracle.norm_rows(x, one, None, oracle.NORM_LAYER, g["eps_ln"])[0], g["ln_unit"], rtol=0, atol=1e-15)
    gam = np.array(g["gamma"], np.float32)
    n = oracle.norm_rows(x, gam, None, oracle.NORM_LAYER, g["eps_ln"])
    assert np.allclose(n[0], g["ln_gamma"], rtol=0, atol=1e-13)
    nb = oracle.norm_rows(x, gam, np.array(g["beta"], np.float32), oracle.NORM_LAYER, g["eps_ln"])
    assert np.allclose(nb[0], g["ln_gamma_beta"], rtol=0, atol=1e-13)
    nn, q, s = oracle.norm_quant_int8(x, gam, None, oracle.NORM_LAYER, g["eps_ln"], dtype=oracle.OUT_BF16)
    assert np.array_equal(nn[0], np.array(g["ln_gamma"], np.float32))
    assert q[0].tolist() == g["codes"] and float(s[0]) == g["scale"]
    r = oracle.norm_rows(np.array([g["x_rms"]], np.float32), one, None, oracle.NORM_RMS, 0.0)
    assert np.allclose(r[0], g["rms_unit"], rtol=0, atol=1e-15)


def test_o8_layernorm_output_has_zero_mean_unit_variance_and_is_shift_scale_invariant(oracle):
    rng = np.random.default_rng(21)
    x = (rng.standard_normal((7, 96)) * 3 + 1.5).astype(np.float32)
    one = np.ones(96, np.float32)
    n = oracle.norm_rows(x, one, None, oracle.NORM_LAYER, 0.0)
    assert np.abs(n.mean(axis=1)).max() < 1e-14 and np.abs(n.var(axis=1) - 1.0).max() < 1e-13
    # exactly representable shift / scale (powers of two keep the fp32 inputs exact)
    assert np.allclose(oracle.norm_rows(x * 4.0, one, None, oracle.NORM_LAYER, 0.0), n, rtol=0, atol=1e-13)
    x2 = rng.integers(-8, 9, size=(5, 64)).astype(np.float32)
    a = oracle.norm_rows(x2, np.ones(64, np.float32), None, oracle.NORM_LAYER, 0.0)
    b = oracle.norm_rows(x2 + 32.0, np.ones(64, np.float32), None, oracle.NORM_LAYER, 0.0)
    assert np.allclose(a, b, rtol=0, atol=1e-13)
    # RMSNorm is NOT shift invariant but has unit mean square; sign flip flips the output
    r = oracle.norm_rows(x, one, None, oracle.NORM_RMS, 0.0)
    assert np.abs((r ** 2).mean(axis=1) - 1.0).max() < 1e-13
    assert np.array_equal(oracle.norm_rows(-x, one, None, oracle.NORM_RMS, 0.0), -r)
    assert not np.allclose(oracle.norm_rows(x + 32.0, one, None, oracle.NORM_RMS, 0.0), r, atol=1e-3)


def test_o8_matches_torch_fp64_layer_norm_and_eps_gamma_beta_placement(oracle):
    rng = np.random.default_rng(22)
    x = rng.standard_normal((11, 160)).astype(np.float32)
    gam = (1.0 + 0.1 * rng.standard_normal(160)).astype(np.float32)
    bet = (0.05 * rng.standard_normal(160)).astype(np.float32)
    for eps in (1e-5, 1e-2):
        ref = torch.nn.functional.layer_norm(torch.from_numpy(x).double(), (160,), torch.from_numpy(gam).double(),
                                             torch.from_numpy(bet).double(), eps).numpy()
        assert np.allclose(oracle.norm_rows(x, gam, bet, oracle.NORM_LAYER, eps), ref, rtol=1e-13, atol=1e-14)
        xd = x.astype(np.float64)
        rref = xd / np.sqrt((xd ** 2).mean(axis=1, keepdims=True) + eps) * gam.astype(np.float64) + bet.astype(np.float64)
        assert np.allclose(oracle.norm_rows(x, gam, bet, oracle.NORM_RMS, eps), rref, rtol=1e-13, atol=1e-14)


def test_o8_norm_then_o1_keeps_the_s1_invariants(oracle):
    rng = np.random.default_rng(23)
    x = rng.standard_normal((9, 128)).astype(np.float32)
    gam = np.ones(128, np.float32)
    n, q, s = oracle.norm_quant_int8(x, gam, None, oracle.NORM_LAYER, 1e-5, dtype=oracle.OUT_BF16)
    q2, s2 = oracle.quant_int8_rows(n)
    assert np.array_equal(q, q2) and np.array_equal(s, s2)          # it IS O1 of the rounded tensor
    assert np.abs(q).max() == 127 and np.all(np.abs(n - q * s[:, None]) <= s[:, None] / 2 * (1 + 2.0 ** -10))
    # bf16 rounding really happened before S1: n holds bf16 values only
    assert np.array_equal((n.view(np.uint32) & 0xFFFF), np.zeros_like(n, dtype=np.uint32))


# ------------------------------------------------------------------ O9: attention
def _qkv(rng, B, S, H, Dh, std=1.0):
    return (rng.standard_normal((B * S, 3 * H * Dh)) * std).astype(np.float32)


def test_o9_hand_example_h6(oracle):
    g = _gold("h6_attention.json")
    o = oracle.attention(np.array(g["qkv"], np.float32), 1, g["S"], g["H"], g["Dh"], g["scale"])
    assert np.allclose(o, np.array(g["o"]), rtol=0, atol=g["tol"])


def test_o9_equal_keys_give_the_mean_of_v_and_a_dominant_key_selects_its_v(oracle):
    rng = np.random.default_rng(31)
    B, S, H, Dh = 2, 9, 3, 4
    x = _qkv(rng, B, S, H, Dh)
    x3 = x.reshape(B, S, 3, H, Dh)
    x3[:, :, 1] = x3[:, :1, 1]                       # every key of a (sequence, head) equal
    o = oracle.attention(x, B, S, H, Dh).reshape(B, S, H, Dh)
    vmean = x3[:, :, 2].astype(np.float64).mean(axis=1, keepdims=True)
    assert np.allclose(o, np.broadcast_to(vmean, o.shape), rtol=1e-13, atol=1e-14)
    # one key aligned with every query and scaled up: softmax -> one-hot on that key, per sequence and head
    y = _qkv(rng, B, S, H, Dh)
    y3 = y.reshape(B, S, 3, H, Dh)
    y3[:, :, 0] = 1.0
    y3[:, :, 1] = 0.0
    y3[:, 5, 1] = 64.0                               # key 5: score 64*Dh*scale, others 0
    o = oracle.attention(y, B, S, H, Dh).reshape(B, S, H, Dh)
    assert np.allclose(o, np.broadcast_to(y3[:, 5:6, 2].astype(np.float64), o.shape), rtol=1e-12, atol=1e-12)


def test_o9_invariances_key_permutation_key_shift_and_head_sequence_independence(oracle):
    rng = np.random.default_rng(32)
    B, S, H, Dh = 2, 12, 2, 8
    x = _qkv(rng, B, S, H, Dh)
    o = oracle.attention(x, B, S, H, Dh)
    x3 = x.reshape(B, S, 3, H, Dh)
    # permuting the (k, v) pairs of a sequence leaves every query's output unchanged
    perm = rng.permutation(S)
    y3 = x3.copy()
    y3[:, :, 1:] = x3[:, perm, 1:]
    assert np.allclose(oracle.attention(y3.reshape(B * S, -1), B, S, H, Dh), o, rtol=1e-12, atol=1e-13)
    # adding one vector c to every key adds q.c to every score of a query: softmax is unchanged
    z3 = x3.copy()
    z3[:, :, 1] += np.float32(0.5)                   # exactly representable shift
    assert np.allclose(oracle.attention(z3.reshape(B * S, -1), B, S, H, Dh), o, rtol=1e-6, atol=1e-7)
    # changing sequence 1 / head 1 does not touch sequence 0 / head 0
    w3 = x3.copy()
    w3[1] = rng.standard_normal(w3[1].shape).astype(np.float32)
    w3[:, :, :, 1] = rng.standard_normal(w3[:, :, :, 1].shape).astype(np.float32)
    o2 = oracle.attention(w3.reshape(B * S, -1), B, S, H, Dh).reshape(B, S, H, Dh)
    assert np.array_equal(o2[0, :, 0], o.reshape(B, S, H, Dh)[0, :, 0])
    # the scale matters (a dropped 1/sqrt(Dh) changes the result) and defaults to 1/sqrt(Dh)
    assert np.array_equal(oracle.attention(x, B, S, H, Dh, 1.0 / math.sqrt(Dh)), o)
    assert not np.allclose(oracle.attention(x, B, S, H, Dh, 1.0), o, atol=1e-3)


def test_o9_matches_torch_fp64_scaled_dot_product_attention(oracle):
    rng = np.random.default_rng(33)
    B, S, H, Dh = 2, 37, 3, 16
    x = _qkv(rng, B, S, H, Dh)
    t = torch.from_numpy(x).double().reshape(B, S, 3, H, Dh).permute(2, 0, 3, 1, 4)    # [3, B, H, S, Dh]
    ref = torch.nn.functional.scaled_dot_product_attention(t[0], t[1], t[2])           # default scale 1/sqrt(Dh)
    ref = ref.permute(0, 2, 1, 3).reshape(B * S, H * Dh).numpy()
    assert np.allclose(oracle.attention(x, B, S, H, Dh), ref, rtol=1e-12, atol=1e-13)
    # brute force on one output element, straight from the definition
    b, i, h, d = 1, 20, 2, 5
    x3 = x.astype(np.float64).reshape(B, S, 3, H, Dh)
    s = (x3[b, :, 1, h] @ x3[b, i, 0, h]) / math.sqrt(Dh)
    p = np.exp(s - s.max())
    p /= p.sum()
    assert abs(oracle.attention(x, B, S, H, Dh)[b * S + i, h * Dh + d] - p @ x3[b, :, 2, h, d]) < 1e-14
