"""GPU parity of the NEXT-2 row: the normalisation fused with S1 and the fused self-attention,
through the C ABI, against oracle O8 / O9.  Codes and scales are teacher-forced: the GPU's own
normalised tensor is what the oracle quantises, so bit-exactness is a statement about the quantiser; the
normalised tensor and the attention output are compared by tolerance (R20-R22)."""
import numpy as np
import pytest
import torch

from aria_testutil import check_bf16_out, dev_bf16, dev_f32, host_bits16, host_f32, rel_err
from paper_2607_08526_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def aria():
    from paper_2607_08526_b200 import binding
    binding.lib()
    return binding


def _norm_case(aria, oracle, M, K, dtype, kind, with_beta, eps=1e-5, tid=0, x=None):
    if x is None:
        bits, x = inputs.residual_stream(M, K, tid)
        if dtype == "f32":
            x = (x + inputs.normal_f32((M, K), 1e-3, 8, 900 + tid)).astype(np.float32)   # not bf16-representable
    elif dtype == "bf16":
        x = inputs.bf16_as_f32(inputs.bf16_bits(x))          # the oracle sees exactly the bf16 values the GPU gets
    g, b = inputs.norm_params(K, tid)
    X = dev_f32(x) if dtype == "f32" else dev_bf16(inputs.bf16_bits(x))
    G, Bt = dev_f32(g), dev_f32(b) if with_beta else None
    xq, sx, xn = aria.aria_norm_quantize_act_int8(X, G, Bt, kind, eps, want_xn=True)
    xq2, sx2 = aria.aria_norm_quantize_act_int8(X, G, Bt, kind, eps)                    # without the Xn store
    torch.cuda.synchronize()
    assert torch.equal(xq, xq2) and torch.equal(sx, sx2)
    ref = oracle.norm_rows(x, g, b if with_beta else None, kind, eps)
    xn_h = host_f32(xn)
    if dtype == "f32":
        assert rel_err(xn_h, ref) <= 1e-5
    else:
        ref_bits = inputs.bf16_bits(oracle.round_out(ref, oracle.OUT_BF16))
        check_bf16_out(host_bits16(xn), ref, ref_bits, 2e-6, 0.01)
    # teacher-forced S1: exactly O1 of the tensor the kernel normalised to
    q_o, s_o = oracle.quant_int8_rows(xn_h)
    assert np.array_equal(xq.cpu().numpy(), q_o) and np.array_equal(sx.cpu().numpy(), s_o)
    # and exactly what the stand-alone S1 kernel makes of it
    q_g, s_g = aria.aria_quantize_act_int8(xn)
    assert torch.equal(q_g, xq) and torch.equal(s_g, sx)
    # free-running: codes differ from the all-fp64 pipeline by at most one step, rarely
    _, q_f, s_f = oracle.norm_quant_int8(x, g, b if with_beta else None, kind, eps,
                                         dtype=oracle.OUT_F32 if dtype == "f32" else oracle.OUT_BF16)
    d = np.abs(xq.cpu().numpy().astype(np.int32) - q_f.astype(np.int32))
    assert d.max() <= 1 and (d != 0).mean() <= 0.01
    assert np.allclose(sx.cpu().numpy(), s_f, rtol=2.0 ** -7, atol=0)


@pytest.mark.parametrize("M,K", [(512, 1536), (200, 1024), (3, 32), (9, 96), (64, 6144), (5, 9984), (2048, 1536)])
@pytest.mark.parametrize("kind", [0, 1])
def test_norm_quant_bf16_shapes(aria, oracle, M, K, kind):
    _norm_case(aria, oracle, M, K, "bf16", kind, with_beta=(K % 64 == 0), tid=K % 7)


@pytest.mark.parametrize("M,K", [(100, 1536), (7, 64), (33, 4096), (3, 24576)])
@pytest.mark.parametrize("kind", [0, 1])
def test_norm_quant_fp32(aria, oracle, M, K, kind):
    _norm_case(aria, oracle, M, K, "f32", kind, with_beta=True, tid=3)


def test_norm_quant_degenerate_rows(aria, oracle):
    # a zero row and a constant row have zero variance: n = beta (LayerNorm); with beta = None the row is all
    # zero and S1's zero-row rule applies (scale 1, codes 0)
    K = 256
    x = inputs.residual_stream(6, K, 5, outliers=False)[1].copy()
    x[1] = 0.0
    x[3] = 2.5
    _norm_case(aria, oracle, 6, K, "bf16", 0, with_beta=True, x=x)
    g, _ = inputs.norm_params(K, 0)
    xq, sx, xn = aria.aria_norm_quantize_act_int8(dev_bf16(inputs.bf16_bits(x)), dev_f32(g), None, 0, 1e-5, want_xn=True)
    assert float(sx[1]) == 1.0 and float(sx[3]) == 1.0 and int(xq[1].abs().max()) == 0 and int(xq[3].abs().max()) == 0
    assert float(xn[1].float().abs().max()) == 0.0
    # large eps, tiny values: still the definition
    _norm_case(aria, oracle, 6, K, "bf16", 1, with_beta=False, eps=1e-2, x=(x * 1e-3).astype(np.float32))


def test_norm_quant_feeds_the_int8_gemm(aria, oracle):
    # LN -> S1 -> QKV projection (aria_linear_w8a8_q), teacher-forced on the kernel's normalised tensor
    M, K, N = 256, 1536, 4608
    bits, x = inputs.residual_stream(M, K, 1)
    g, b = inputs.norm_params(K, 1)
    W = inputs.normal_f32((N, K), inputs.W_STD, 8, 50)
    bias_bits, bias = inputs.normal_bf16((N,), inputs.B_STD, 8, 51)
    wq, sw = aria.aria_quantize_weights_int8(dev_f32(W))
    xq, sx, xn = aria.aria_norm_quantize_act_int8(dev_bf16(bits), dev_f32(g), dev_f32(b), 0, 1e-5, want_xn=True)
    y = aria.aria_linear_w8a8_q(xq, sx, wq, sw, dev_bf16(bias_bits), aria.ACT_NONE, aria.F32)
    wq_o, sw_o = oracle.quant_int8_rows(W)
    r = oracle.linear_w8a8(host_f32(xn), wq_o, sw_o, bias.astype(np.float64))
    assert np.array_equal(xq.cpu().numpy(), r["xq"])
    assert rel_err(host_f32(y), r["y"]) <= 1e-3


# ------------------------------------------------------------------ attention
ATT_TOL = 1e-2       # DESIGN.md R22: bf16 probabilities (2^-9 each) + bf16 output rounding; north_star's bf16 gate is 2e-2


def _att_case(aria, oracle, B, S, H, tid=0, q_gain=1.0, scale=None, sample_bh=None):
    bits, x = inputs.qkv_activations(B, S, H, 64, tid, q_gain)
    QKV = dev_bf16(bits)
    amax = torch.zeros((B * S,), dtype=torch.float32, device="cuda")
    O = aria.aria_attention(QKV, B, S, H, 64, scale, row_absmax=amax)
    O2 = aria.aria_attention(QKV, B, S, H, 64, scale)
    torch.cuda.synchronize()
    assert torch.equal(O, O2)
    got = host_f32(O)
    # the fused absmax is exactly the row maximum of what was stored
    assert np.array_equal(amax.cpu().numpy(), np.abs(got).max(axis=1))
    if sample_bh is None:
        ref = oracle.attention(x, B, S, H, 64, scale)
        e = rel_err(got, ref)
        assert e <= ATT_TOL, e
        # element-wise: |err| <= 2^-8 |ref| (output rounding) + a P-rounding term relative to the row's magnitude
        bound = 2.0 ** -8 * np.abs(ref) + 2.0 ** -8 * np.abs(ref).max()
        assert np.all(np.abs(got - ref) <= bound)
        return e
    # full-size case: the oracle on sampled (sequence, head) pairs, all queries of each (exact: a head's output
    # depends only on its own q, k, v columns of its own sequence)
    x3 = x.reshape(B, S, 3, H, 64)
    g3 = got.reshape(B, S, H, 64)
    worst = 0.0
    for (b, h) in sample_bh:
        sub = np.ascontiguousarray(x3[b, :, :, h, :]).reshape(S, 3 * 64)
        ref = oracle.attention(sub, 1, S, 1, 64, scale)
        worst = max(worst, rel_err(g3[b, :, h, :], ref))
    assert worst <= ATT_TOL, worst
    return worst


@pytest.mark.parametrize("B,S,H", [(1, 128, 1), (2, 256, 3), (1, 384, 2), (3, 512, 2)])
def test_attention_whole_tiles(aria, oracle, B, S, H):
    _att_case(aria, oracle, B, S, H, tid=S % 5)


@pytest.mark.parametrize("B,S,H", [(1, 1, 1), (1, 37, 1), (2, 100, 2), (1, 129, 1), (2, 300, 3), (1, 1000, 2)])
def test_attention_ragged_sequences(aria, oracle, B, S, H):
    # key tail masked, query tail not stored, and a sequence's last tile never reads the next sequence
    _att_case(aria, oracle, B, S, H, tid=S % 7)


@pytest.mark.parametrize("q_gain,scale", [(4.0, None), (0.05, None), (1.0, 1.0), (12.0, 0.125)])
def test_attention_peaked_flat_and_scaled(aria, oracle, q_gain, scale):
    # sharp softmax (running maximum moves often: the O rescale path), near-uniform softmax, a non-default scale
    _att_case(aria, oracle, 2, 640, 2, tid=2, q_gain=q_gain, scale=scale)


def test_attention_structured_exact(aria, oracle):
    # every key of a sequence equal -> uniform weights -> O = mean of V; V on a coarse grid so the mean of 256
    # values is exact in bf16 arithmetic up to the final rounding
    B, S, H = 1, 256, 2
    bits, x = inputs.qkv_activations(B, S, H, 64, 9)
    x3 = x.reshape(B, S, 3, H, 64)
    x3[:, :, 1] = x3[:, :1, 1]
    x3[:, :, 2] = np.round(x3[:, :, 2] * 4) / 4
    O = aria.aria_attention(dev_bf16(inputs.bf16_bits(x3.reshape(B * S, -1))), B, S, H)
    ref = np.broadcast_to(x3[:, :, 2].astype(np.float64).mean(axis=1, keepdims=True), (B, S, H, 64)).reshape(B * S, -1)
    assert np.abs(host_f32(O) - ref).max() <= 2.0 ** -8 * np.abs(ref).max() + 1e-6


def test_attention_medium_and_small_music_full_size(aria, oracle):
    # the shapes of the bench: 2 CFG branches x 1024 tokens, 24 heads (medium) / 16 heads (small-music)
    _att_case(aria, oracle, 2, 1024, 24, tid=1, sample_bh=[(0, 0), (1, 23), (0, 11), (1, 5)])
    _att_case(aria, oracle, 2, 1024, 16, tid=2, sample_bh=[(0, 15), (1, 0), (1, 8)])


def test_attention_rejects_what_it_does_not_support(aria):
    QKV = torch.zeros((128, 3 * 32), dtype=torch.bfloat16, device="cuda")
    O = torch.zeros((128, 32), dtype=torch.bfloat16, device="cuda")
    L = aria.lib()
    st = torch.cuda.current_stream().cuda_stream
    assert L.aria_attention(QKV.data_ptr(), 1, 128, 1, 32, 0.125, O.data_ptr(), None, st) == -2     # Dh != 64
    assert L.aria_attention(QKV.data_ptr(), 1, 128, 1, 64, 0.0, O.data_ptr(), None, st) == -2       # scale <= 0
    assert L.aria_attention(None, 1, 128, 1, 64, 0.125, O.data_ptr(), None, st) == -1


# ------------------------------------------------------------------ the pieces chained as in a DiT block
def test_block_attention_half_chained_and_teacher_forced(aria, oracle):
    """x -> LayerNorm+S1 -> QKV (W8A8) -> attention (+ fused per-token absmax) -> rounding-only S1 -> out-proj."""
    B, S, H = 2, 256, 4
    M, D = B * S, H * 64
    bits, x = inputs.residual_stream(M, D, 4)
    g, b = inputs.norm_params(D, 4)
    Wqkv = inputs.normal_f32((3 * D, D), 0.06, 8, 60)        # scores of O(1) magnitude at this small width
    Wout = inputs.normal_f32((D, D), inputs.W_STD, 8, 61)
    bq_bits, bq = inputs.normal_bf16((3 * D,), inputs.B_STD, 8, 62)
    bo_bits, bo = inputs.normal_bf16((D,), inputs.B_STD, 8, 63)
    wq1, sw1 = aria.aria_quantize_weights_int8(dev_f32(Wqkv))
    wq2, sw2 = aria.aria_quantize_weights_int8(dev_f32(Wout))
    xq, sx, xn = aria.aria_norm_quantize_act_int8(dev_bf16(bits), dev_f32(g), dev_f32(b), 0, 1e-5, want_xn=True)
    qkv = aria.aria_linear_w8a8_q(xq, sx, wq1, sw1, dev_bf16(bq_bits), aria.ACT_NONE, aria.BF16)
    amax = torch.zeros((M,), dtype=torch.float32, device="cuda")
    o = aria.aria_attention(qkv, B, S, H, 64, None, row_absmax=amax)
    oq, so = aria.aria_round_act_int8(o, amax)
    assert float(amax.min()) > 0.0                                # clear = False leaves the buffer alone
    y = aria.aria_linear_w8a8_q(oq, so, wq2, sw2, dev_bf16(bo_bits), aria.ACT_NONE, aria.F32)
    torch.cuda.synchronize()
    # stage by stage, each oracle stage fed the GPU's actual input of that stage
    w1_o, s1_o = oracle.quant_int8_rows(Wqkv)
    r1 = oracle.linear_w8a8(host_f32(xn), w1_o, s1_o, bq.astype(np.float64))
    assert np.array_equal(xq.cpu().numpy(), r1["xq"])
    assert rel_err(host_f32(qkv), r1["y"]) <= 2.0 ** -8
    ref_o = oracle.attention(host_f32(qkv), B, S, H, 64)
    assert rel_err(host_f32(o), ref_o) <= ATT_TOL
    q_o, s_o = oracle.quant_int8_rows(host_f32(o))               # fused absmax + rounding pass == S1 of O
    assert np.array_equal(oq.cpu().numpy(), q_o) and np.array_equal(so.cpu().numpy(), s_o)
    q_g, s_g = aria.aria_quantize_act_int8(o)
    assert torch.equal(q_g, oq) and torch.equal(s_g, so)
    w2_o, s2_o = oracle.quant_int8_rows(Wout)
    r2 = oracle.linear_w8a8(host_f32(o), w2_o, s2_o, bo.astype(np.float64))
    assert rel_err(host_f32(y), r2["y"]) <= 1e-3


def test_block_stack_every_stage_teacher_forced_and_graph_replay(aria, oracle):
    """BlockStack (stack.py): 2 whole DiT blocks, 9 launches each; every stage's output against the oracle fed the
    GPU's actual input of that stage; the captured graph reproduces the eager run bit for bit."""
    from paper_2607_08526_b200.stack import BlockStack
    st = BlockStack(B=2, S=160, n_blocks=2, d_model=256, keep_host=True)
    st.run(tap=True)
    torch.cuda.synchronize()
    taps = st.taps
    for blk, (t, hst) in enumerate(zip(taps, st.host)):
        f = lambda k: host_f32(t[k])
        # LayerNorm 1 + S1
        ref = oracle.norm_rows(f("src"), hst["g1"], hst["b1"], 0, 1e-5)
        check_bf16_out(host_bits16(t["xn1"]), ref, inputs.bf16_bits(oracle.round_out(ref, 1)), 2e-6, 0.01)
        q, s = oracle.quant_int8_rows(f("xn1"))
        assert np.array_equal(t["xq1"].cpu().numpy(), q) and np.array_equal(t["sx1"].cpu().numpy(), s)
        # QKV
        wq, sw = oracle.quant_int8_rows(hst["qkv"]["W"])
        y = oracle.epilogue_w8a8(oracle.gemm_i8(q, wq), s, sw, hst["qkv"]["b"].astype(np.float64))
        assert rel_err(f("qkv"), y) <= 2.0 ** -8
        # attention, fused absmax + rounding-only S1
        assert rel_err(f("att"), oracle.attention(f("qkv"), st.B, st.S, st.H, 64)) <= ATT_TOL
        q, s = oracle.quant_int8_rows(f("att"))
        assert np.array_equal(t["xq2"].cpu().numpy(), q) and np.array_equal(t["sx2"].cpu().numpy(), s)
        # out-projection
        wq, sw = oracle.quant_int8_rows(hst["out"]["W"])
        y = oracle.epilogue_w8a8(oracle.gemm_i8(q, wq), s, sw, hst["out"]["b"].astype(np.float64))
        assert rel_err(f("h2"), y) <= 2.0 ** -8
        # LayerNorm 2 + S1, MLP up + GELU, S1 + MLP down
        ref = oracle.norm_rows(f("h2"), hst["g2"], hst["b2"], 0, 1e-5)
        check_bf16_out(host_bits16(t["xn3"]), ref, inputs.bf16_bits(oracle.round_out(ref, 1)), 2e-6, 0.01)
        q, s = oracle.quant_int8_rows(f("xn3"))
        assert np.array_equal(t["xq3"].cpu().numpy(), q) and np.array_equal(t["sx3"].cpu().numpy(), s)
        wq, sw = oracle.quant_int8_rows(hst["up"]["W"])
        y = oracle.epilogue_w8a8(oracle.gemm_i8(q, wq), s, sw, hst["up"]["b"].astype(np.float64), oracle.ACT_GELU_ERF)
        assert rel_err(f("mid"), y) <= 2.0 ** -8
        wq, sw = oracle.quant_int8_rows(hst["down"]["W"])
        r = oracle.linear_w8a8(f("mid"), wq, sw, hst["down"]["b"].astype(np.float64))
        assert rel_err(f("h"), r["y"]) <= 2.0 ** -8
        if blk + 1 < len(taps):
            assert torch.equal(taps[blk + 1]["src"], t["h"])          # truly chained
    eager = st.h.clone()
    assert float(st.amax.abs().max()) == 0.0                          # the rounding pass left the buffer cleared
    st.capture()
    st.h.zero_()
    st.replay()
    st.replay()
    torch.cuda.synchronize()
    assert torch.equal(st.h, eager)


@pytest.mark.parametrize("B,S,H", [(1, 2304, 2), (5, 256, 1), (1, 4000, 1)])
def test_attention_long_and_many_sequences(aria, oracle, B, S, H):
    # more key tiles than the bench shape (barrier phases wrap many times), more sequences than CFG's two
    _att_case(aria, oracle, B, S, H, tid=S % 11, sample_bh=[(0, 0), (B - 1, H - 1)])


def test_block_stack_full_size_as_benched_sampled(aria, oracle):
    """BlockStack at the size bench.py times (2 x 1024 tokens, d_model 1536, 24 heads), 2 blocks: every stage against
    the oracle on sampled rows / heads, each stage fed the GPU's actual input (a row of a linear depends only on its
    own input row; a head's attention only on its own columns of its own sequence)."""
    from paper_2607_08526_b200.stack import BlockStack
    st = BlockStack(B=2, S=1024, n_blocks=2, d_model=1536, keep_host=True)
    st.run(tap=True)
    torch.cuda.synchronize()
    rows = np.array([0, 1, 511, 1023, 1024, 1500, 2047])
    for t, hst in zip(st.taps, st.host):
        f = lambda k, r=None: host_f32(t[k] if r is None else t[k][r])        # noqa: E731
        ridx = torch.from_numpy(rows).cuda()
        # LayerNorm + S1 (rows), QKV (rows)
        src = f("src", ridx)
        ref = oracle.norm_rows(src, hst["g1"], hst["b1"], 0, 1e-5)
        xn = f("xn1", ridx)
        check_bf16_out(host_bits16(t["xn1"][ridx]), ref, inputs.bf16_bits(oracle.round_out(ref, 1)), 2e-6, 0.01)
        q, s = oracle.quant_int8_rows(xn)
        assert np.array_equal(t["xq1"][ridx].cpu().numpy(), q) and np.array_equal(t["sx1"][ridx].cpu().numpy(), s)
        wq, sw = oracle.quant_int8_rows(hst["qkv"]["W"])
        y = oracle.epilogue_w8a8(oracle.gemm_i8(q, wq), s, sw, hst["qkv"]["b"].astype(np.float64))
        assert rel_err(f("qkv", ridx), y) <= 2.0 ** -8
        # attention on sampled (sequence, head) pairs, all queries
        qkv3 = f("qkv").reshape(st.B, st.S, 3, st.H, 64)
        att3 = f("att").reshape(st.B, st.S, st.H, 64)
        for (b, h) in [(0, 0), (1, st.H - 1), (0, 7)]:
            sub = np.ascontiguousarray(qkv3[b, :, :, h, :]).reshape(st.S, 192)
            assert rel_err(att3[b, :, h, :], oracle.attention(sub, 1, st.S, 1, 64)) <= ATT_TOL
        # fused absmax + rounding-only S1 of the attention output, out-projection
        q, s = oracle.quant_int8_rows(f("att", ridx))
        assert np.array_equal(t["xq2"][ridx].cpu().numpy(), q) and np.array_equal(t["sx2"][ridx].cpu().numpy(), s)
        wq, sw = oracle.quant_int8_rows(hst["out"]["W"])
        y = oracle.epilogue_w8a8(oracle.gemm_i8(q, wq), s, sw, hst["out"]["b"].astype(np.float64))
        assert rel_err(f("h2", ridx), y) <= 2.0 ** -8
        # LayerNorm 2 + S1, up + GELU, S1 + down
        ref = oracle.norm_rows(f("h2", ridx), hst["g2"], hst["b2"], 0, 1e-5)
        check_bf16_out(host_bits16(t["xn3"][ridx]), ref, inputs.bf16_bits(oracle.round_out(ref, 1)), 2e-6, 0.01)
        q, s = oracle.quant_int8_rows(f("xn3", ridx))
        assert np.array_equal(t["xq3"][ridx].cpu().numpy(), q) and np.array_equal(t["sx3"][ridx].cpu().numpy(), s)
        wq, sw = oracle.quant_int8_rows(hst["up"]["W"])
        y = oracle.epilogue_w8a8(oracle.gemm_i8(q, wq), s, sw, hst["up"]["b"].astype(np.float64), oracle.ACT_GELU_ERF)
        assert rel_err(f("mid", ridx), y) <= 2.0 ** -8
        wq, sw = oracle.quant_int8_rows(hst["down"]["W"])
        r = oracle.linear_w8a8(f("mid", ridx), wq, sw, hst["down"]["b"].astype(np.float64))
        assert rel_err(f("h", ridx), r["y"]) <= 2.0 ** -8
