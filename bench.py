#!/usr/bin/env python
"""bench.py -- throughput of the quantized DiT linear path on B200 (BASELINE.json metric).

A STEP is one pass of the whole hot path over config C5: one denoising step's 96 linears
(24 blocks x QKV / out-proj / MLP up+GELU / MLP down, M = 2048 tokens), replayed as a CUDA graph
once in W8A8 mode (S1 activation quantisation + S2 int8 tcgen05 GEMM + S3 rescale/bias/GELU
epilogue) and once in W4A16 mode (S4 on-chip int4 dequant + bf16 tcgen05 GEMM).  Weights are
quantised once at load (S0) and are resident; inputs are resident for `value`, and come from /
return to pinned HOST buffers through aria_denoiser_linears_host for `e2e`.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--no-per-linear]

One JSON line on stdout (rank 0).  See DESIGN.md "Measurement" for every field.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "quantized DiT linear throughput: W8A8 int8 TOPS + W4A16 effective bf16 TFLOPS over one C5 denoising-step stack"
UNIT = "Top/s"
WORKLOAD = "C5: 24 blocks x (QKV 1536->4608, out 1536->1536, MLP 1536->6144->1536), M=2048, all-W8A8 then all-W4A16, CUDA-graph replay"
W4A16_TRAFFIC_SRC = "profiles/r2_w4a16_full.md"   # ncu --set full summaries the `traffic` figures are read from
W8A8_TRAFFIC_SRC = "profiles/r2_w8a8_full.md"
NOMINAL_INT8_OVER_BF16 = 2.0     # B200_PROFILING.md: 4.5 POP/s int8 vs 2.25 PFLOP/s bf16, dense
BURST_REGION_S = 1.0             # a timed region shorter than this runs at burst clocks: score against the burst peak


def profile_traffic(rel_path: str):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum, mean over the captured launches) read
    from a committed ncu summary under profiles/ -- nothing typed in by hand.  None if the file or rows are missing."""
    unit = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    tot = {}
    try:
        for ln in open(os.path.join(ROOT, rel_path)):
            c = [x.strip() for x in ln.strip().strip("|").split("|")]
            if len(c) >= 3 and c[0] in ("dram__bytes_read.sum", "dram__bytes_write.sum") and c[1] in unit:
                tot[c[0]] = [float(v) * unit[c[1]] for v in c[2:]]
    except OSError:
        return None
    if len(tot) != 2 or len(tot["dram__bytes_read.sum"]) != len(tot["dram__bytes_write.sum"]):
        return None
    per = [r + w for r, w in zip(tot["dram__bytes_read.sum"], tot["dram__bytes_write.sum"])]
    return sum(per) / len(per)


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "bf16_burst": d["bf16_tflops"],
                "bf16_sustained": d.get("bf16_tflops_sustained", d["bf16_tflops"]), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_burst": 1590.0, "bf16_sustained": 1400.0, "source": "fallback"}


class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                   "--format=csv,noheader,nounits", "-lms", "100"],
                                  stdout=self.f, stderr=subprocess.DEVNULL)

    def stop(self):
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(", ") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        sm, mx, reasons = [], 0.0, set()
        for r in rows:
            try:
                sm.append(float(r[0])); mx = max(mx, float(r[1]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.strip().lower().startswith("active"):
                    reasons.add(name)
        busy = [c for c in sm if c > 0.5 * mx] or sm
        return {"sm_mhz": statistics.median(busy) if busy else None, "sm_max_mhz": mx or None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------ reference arm (the oracle)
def oracle_sample(rows: int):
    """Time the oracle, as it stands, on block 0's four linears at `rows` tokens, both modes."""
    from oracle import oracle as orc
    from paper_2607_08526_b200 import inputs
    orc.build()
    ops, t = 0, 0.0
    for which in range(4):
        L = inputs.c5_layer(0, which, M=rows)
        x, W, b = L["X"], L["W"], L["b"][1].astype(np.float64)
        act = 1 if L["act"] == "gelu" else 0
        wq, sw = orc.quant_int8_rows(W)                      # S0 is load-time: not timed
        codes, sg, _ = orc.quant_int4_groups(W)
        t0 = time.perf_counter()
        y8 = orc.linear_w8a8(x, wq, sw, b, act)["y"]         # S1 + S2 + S3
        orc.round_out(y8, orc.OUT_BF16)
        y4 = orc.linear_w4a16(x, codes, sg, b, act, variant=0)  # S4
        orc.round_out(y4, orc.OUT_BF16)
        t += time.perf_counter() - t0
        ops += 2 * (2 * rows * L["K"] * L["N"])
    return ops, t, orc.num_threads()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    rows = 128
    for _ in range(args.warmup):
        oracle_sample(8)
    tot_ops, tot_t, cores = 0, 0.0, 1
    for _ in range(args.steps):
        ops, t, cores = oracle_sample(rows)
        tot_ops += ops
        tot_t += t
    v = tot_ops / tot_t / 1e12
    sample = f"per step: block 0's 4 linears at {rows} tokens, W8A8 (S1-S3) + W4A16 (S4), bf16 out"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int64/f64",
        "data": "synthetic", "config": {"workload": WORKLOAD, "sample": sample},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ------------------------------------------------------------------ our arm
def max_over_ranks(value: float, dist, device="cuda") -> float:
    """Replicas only: the job's step time is the slowest rank's; no data-path collective."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def time_region(torch, fn, iters):
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(iters):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / iters      # ms per call


def tensor_peaks(aria):
    """The tensor pipe's own peak on this device (aria_tensor_peak: back-to-back tcgen05.mma issue loop, no
    memory traffic): int8 and bf16, BURST (one ~5 ms launch).  Best of 1-CTA / CTA-pair issue."""
    out = {}
    for name, kind in (("int8", 0), ("bf16", 1)):
        best = None
        for ctas in (2, 1):
            b = aria.aria_tensor_peak(kind, ctas, 16384, 0.0)
            if best is None or b["ops_per_s"] > best[1]["ops_per_s"]:
                best = (ctas, b)
        ctas, b = best
        out[name] = {"burst": b["ops_per_s"] / 1e12, "burst_sm_mhz": round(b["sm_mhz"], 1),
                     "cycles_per_mma": round(b["cycles_per_mma"], 2), "ctas": ctas, "unit": "Top/s",
                     "how": "aria_tensor_peak: 16384 x 4 tcgen05.mma 128*ctas x 256 x K per SM, operands in shared memory"}
    return out


def tensor_peaks_sustained(aria, tp, seconds=3.0):
    """Same loop, launched back to back for `seconds`; the last launch runs at the clocks the power cap allows."""
    for name, kind in (("int8", 0), ("bf16", 1)):
        su = aria.aria_tensor_peak(kind, tp[name]["ctas"], 16384, seconds)
        tp[name]["sustained"] = su["ops_per_s"] / 1e12
        tp[name]["sustained_sm_mhz"] = round(su["sm_mhz"], 1)


def sustained_record(torch, step, ops_step, ms_short, index, seconds=3.0):
    """The same step replayed back to back for >= `seconds`: what a long denoising job sees once the part
    sits at its power cap (the 20-step number above is a burst number)."""
    sampler = ClockSampler(index)
    torch.cuda.synchronize()
    n = max(20, int(seconds / (ms_short * 1e-3) * 1.1))
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    ev[0].record()
    for i in range(n):
        step()
        if i == n - n // 4 - 1:
            ev[1].record()
    ev[2].record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    tail_ms = ev[1].elapsed_time(ev[2]) / (n // 4)        # the last quarter: clocks have settled
    all_ms = ev[0].elapsed_time(ev[2]) / n
    return {"seconds": round(ev[0].elapsed_time(ev[2]) * 1e-3, 2), "steps": n, "ms_per_step": all_ms,
            "ms_per_step_last_quarter": tail_ms, "value_last_quarter": ops_step / (tail_ms * 1e-3) / 1e12,
            "ratio_to_short_run": ms_short / tail_ms, "clocks": clocks}


def per_linear_table(torch, aria, inputs, pk):
    """BASELINE metric per DiT linear: C2, C3 (W8A8) and the 9 C4 cases (W4A16), each launched from
    a CUDA graph that cycles through enough distinct weight copies to exceed 2 x L2 (HBM-cold)."""
    out = []
    L2 = 126e6
    try:
        peak8 = tensor_peaks(aria)["int8"]["burst"]
    except Exception:                            # noqa: BLE001
        peak8 = pk["bf16_burst"] * NOMINAL_INT8_OVER_BF16

    def dev_bf16(bits):
        return torch.from_numpy(bits.view(np.int16).copy()).cuda().view(torch.bfloat16)

    def bench_case(name, mode, M, K, N, act):
        bits, _ = inputs.normal_bf16((M, K), 1.0, 9, M + K + N)
        X = dev_bf16(bits)
        W = torch.from_numpy(inputs.normal_f32((N, K), inputs.W_STD, 9, M + K + N + 1)).cuda()
        b = dev_bf16(inputs.normal_bf16((N,), inputs.B_STD, 9, M + K + N + 2)[0])
        if mode in ("w8a8", "w8a8_gemm"):
            wq, sc = aria.aria_quantize_weights_int8(W)
            wbytes = N * K + 4 * N
        else:
            wq, sc = aria.aria_quantize_weights_int4(W)
            wbytes = N * K // 2 + 2 * N * K // 32
        del W
        ncopy = max(2, int(2 * L2 // wbytes) + 1)
        ncopy = min(ncopy, 64)
        wqs = [wq.clone() for _ in range(ncopy)]
        scs = [sc.clone() for _ in range(ncopy)]
        Y = torch.empty((M, N), dtype=torch.bfloat16, device="cuda")
        ws = aria.workspace(aria.aria_workspace_bytes(M, K, N, aria.W8A8 if mode.startswith("w8a8") else aria.W4A16))

        xq_sx = aria.aria_quantize_act_int8(X) if mode == "w8a8_gemm" else None

        def launch_all():
            for i in range(ncopy):
                if mode == "w8a8":
                    aria.aria_linear_w8a8(X, wqs[i], scs[i], b, act, aria.BF16, ws=ws, out=Y)
                elif mode == "w8a8_gemm":      # S2 + S3 alone, on already-quantised activations
                    aria.aria_linear_w8a8_q(xq_sx[0], xq_sx[1], wqs[i], scs[i], b, act, aria.BF16, out=Y)
                else:
                    aria.aria_linear_w4a16(X, wqs[i], scs[i], b, act, aria.BF16, ws=ws, out=Y)
        launch_all()
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            launch_all()
        g.replay()
        ms = time_region(torch, g.replay, 5) / ncopy
        ops = 2.0 * M * N * K
        abytes = M * K * 2 + wbytes + 2 * N + M * N * 2          # X + weights(+scales) + bias + Y
        tput = ops / (ms * 1e-3) / 1e12
        i8 = mode.startswith("w8a8")
        # int8: the MEASURED tensor peak (issue loop, burst); bf16: the driver-measured cuBLAS burst figure
        peak_t = peak8 if i8 else pk["bf16_burst"]
        if mode == "w8a8_gemm":
            abytes = M * K + 4 * M + wbytes + 2 * N + M * N * 2  # Xq + sx instead of X
        t_roof = max(ops / (peak_t * 1e12), abytes / (pk["hbm_gbs"] * 1e9))
        out.append({"case": name, "mode": mode, "M": M, "K": K, "N": N, "us": round(ms * 1e3, 2),
                    "tput": round(tput, 1), "unit": "TOPS" if i8 else "eff_TFLOPS",
                    "frac_of_tensor_peak": round(tput / peak_t, 3),
                    "gbs": round(abytes / (ms * 1e-3) / 1e9, 1),
                    "bound": "tensor" if ops / (peak_t * 1e12) >= abytes / (pk["hbm_gbs"] * 1e9) else "hbm",
                    "roofline_frac": round(t_roof / (ms * 1e-3), 3)})
        del wqs, scs

    bench_case("C2 qkv", "w8a8", 512, 1536, 4608, aria.ACT_NONE)
    bench_case("C2 out", "w8a8", 512, 1536, 1536, aria.ACT_NONE)
    bench_case("C3 up+gelu", "w8a8", 4096, 1536, 6144, aria.ACT_GELU_ERF)
    bench_case("C3 down", "w8a8", 4096, 6144, 1536, aria.ACT_NONE)
    # north_star's large-M target is stated for the int8 GEMM: S2 + S3 alone on pre-quantised activations
    bench_case("C3 up+gelu GEMM only", "w8a8_gemm", 4096, 1536, 6144, aria.ACT_GELU_ERF)
    bench_case("C3 down GEMM only", "w8a8_gemm", 4096, 6144, 1536, aria.ACT_NONE)
    for M in inputs.C4_MS:
        for (K, N) in inputs.C4_SHAPES:
            bench_case(f"C4 M={M}", "w4a16", M, K, N, aria.ACT_NONE)
    return out


def next_rows(torch, aria, inputs, pk):
    """SURVEY S8(f) rows built in round 2, each timed the same way as the main step (CUDA-graph replay, CUDA
    events): NEXT-1 the C5 stack in q8 weight-only mode (W8A16), NEXT-3/4 the paper's per-clip unit -- 8
    sampling steps of the small-music stack (d_model 1024 x 20 blocks, L47) in W8A8 with the
    steering step inside the captured graph (L77), strength refreshed per step."""
    from paper_2607_08526_b200.stack import LinearStack
    out = {}
    st = LinearStack(aria.W8A16, M=2048)
    st.capture()
    for _ in range(3):
        st.replay()
    ms = time_region(torch, st.replay, 10)
    out["w8a16_c5_stack"] = {"ms": ms, "eff_tflops": st.ops / (ms * 1e-3) / 1e12,
                             "frac_of_bf16_burst": st.ops / (ms * 1e-3) / 1e12 / pk["bf16_burst"],
                             "launches": len(st.specs), "weight_mb": round(st.weight_bytes / 1e6, 1)}
    del st
    # NEXT-2: the producers around the linears.  (a) aria_attention alone at the step's shape (2 CFG branches x
    # 1024 tokens, 24 heads of 64): the exponential unit is its ceiling (16 MUFU lanes per SM: 16384 ex2 per
    # 128 x 128 tile = 1024 cycles against 640 cycles of tensor work); reported as a ceiling beside the
    # measured cycles per tile, because the kernel is not bound by it today (attention.cu header).
    # (b) aria_norm_quantize_act_int8 alone (HBM bound: 2 bytes in, 1 byte out per element).  (c) the whole
    # truly chained W8A8 step with both inside the captured graph (BlockStack).
    from paper_2607_08526_b200.stack import BlockStack
    B, S, H = 2, 1024, inputs.D_MODEL // inputs.HEAD_DIM
    bits, _ = inputs.qkv_activations(B, S, H, inputs.HEAD_DIM, 0)
    qkvs = [torch.from_numpy(bits.view(np.int16).copy()).cuda().view(torch.bfloat16) for _ in range(8)]   # 8 x 18.9 MB > L2
    O = torch.empty((B * S, H * inputs.HEAD_DIM), dtype=torch.bfloat16, device="cuda")

    def att_all():
        for q in qkvs:
            aria.aria_attention(q, B, S, H, inputs.HEAD_DIM, None, out=O)
    att_all()
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        att_all()
    g.replay()
    ms = time_region(torch, g.replay, 10) / len(qkvs)
    flops = 4.0 * B * H * S * S * inputs.HEAD_DIM
    exps = float(B * H * S * S)
    # SM clock UNDER this kernel (nvidia-smi sampled over ~0.4 s of back-to-back replays), SM count from the device
    cs = ClockSampler(torch.cuda.current_device())
    t_end = time.time() + 0.4
    while time.time() < t_end:
        for _ in range(50):
            g.replay()
        torch.cuda.synchronize()
    clk = cs.stop()
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    sm_hz = (clk.get("sm_mhz") or 1850.0) * 1e6
    tiles = B * H * (S // 128) * (S // 128)                    # (128-query tile, 128-key tile) pairs
    cyc_per_tile_sm = ms * 1e-3 * sm_hz * sms / tiles         # SM cycles spent per pair, per SM
    out["attention_2x1024x24x64"] = {
        "us": ms * 1e3, "tflops": flops / (ms * 1e-3) / 1e12, "gexp_per_s": exps / (ms * 1e-3) / 1e9,
        # a CEILING, not the measured bound: attention.cu's role timings show the kernel bound by the per-tile chain of
        # dependent phases (2990 cycles per key tile per CTA, 2 CTAs per SM); removing every ex2 gains only 16 %
        "ceiling": "alu (MUFU ex2)", "ceiling_gexp_per_s": sms * 16 * sm_hz / 1e9,
        "frac_of_mufu_ceiling": exps / (ms * 1e-3) / (sms * 16 * sm_hz),
        "sm_mhz_under_kernel": clk.get("sm_mhz"), "sms": sms,
        "cycles_per_tile_per_sm": {"measured": cyc_per_tile_sm, "mufu_floor": 1024, "tensor_floor": 640},
        "ceiling_note": "SMs x 16 ex2 / clk x sampled SM clock (B300_MICROARCH.md unit counts); 16384 ex2 per 128x128 "
                        "tile = 1024 cycles, 640 cycles of tcgen05.mma per tile (attention.cu header)",
        "frac_of_bf16_burst": flops / (ms * 1e-3) / 1e12 / pk["bf16_burst"]}
    del qkvs
    xs = [torch.from_numpy(inputs.residual_stream(2048, inputs.D_MODEL, i)[0].view(np.int16).copy()).cuda().view(torch.bfloat16)
          for i in range(24)]                                                                              # 24 x 6.3 MB > L2
    gm, bt = inputs.norm_params(inputs.D_MODEL, 0)
    gm, bt = torch.from_numpy(gm).cuda(), torch.from_numpy(bt).cuda()
    xq = torch.empty((2048, inputs.D_MODEL), dtype=torch.int8, device="cuda")
    sx = torch.empty((2048,), dtype=torch.float32, device="cuda")

    def nq_all():
        for x in xs:
            aria.aria_norm_quantize_act_int8(x, gm, bt, aria.NORM_LAYER, 1e-5, out=(xq, sx))
    nq_all()
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        nq_all()
    g.replay()
    ms = time_region(torch, g.replay, 10) / len(xs)
    nbytes = 2048 * inputs.D_MODEL * 3 + 2048 * 4 + 2 * 4 * inputs.D_MODEL
    out["norm_quant_2048x1536"] = {"us": ms * 1e3, "gbs": nbytes / (ms * 1e-3) / 1e9,
                                   "hbm_frac_measured": nbytes / (ms * 1e-3) / 1e9 / pk["hbm_gbs"], "bytes": nbytes}
    del xs
    bs = BlockStack(B=2, S=1024)
    bs.capture()
    for _ in range(3):
        bs.replay()
    ms = time_region(torch, bs.replay, 10)
    out["dit_blocks_w8a8_chained"] = {
        "ms": ms, "launches": bs.launches_per_block * bs.n_blocks,
        "linear_tops": bs.lin_ops / (ms * 1e-3) / 1e12, "all_tops": bs.ops / (ms * 1e-3) / 1e12,
        "what": "24 blocks x (LayerNorm+S1, QKV, attention+absmax, S1 rounding, out-proj, LayerNorm+S1, up+GELU, S1, down), "
                "every tensor chained, one CUDA graph"}
    del bs
    d_model, n_blocks = inputs.MODELS["small-music"]
    sm = LinearStack(aria.W8A8, M=2048, n_blocks=n_blocks, d_model=d_model)
    d, norm = inputs.steer_direction(d_model, 0)
    sm.set_steering(n_blocks // 2, d, norm)
    sm.capture()
    span = [0.0, 0.0, 0.3, 0.3, 0.3, 0.3, 0.0, 0.0]
    off = [0.0] * inputs.SAMPLING_STEPS
    for _ in range(2):
        sm.sample(span)
    ms_on = time_region(torch, lambda: sm.sample(span), 5)
    ms_off = time_region(torch, lambda: sm.sample(off), 5)
    out["small_music_8_steps_w8a8_steered"] = {
        "ms_per_clip": ms_on, "ms_per_clip_strength_0": ms_off, "steps": inputs.SAMPLING_STEPS,
        "tops": inputs.SAMPLING_STEPS * sm.ops / (ms_on * 1e-3) / 1e12, "layers_per_step": len(sm.specs),
        "steering": "additive (eq. 2) after block 10, strength 0.3 in steps 2-5, device scalar refreshed per replay"}
    return out


def hbm_passes(torch, aria, inputs, pk):
    """The HBM-bound passes around the GEMMs, each alone on distinct buffers totalling > 2 x L2 (HBM-cold), replayed
    from one CUDA graph: S1 (aria_quantize_act_int8) and norm + S1 (aria_norm_quantize_act_int8) at the step's
    shape, at C3's down-projection input and at a large token count.  Bytes are algorithmic: 2 in + 1 out per
    element + 4 per row."""
    out = []
    for (M, K) in ((2048, 1536), (4096, 6144), (16384, 1536)):
        nbuf = max(2, int(2 * 126e6 // (M * K * 2)) + 1)
        xs = [torch.randn((M, K), device="cuda").to(torch.bfloat16) for _ in range(nbuf)]
        xq = torch.empty((M, K), dtype=torch.int8, device="cuda")
        sx = torch.empty((M,), dtype=torch.float32, device="cuda")
        gm = torch.ones((K,), dtype=torch.float32, device="cuda")
        bt = torch.zeros((K,), dtype=torch.float32, device="cuda")
        L = aria.lib()
        import ctypes
        st = lambda: ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)   # noqa: E731

        def s1_all():
            for x in xs:
                rc = L.aria_quantize_act_int8(x.data_ptr(), aria.BF16, M, K, xq.data_ptr(), sx.data_ptr(), st())
                assert rc == 0

        def nq_all():
            for x in xs:
                aria.aria_norm_quantize_act_int8(x, gm, bt, aria.NORM_LAYER, 1e-5, out=(xq, sx))
        for name, fn in (("S1", s1_all), ("LayerNorm+S1", nq_all)):
            fn()
            torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                fn()
            g.replay()
            ms = time_region(torch, g.replay, 5) / nbuf
            nbytes = M * K * 3 + 4 * M
            out.append({"pass": name, "M": M, "K": K, "us": round(ms * 1e3, 2), "gbs": round(nbytes / (ms * 1e-3) / 1e9, 1),
                        "hbm_frac_measured": round(nbytes / (ms * 1e-3) / 1e9 / pk["hbm_gbs"], 3)})
        del xs
    return out


def small_m_stream(torch, aria, inputs, pk, iters=20):
    """SURVEY S8(d) 'C5-shaped stack at M=32, W4A16': the weight-bound regime.  One plan
    (aria_stack_plan_*) = ONE persistent weight-streaming kernel over all 96 layers, captured in a CUDA
    graph; 382 MB of packed weights + scales per replay exceed the 126 MB L2, so every replay is
    HBM-cold.  Also the three C4 shapes at M=32, each as a plan over enough independent linears of
    that shape to exceed 2 x L2.  Bytes are ALGORITHMIC: X + packed weights + scales + bias + Y."""
    from paper_2607_08526_b200.stack import LinearStack
    M = 32
    out = {}

    def timed_graph(run):
        run()
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            run()
        for _ in range(3):
            g.replay()
        # back-to-back replays inside one CUDA-event region (as the denoising loop issues them): a replay
        # timed on its own also counts the ~10 us the idle GPU waits for the graph launch
        ts = []
        for _ in range(5):
            ts.append(time_region(torch, g.replay, iters))
        return statistics.median(ts), min(ts)

    st = LinearStack(aria.W4A16, M=M, use_plan=True)
    assert aria.aria_stack_plan_is_streaming(st.plan), "M=32 W4A16 stack must take the stream kernel"
    abytes = sum(M * s["K"] * 2 + s["K"] * s["N"] // 2 + s["K"] * s["N"] // 16 + 2 * s["N"] + M * s["N"] * 2
                 for s in st.specs)
    med, best = timed_graph(st.run)
    out["c5_stack_m32"] = {"layers": len(st.specs), "launches_per_step": 2, "memsets_per_step": 1,
                           "launch_note": "stream kernel + the armed bf16 fallback kernel (exits at once unless the "
                                          "fp16 domain flag fired; both cooperative, inside the timed step) + one memset",
                           "us": round(med * 1e3, 2),
                           "us_best": round(best * 1e3, 2), "bytes": abytes,
                           "gbs": round(abytes / (med * 1e-3) / 1e9, 1),
                           "hbm_frac_measured": round(abytes / (med * 1e-3) / 1e9 / pk["hbm_gbs"], 3),
                           "hbm_frac_nominal_8000": round(abytes / (med * 1e-3) / 1e9 / 8000.0, 3),
                           "eff_tflops": round(st.ops / (med * 1e-3) / 1e12, 1)}
    del st
    cases = []
    for (K, N) in inputs.C4_SHAPES:
        wbytes = N * K // 2 + N * K // 16
        ncopy = int(2 * 126e6 // wbytes) + 1
        W = torch.from_numpy(inputs.normal_f32((N, K), inputs.W_STD, 9, K + N + 1)).cuda()
        wq, sc = aria.aria_quantize_weights_int4(W)
        del W
        bits, _ = inputs.normal_bf16((M, K), 1.0, 9, K + N)
        X = torch.from_numpy(bits.view(np.int16).copy()).cuda().view(torch.bfloat16)
        b = torch.from_numpy(inputs.normal_bf16((N,), inputs.B_STD, 9, K + N + 2)[0].view(np.int16).copy()).cuda().view(torch.bfloat16)
        specs = [{"K": K, "N": N, "act": aria.ACT_NONE, "in": X, "wq": wq.clone(), "w_scale": sc.clone(), "bias": b,
                  "out": torch.empty((M, N), dtype=torch.bfloat16, device="cuda")} for _ in range(ncopy)]
        layers = aria.make_layers(specs)
        plan = aria.aria_stack_plan_create(layers, M, aria.W4A16, aria.BF16)
        try:
            assert aria.aria_stack_plan_is_streaming(plan)
            med, best = timed_graph(lambda: aria.aria_stack_plan_run(plan))
        finally:
            torch.cuda.synchronize()
            aria.aria_stack_plan_destroy(plan)
        ab = M * K * 2 + wbytes + 2 * N + M * N * 2
        us = med * 1e3 / ncopy
        cases.append({"case": f"C4 M=32 {K}->{N}", "linears_per_launch": ncopy, "us_per_linear": round(us, 3),
                      "gbs": round(ab / (us * 1e-6) / 1e9, 1),
                      "hbm_frac_measured": round(ab / (us * 1e-6) / 1e9 / pk["hbm_gbs"], 3),
                      "eff_tflops": round(2.0 * M * N * K / (us * 1e-6) / 1e12, 1)})
        del specs, layers
    out["c4_m32_batched"] = cases
    return out


def run_ours(args):
    import torch
    from paper_2607_08526_b200 import binding as aria
    from paper_2607_08526_b200 import inputs
    from paper_2607_08526_b200.stack import LinearStack

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    aria.lib()
    pk = peaks()
    M = 2048
    t_load = time.perf_counter()
    st8 = LinearStack(aria.W8A8, M=M)
    st4 = LinearStack(aria.W4A16, M=M)
    st8.capture()
    st4.capture()
    torch.cuda.synchronize()
    log(f"[bench] stacks built + captured in {time.perf_counter() - t_load:.1f}s "
        f"(W8A8 {st8.weight_bytes / 1e6:.0f} MB, W4A16 {st4.weight_bytes / 1e6:.0f} MB resident)")

    def step():
        st8.replay()
        st4.replay()

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()

    sampler = ClockSampler(local) if rank == 0 else None
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * args.steps + 1)]
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    ev[0].record()
    for i in range(args.steps):
        st8.replay()
        ev[2 * i + 1].record()
        st4.replay()
        ev[2 * i + 2].record()
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    total_ms = ev[0].elapsed_time(ev[-1])
    t8 = sum(ev[2 * i].elapsed_time(ev[2 * i + 1]) for i in range(args.steps)) / args.steps
    t4 = sum(ev[2 * i + 1].elapsed_time(ev[2 * i + 2]) for i in range(args.steps)) / args.steps
    total_ms = max_over_ranks(total_ms, dist)
    ms_step = total_ms / args.steps
    ops_step = st8.ops + st4.ops
    value = world * ops_step / (ms_step * 1e-3) / 1e12

    # ---- roofline of the dominant kernel: the W8A8 tcgen05 GEMM (S2+S3), launched alone for the
    # same 96 layers on already-quantised activations, timed with CUDA events on its stream.
    xq = {}
    for K in {s["K"] for s in st8.specs}:
        X = next((s["in"] for s in st8.specs if s["K"] == K and s["in"] is not None), None)
        if X is None:
            X = st8.specs[2]["out"]               # the MLP hidden state feeds the down-projection
        xq[K] = aria.aria_quantize_act_int8(X)

    def gemm_only():
        for s in st8.specs:
            q, sx = xq[s["K"]]
            aria.aria_linear_w8a8_q(q, sx, s["wq"], s["w_scale"], s["bias"], s["act"], aria.BF16, out=s["out"])
    gemm_only()
    torch.cuda.synchronize()
    gg = torch.cuda.CUDAGraph()
    with torch.cuda.graph(gg):
        gemm_only()
    for _ in range(3):
        gg.replay()
    g_ms = time_region(torch, gg.replay, args.steps)
    n_l = len(st8.specs)
    dur = g_ms * 1e-3 / n_l
    ach = (st8.ops / n_l) / dur / 1e12
    region_s = args.steps * ms_step * 1e-3
    burst = region_s < BURST_REGION_S
    tp = None
    if world == 1:
        try:
            tp = tensor_peaks(aria)
        except Exception as ex:                  # noqa: BLE001
            log(f"[bench] tensor peak measurement failed: {ex!r}")
    # W8A8 GEMM against the MEASURED int8 tensor peak (tcgen05 kind::i8 issue loop on this device); the
    # bf16-derived figures stay beside it as context
    if tp and not burst:
        tensor_peaks_sustained(aria, tp)
    if tp:
        peak8 = tp["int8"]["burst" if burst else "sustained"]
        src8 = f"measured: aria_tensor_peak kind::i8 issue loop, {'burst' if burst else 'sustained'}"
    else:
        peak8 = (pk["bf16_burst"] if burst else pk["bf16_sustained"]) * NOMINAL_INT8_OVER_BF16
        src8 = f"{pk['source']} bf16 {'burst' if burst else 'sustained'} x {NOMINAL_INT8_OVER_BF16:g} (nominal int8/bf16)"
    roofline_w8a8 = {"kernel": "w8a8_gemm_kernel (tcgen05 kind::i8 + fused epilogue), 96 launches on pre-quantised activations",
                "bound": "tensor", "achieved": ach, "peak": peak8, "unit": "TOP/s", "frac": ach / peak8,
                "peak_source": src8,
                "frac_of_2x_bf16_burst": ach / (pk["bf16_burst"] * NOMINAL_INT8_OVER_BF16),
                "frac_of_nominal_4500": ach / 4500.0, "avg_launch_us": dur * 1e6, "launches": n_l,
                "traffic": profile_traffic(W8A8_TRAFFIC_SRC), "traffic_unit": f"bytes/launch, mean of the launches in {W8A8_TRAFFIC_SRC} (ncu, shared-input step: X is L2-resident there)"}

    # ---- roofline of the DOMINANT kernel of the step: w4a16_gemm_kernel.  The W4A16 half of the step is 96
    # launches of that kernel and nothing else, so its average launch duration is t4 / 96 from the CUDA
    # events recorded around every replay in the timed region above.  Peak: the driver-measured cuBLAS bf16
    # figure (MEASURED_PEAKS.json) -- the BURST one while the timed region is under a second.
    dur4 = t4 * 1e-3 / n_l
    ach4 = (st4.ops / n_l) / dur4 / 1e12
    peak4 = pk["bf16_burst"] if burst else pk["bf16_sustained"]
    roofline = {"kernel": "w4a16_gemm_kernel (on-chip int4 dequant -> tcgen05 kind::f16 bf16, fused epilogue)",
                "bound": "tensor", "achieved": ach4, "peak": peak4, "unit": "TFLOP/s",
                "frac": ach4 / peak4,
                "peak_source": f"{pk['source']} bf16 {'burst' if burst else 'sustained'} (timed region {region_s:.2f} s)",
                "frac_of_sustained": ach4 / pk["bf16_sustained"], "frac_of_nominal_2250": ach4 / 2250.0,
                "frac_of_issue_loop_peak": (ach4 / tp["bf16"]["burst" if burst else "sustained"]) if tp else None,
                "avg_launch_us": dur4 * 1e6, "launches": n_l, "share_of_step": t4 / (t8 + t4),
                "algorithmic_flops_per_launch": st4.ops / n_l,
                "traffic": profile_traffic(W4A16_TRAFFIC_SRC), "traffic_unit": f"bytes/launch, mean of the launches in {W4A16_TRAFFIC_SRC} (ncu, shared-input step: X is L2-resident there)"}

    # ---- e2e: same step through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    try:
        e2e = run_e2e(torch, aria, st8, st4, M, min(args.steps, 5), world)
    except Exception as ex:                      # noqa: BLE001
        log(f"[bench] e2e failed: {ex!r}")
    clocks = sampler.stop() if sampler else None

    if rank != 0:
        return
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        ops, t, cores = oracle_sample(1024)
        cpu = {"value": ops / t / 1e12, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"block 0's 4 linears at 1024 of the 2048 tokens, both modes, {t:.1f} s"}
    ops8, ops4 = st8.ops, st4.ops
    table = small = nxt = hbm = None
    if world == 1 and not args.no_per_linear:
        table = per_linear_table(torch, aria, inputs, pk)
        small = small_m_stream(torch, aria, inputs, pk)
        try:
            hbm = hbm_passes(torch, aria, inputs, pk)
        except Exception as ex:                  # noqa: BLE001
            log(f"[bench] hbm_passes failed: {ex!r}")
        try:
            nxt = next_rows(torch, aria, inputs, pk)
        except Exception as ex:                  # noqa: BLE001
            log(f"[bench] next_rows failed: {ex!r}")
    # Reading R14 says every linear reads its OWN N(0,1) input.  The headline step above shares one input buffer per
    # distinct K (three buffers, L2-resident); here the same step with 72 distinct external inputs (453 MB, HBM-cold
    # on every replay), timed the same way.  Built after the headline so its memory and time cannot disturb it.
    distinct = None
    if world == 1 and not args.no_per_linear:
        try:
            d8 = LinearStack(aria.W8A8, M=M, shared_inputs=False)
            d4 = LinearStack(aria.W4A16, M=M, shared_inputs=False)
            d8.capture()
            d4.capture()
            for _ in range(3):
                d8.replay()
                d4.replay()
            m8 = time_region(torch, d8.replay, args.steps)
            m4 = time_region(torch, d4.replay, args.steps)
            distinct = {"ms_w8a8": m8, "ms_w4a16": m4, "ms_per_step": m8 + m4,
                        "value": (ops8 + ops4) / ((m8 + m4) * 1e-3) / 1e12, "unit": UNIT,
                        "ratio_to_shared_inputs": (m8 + m4) / (t8 + t4),
                        "what": "the C5 step with one N(0,1) input buffer per linear (72 external inputs, reading R14) "
                                "instead of one per distinct K; each half timed over its own replays"}
            del d8, d4
            torch.cuda.empty_cache()
        except Exception as ex:                  # noqa: BLE001
            log(f"[bench] distinct-input step failed: {ex!r}")
    # last (they heat the part): the long replay of the same step, then the sustained tensor peaks
    sustained = None
    if world == 1 and not args.no_sustained:
        sustained = sustained_record(torch, step, ops_step, ms_step, local)
        if tp and "sustained" not in tp["int8"]:
            tensor_peaks_sustained(aria, tp)
        if tp:
            sustained["int8_sustained_peak"] = tp["int8"]["sustained"]
            sustained["bf16_sustained_issue_loop_peak"] = tp["bf16"]["sustained"]
    # `value` sums int8 operations and effective bf16 flops of the two halves of the step (the driver's single
    # number); the per-mode figures that BASELINE.json's metric names come FIRST in the line
    line = {
        "metric": METRIC, "value": value, "unit": UNIT,
        "modes": {"w8a8": {"ms": t8, "tops": ops8 / (t8 * 1e-3) / 1e12,
                           "frac_of_int8_peak": ops8 / (t8 * 1e-3) / 1e12 / peak8, "peak": peak8, "peak_source": src8},
                  "w4a16": {"ms": t4, "eff_tflops": ops4 / (t4 * 1e-3) / 1e12,
                            "frac_of_bf16_peak": ops4 / (t4 * 1e-3) / 1e12 / peak4, "peak": peak4}},
        "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "int8xint8->int32 / int4->bf16xbf16->f32",
        "data": "synthetic",
        "config": {"workload": WORKLOAD, "tokens": M, "layers": n_l, "l2": "weights 680 MB + 382 MB per step exceed the 126 MB L2",
                   "multi_gpu": "replicas only"},
        "roofline": roofline, "roofline_w8a8_gemm": roofline_w8a8, "tensor_peaks": tp, "sustained": sustained,
        "cpu_baseline": cpu, "e2e": e2e,
        # kernels of this library launched inside the timed region: per step 96 W4A16 GEMMs + 96 W8A8 GEMMs + the
        # stand-alone S1 passes the W8A8 chain keeps (layer 0, and the rounding pass of every chained layer)
        "gpu_launches": args.steps * (2 * n_l + 1 + sum(1 for s in st8.specs if s["in"] is None)), "clocks": clocks, "per_linear": table,
        "small_m": small, "hbm_passes": hbm, "next_rows": nxt, "distinct_inputs": distinct,
    }
    log("[bench] " + json.dumps({k: line[k] for k in ("value", "ms_per_step", "modes", "roofline", "roofline_w8a8_gemm",
                                                       "tensor_peaks", "sustained")}))
    print(json.dumps(line))


def run_e2e(torch, aria, st8, st4, M, steps, world):
    """aria_denoiser_linears_host: every layer's input comes from pinned host memory and every
    layer's output goes back to pinned host memory inside the timed region."""
    host_in = {}
    outs = {}
    results = {}
    h2d = d2h = 0
    for st, tag in ((st8, "w8a8"), (st4, "w4a16")):
        specs = []
        for s in st.specs:
            K, N = s["K"], s["N"]
            if s["in"] is not None and K not in host_in:
                host_in[K] = s["in"].cpu().pin_memory()
            if N not in outs:
                outs[N] = torch.empty((M, N), dtype=torch.bfloat16).pin_memory()
            d = dict(s)
            d["in"] = host_in[K] if s["in"] is not None else None
            d["out"] = outs[N]
            specs.append(d)
            h2d += (M * K * 2) if s["in"] is not None else 0
            d2h += M * N * 2
        layers = aria.make_layers(specs)
        maxK = max(s["K"] for s in specs)
        maxN = max(s["N"] for s in specs)
        ws = aria.workspace(aria.aria_workspace_bytes_host(M, maxK, maxN, st.mode, aria.BF16))
        results[tag] = (layers, ws, st.mode, specs)
    def step():
        for tag in ("w8a8", "w4a16"):
            layers, ws, mode, _ = results[tag]
            aria.aria_denoiser_linears_host(layers, M, mode, aria.BF16, ws)
    step()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    ms = max(e0.elapsed_time(e1), (time.perf_counter() - t0) * 1e3) / steps
    ops = st8.ops + st4.ops
    return {"value": world * ops / (ms * 1e-3) / 1e12, "unit": UNIT, "ms_per_step": ms, "steps": steps,
            "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
            "api": "aria_denoiser_linears_host (pinned host in/out per layer, weights resident)"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-per-linear", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sustained", action="store_true")
    ap.add_argument("--per-linear-only", action="store_true",
                    help="only the per-linear table C2/C3/C4 (used for ncu captures)")
    ap.add_argument("--small-m-only", action="store_true",
                    help="only the M=32 W4A16 stream-kernel section (used for ncu captures)")
    ap.add_argument("--next-rows-only", action="store_true",
                    help="only the SURVEY S8(f) rows: W8A16 stack, attention, norm+S1, chained blocks, 8-step clip")
    args = ap.parse_args()
    if args.next_rows_only:
        import torch
        from paper_2607_08526_b200 import binding as aria
        from paper_2607_08526_b200 import inputs
        aria.lib()
        print(json.dumps({"next_rows": next_rows(torch, aria, inputs, peaks()),
                          "hbm_passes": hbm_passes(torch, aria, inputs, peaks())}))
        return
    if args.per_linear_only:
        import torch
        from paper_2607_08526_b200 import binding as aria
        from paper_2607_08526_b200 import inputs
        aria.lib()
        print(json.dumps({"per_linear": per_linear_table(torch, aria, inputs, peaks())}))
        return
    if args.small_m_only:
        import torch
        from paper_2607_08526_b200 import binding as aria
        from paper_2607_08526_b200 import inputs
        aria.lib()
        print(json.dumps({"small_m": small_m_stream(torch, aria, inputs, peaks(), iters=max(args.steps, 3))}))
        return
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
