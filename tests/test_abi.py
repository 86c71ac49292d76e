"""The C-ABI library builds, loads without a GPU, and exports every symbol include/aria.h declares."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "aria.h")).read()
    return sorted(set(re.findall(r"ARIA_API\s+[\w\s\*]+?\b(aria_\w+)\s*\(", src)))


def test_header_declares_the_north_star_entry_points():
    names = _declared()
    for need in ("aria_quantize_weights_int8", "aria_quantize_weights_int4", "aria_quantize_act_int8",
                 "aria_linear_w8a8", "aria_linear_w4a16", "aria_denoiser_linears"):
        assert need in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2607_08526_b200 import binding, build
    path = build.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    names = _declared()
    assert len(names) >= 12
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(binding.EXPORTS) == names
    L = binding.lib()
    assert b"sm_100a" in L.aria_version()
    assert L.aria_status_string(0) == b"ok"
    assert L.aria_status_string(-5).startswith(b"device is not sm_100")


def test_validation_errors_need_no_gpu():
    # argument validation happens before any CUDA call
    from paper_2607_08526_b200 import binding
    L = binding.lib()
    assert L.aria_quantize_act_int8(None, 0, 4, 32, None, None, None) == -1           # NULL
    buf = (ctypes.c_char * 4096)()
    p = ctypes.addressof(buf)
    p16 = (p + 15) // 16 * 16
    assert L.aria_quantize_act_int8(p16, 0, 4, 33, p16, p16, None) == -2               # K % 32
    assert L.aria_quantize_act_int8(p16, 7, 4, 32, p16, p16, None) == -4               # dtype
    assert L.aria_quantize_act_int8(p16 + 4, 0, 4, 32, p16, p16, None) == -3           # alignment
    assert L.aria_quantize_weights_int4(p16, 0, 4, 64, 16, p16, p16, None) == -2       # group != 32
    assert L.aria_linear_w8a8(p16, 1, 4, 64, p16, p16, 12, None, 0, 0, p16, 1, p16, 1 << 20, None) == -2  # N % 8
    assert L.aria_linear_w8a8(p16, 1, 4, 64, p16, p16, 16, None, 0, 0, p16, 1, p16, 16, None) == -6       # ws too small
    assert L.aria_workspace_bytes(0, 64, 64, 0) == 0
    assert L.aria_workspace_bytes(128, 1536, 4608, 0) >= 128 * 1536 + 128 * 4
    # round-2 entry points
    st = None
    assert L.aria_linear_w8a16(p16, 4, 64, p16, p16, 12, None, 0, p16, 1, None, 0, st) == -2             # N % 8
    assert L.aria_linear_w8a16(None, 4, 64, p16, p16, 16, None, 0, p16, 1, None, 0, st) == -1            # NULL
    assert L.aria_norm_quantize_act_int8(p16, 1, 4, 48, p16, None, 0, 1e-5, None, p16, p16, st) == -2    # K % 32
    assert L.aria_norm_quantize_act_int8(p16, 1, 4, 64, None, None, 0, 1e-5, None, p16, p16, st) == -1   # gamma NULL
    assert L.aria_norm_quantize_act_int8(p16, 1, 4, 64, p16, None, 5, 1e-5, None, p16, p16, st) == -4    # unknown norm
    assert L.aria_norm_quantize_act_int8(p16, 1, 4, 64, p16, None, 0, -1.0, None, p16, p16, st) == -2    # eps < 0
    assert L.aria_attention(p16, 1, 128, 2, 32, 0.125, p16, None, st) == -2                              # head_dim != 64
    assert L.aria_attention(p16, 1, 128, 2, 64, -1.0, p16, None, st) == -2                               # scale <= 0
    assert L.aria_attention(p16, 0, 128, 2, 64, 0.125, p16, None, st) == -2                              # B <= 0
    assert L.aria_attention(p16 + 8, 1, 128, 2, 64, 0.125, p16, None, st) == -3                          # alignment
    assert L.aria_round_act_int8(p16, 1, 4, 64, None, 0, p16, p16, st) == -1                             # absmax NULL
    assert L.aria_steer(p16, 1, 4, 12, p16, p16, 1.0, 0, st) == -2                                       # D % 8
    assert L.aria_steer(p16, 1, 4, 16, p16, p16, 1.0, 9, st) == -4                                       # unknown op
    assert L.aria_tensor_peak(3, 1, 16, 0.0, None, st) == -1


def test_tile_plans_reach_every_compiled_variant_on_148_sms():
    """Host logic: the launchers' plans for a 148-SM device.  The GPU tests run exactly these shapes, so
    every compiled kernel instantiation is exercised (tests/test_gpu_w8a8.py, tests/test_gpu_w4a16.py)."""
    from paper_2607_08526_b200 import binding as aria
    w8 = {(64, 256): (64, 1), (128, 18944): (128, 1), (128, 28416): (192, 1), (100, 37888): (256, 1),
          (512, 1536): (128, 2), (2048, 1536): (192, 2), (1000, 4608): (256, 2),
          (4096, 6144): (256, 2), (2048, 4608): (256, 2)}
    for (M, N), want in w8.items():
        assert aria.aria_w8a8_tile_plan(M, N, 148) == want, (M, N)
    w4 = {(32, 256, 1536): 32, (64, 18944, 256): 64, (512, 1536, 6144): 128, (2000, 1536, 256): 192,
          (1024, 4608, 256): 256, (2048, 4608, 1536): 256, (2048, 1536, 1536): 192}
    for (M, N, K), tt in w4.items():
        assert aria.aria_w4a16_tile_plan(M, N, K, 148)[0] == tt, (M, N, K)
    assert aria.aria_w4a16_tile_plan(512, 1536, 6144, 148)[1] > 1          # split-K at small M
    assert aria.aria_w4a16_tile_plan(4096, 6144, 1536, 148)[1] == 1


def test_product_library_reads_no_environment_variable_and_exports_no_debug_hook():
    """VERDICT r1 / ADVICE: env switches and aria_debug_* exist only in -DARIA_DEBUG builds."""
    import subprocess
    from paper_2607_08526_b200 import build
    path = build.build()
    syms = subprocess.run(["nm", "-D", "--defined-only", path], capture_output=True, text=True).stdout
    exported = sorted(l.split()[-1] for l in syms.splitlines() if " T " in l)
    assert exported == _declared(), set(exported) ^ set(_declared())
    undefined = subprocess.run(["nm", "-D", "--undefined-only", path], capture_output=True, text=True).stdout
    assert "getenv" not in undefined.split()


def test_bench_reads_its_ncu_traffic_figures_from_the_committed_profiles():
    """bench.py's `roofline.traffic` is parsed from the profiles/ summaries it cites (no typed-in constants): the
    files exist, parse, and give the per-launch DRAM bytes their own summary line states."""
    import bench
    w4 = bench.profile_traffic(bench.W4A16_TRAFFIC_SRC)
    w8 = bench.profile_traffic(bench.W8A8_TRAFFIC_SRC)
    assert w4 is not None and abs(w4 - 15.06e6) < 0.02e6      # "mean 15.06" MB in profiles/r2_w4a16_full.md
    assert w8 is not None and abs(w8 - 17.39e6) < 0.02e6      # "mean 17.39" MB in profiles/r2_w8a8_full.md
    assert bench.profile_traffic("profiles/does_not_exist.md") is None
