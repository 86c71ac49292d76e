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
