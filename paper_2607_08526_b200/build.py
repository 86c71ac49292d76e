"""Build libaria_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2607_08526_b200.build [--force] [--verbose] [--debug]

--debug builds libaria_b200_dbg.so with -DARIA_DEBUG instead: the only build in which the library reads
environment switches (ARIA_W8_PLAN, ARIA_WS_DBG, ...) and exports the aria_debug_* role-timestamp
hooks.  The product library has none of them; nothing in the package loads the debug build.

The library links the CUDA runtime statically and resolves the one driver symbol it needs
(cuTensorMapEncodeTiled) at run time, so it loads on a machine without libcuda.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libaria_b200.so")
SOURCES = ["api.cu", "quant.cu", "tensormap.cu", "gemm_w8a8.cu", "gemm_w4a16.cu", "w4a16_stream.cu", "peak.cu", "steer.cu", "norm.cu", "attention.cu", "static_ws.cu"]
HEADERS = ["internal.cuh", "ptx.cuh", "quant_dev.cuh", os.path.join("..", "..", "include", "aria.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
         "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden", "--expt-relaxed-constexpr"]


def _stale(lib: str = LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, debug: bool = False) -> str:
    lib = LIB.replace(".so", "_dbg.so") if debug else LIB
    if not force and not _stale(lib):
        return lib
    objs = []
    procs = []
    bdir = os.path.join(HERE, "build", "dbg" if debug else "rel")
    os.makedirs(bdir, exist_ok=True)
    for s in SOURCES:
        obj = os.path.join(bdir, s.replace(".cu", ".o"))
        cmd = [NVCC, *FLAGS, *(["-DARIA_DEBUG"] if debug else []), "-c", os.path.join(CSRC, s), "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas")
            cmd.insert(2, "-v")
        procs.append((s, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT)))
        objs.append(obj)
    failed = False
    for s, p in procs:
        out = p.communicate()[0].decode()
        if p.returncode != 0 or verbose:
            sys.stderr.write(f"--- {s}\n{out}\n")
        failed |= p.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed")
    subprocess.check_call([NVCC, "-shared", "-o", lib, *objs, "-cudart", "static"])
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, debug="--debug" in sys.argv))
