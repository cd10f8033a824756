#!/usr/bin/env python3
"""Build csrc/libgwlnl.so (the C-ABI library of include/gwlnl.h) with nvcc for sm_100a, in-tree.

    python paper_1904_02863_b200/csrc/build.py [--force] [--verbose]

Cross-compiles without a GPU.  No torch headers are involved: the library is plain CUDA runtime + C-ABI.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
SOURCES = ["gw_api.cu", "gw_kernels.cu"]
HEADERS = ["gw_internal.h", "gw_math.cuh", os.path.join(ROOT, "include", "gwlnl.h")]
LIB = os.path.join(HERE, "libgwlnl.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
         "--fmad=false",            # every FMA in the kernels is explicit; no silent contraction elsewhere
         "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def up_to_date() -> bool:
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    deps = [os.path.join(HERE, s) for s in SOURCES] + [h if os.path.isabs(h) else os.path.join(HERE, h) for h in HEADERS]
    deps.append(os.path.abspath(__file__))
    return all(os.path.getmtime(d) <= t for d in deps)


def build(force: bool = False, verbose: bool = False, defines=(), out: str = LIB) -> str:
    """defines: e.g. ("GW_THREADS=128",) for a tuning variant written to `out` (the default build has none)."""
    if not force and out == LIB and not defines and up_to_date():
        return LIB
    cmd = [NVCC] + FLAGS + [f"-D{d}" for d in defines] + (["-Xptxas", "-v"] if verbose else []) + ["-o", out] + SOURCES
    subprocess.run(cmd, check=True, cwd=HERE)
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
