#!/usr/bin/env python3
"""Build the CUDA libraries with nvcc for sm_100a, in-tree:

    csrc/libgwlnl.so    the product library: C-ABI of include/gwlnl.h, include/gwlnl_tuning.h, include/gwpop.h
    csrc/libgwprobe.so  measurement aids only (include/gwprobe.h): fp64-rate and HBM store / load bandwidth probes
    csrc/libgwlnl_timeline.so  (on demand, build_timeline) the product sources compiled with -DGW_TIMELINE: the fused
                        kernel's CTAs stamp a timeline (gw_kernels.cu); a diagnostic aid for timeline.py, never loaded by
                        the product path

    python paper_1904_02863_b200/csrc/build.py [--force] [--verbose]

Cross-compiles without a GPU.  No torch headers are involved: the libraries are plain CUDA runtime + C-ABI.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
INC = os.path.join(ROOT, "include")
SOURCES = ["gw_api.cu", "gw_kernels.cu", "gw_pop.cu"]
HEADERS = ["gw_internal.h", "gw_math.cuh", os.path.join(INC, "gwlnl.h"), os.path.join(INC, "gwlnl_tuning.h"),
           os.path.join(INC, "gwpop.h")]
LIB = os.path.join(HERE, "libgwlnl.so")
PROBE_SOURCES = ["gw_probe.cu"]
PROBE_HEADERS = [os.path.join(INC, "gwprobe.h")]
PROBE_LIB = os.path.join(HERE, "libgwprobe.so")
TIMELINE_LIB = os.path.join(HERE, "libgwlnl_timeline.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
         "--fmad=false",            # every FMA in the kernels is explicit; no silent contraction elsewhere
         "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def _up_to_date(lib, sources, headers) -> bool:
    if not os.path.exists(lib):
        return False
    t = os.path.getmtime(lib)
    deps = [os.path.join(HERE, s) for s in sources] + [h if os.path.isabs(h) else os.path.join(HERE, h) for h in headers]
    deps.append(os.path.abspath(__file__))
    return all(os.path.getmtime(d) <= t for d in deps)


def up_to_date() -> bool:
    return _up_to_date(LIB, SOURCES, HEADERS)


def build(force: bool = False, verbose: bool = False, defines=(), out: str = LIB) -> str:
    """The product library.  defines: e.g. ("GW_THREADS=128",) for a tuning variant written to `out` (the default
    build has none)."""
    if not force and out == LIB and not defines and up_to_date():
        return LIB
    cmd = [NVCC] + FLAGS + [f"-D{d}" for d in defines] + (["-Xptxas", "-v"] if verbose else []) + ["-o", out] + SOURCES
    subprocess.run(cmd, check=True, cwd=HERE)
    return out


def build_probe(force: bool = False) -> str:
    """The measurement-aid library (bench.py and the probes module load it; the product path does not)."""
    if not force and _up_to_date(PROBE_LIB, PROBE_SOURCES, PROBE_HEADERS):
        return PROBE_LIB
    subprocess.run([NVCC] + FLAGS + ["-o", PROBE_LIB] + PROBE_SOURCES, check=True, cwd=HERE)
    return PROBE_LIB


def build_timeline(force: bool = False) -> str:
    """The diagnostic variant of the product library with the per-CTA timeline stamps (timeline.py loads it)."""
    if not force and _up_to_date(TIMELINE_LIB, SOURCES, HEADERS):
        return TIMELINE_LIB
    return build(force=True, defines=("GW_TIMELINE",), out=TIMELINE_LIB)


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
    print(build_probe(force="--force" in sys.argv))
