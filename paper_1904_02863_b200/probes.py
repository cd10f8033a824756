"""Measurement aids (NOT the product path): ctypes loader of ``csrc/libgwprobe.so`` (include/gwprobe.h).

    python -m paper_1904_02863_b200.probes

prints the fp64 pipe rate of this GPU by operand pattern and the pure-store / pure-load HBM bandwidth -- the measured
roofline denominators that MEASURED_PEAKS.json lacks.  ``bench.py`` calls the same functions.
"""
from __future__ import annotations

import ctypes
import json
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
EXPORTS = ("gw_probe_fp64_fma_rate", "gw_probe_sm_clock", "gw_probe_launch_floor", "gw_probe_store_bandwidth",
           "gw_probe_load_bandwidth")
MODES = {0: "fma(v, imm, imm): one register operand", 1: "fma(a, b, v): three distinct register operands",
         2: "fma(a, m, v): three register operands, one shared by consecutive instructions",
         3: "mma.sync m8n8k4 f64 (DMMA)",
         4: "mode 0 plus 8 independent integer instructions per 8 DFMA (do other pipes issue for free?)",
         5: "mode 0 plus 16 independent integer instructions per 8 DFMA"}
_lib = None


def lib_path() -> str:
    return os.path.join(_HERE, "csrc", "libgwprobe.so")


def load_library():
    global _lib
    if _lib is None:
        path = lib_path()
        if not os.path.exists(path):
            raise RuntimeError(f"{path} is missing: build it with `python paper_1904_02863_b200/csrc/build.py`")
        lib = ctypes.CDLL(path)
        vp, i64, ci, dp = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.POINTER(ctypes.c_double)
        lib.gw_probe_fp64_fma_rate.argtypes = [ci, ci, dp, dp, vp]
        lib.gw_probe_sm_clock.argtypes = [dp, vp]
        lib.gw_probe_launch_floor.argtypes = [ci, ci, ci, ci, dp, vp]
        lib.gw_probe_store_bandwidth.argtypes = [i64, ci, dp, dp, vp]
        lib.gw_probe_load_bandwidth.argtypes = [i64, ci, dp, dp, vp]
        for n in EXPORTS:
            getattr(lib, n).restype = ci
        _lib = lib
    return _lib


def _stream_ptr(stream) -> int:
    import torch
    return int((stream or torch.cuda.current_stream()).cuda_stream)


def fp64_fma_rate(n_iter: int = 4096, mode: int = 0, stream=None):
    """(fp64 FMA/s, elapsed ms) of the register-resident probe kernel; mode: see gwprobe.h."""
    rate, ms = ctypes.c_double(), ctypes.c_double()
    rc = load_library().gw_probe_fp64_fma_rate(int(n_iter), int(mode), ctypes.byref(rate), ctypes.byref(ms),
                                               _stream_ptr(stream))
    if rc != 0:
        raise RuntimeError(f"gw_probe_fp64_fma_rate: error {rc}")
    return rate.value, ms.value


def sm_clock_mhz(stream=None) -> float:
    """The SM clock actually running (MHz, median over SMs), measured right behind whatever the stream just ran."""
    mhz = ctypes.c_double()
    rc = load_library().gw_probe_sm_clock(ctypes.byref(mhz), _stream_ptr(stream))
    if rc != 0:
        raise RuntimeError(f"gw_probe_sm_clock: error {rc}")
    return mhz.value


def launch_floor_ms(grid: int = 148, block: int = 256, dyn_smem_bytes: int = 0, n_rep: int = 50, stream=None) -> float:
    """Median event-to-event time (ms) of an empty kernel with this launch shape: what a kernel-alone timing includes."""
    ms = ctypes.c_double()
    rc = load_library().gw_probe_launch_floor(int(grid), int(block), int(dyn_smem_bytes), int(n_rep), ctypes.byref(ms),
                                              _stream_ptr(stream))
    if rc != 0:
        raise RuntimeError(f"gw_probe_launch_floor: error {rc}")
    return ms.value


def _bandwidth(fn, n_bytes, n_rep, stream):
    gbs, ms = ctypes.c_double(), ctypes.c_double()
    rc = fn(int(n_bytes), int(n_rep), ctypes.byref(gbs), ctypes.byref(ms), _stream_ptr(stream))
    if rc != 0:
        raise RuntimeError(f"bandwidth probe: error {rc}")
    return gbs.value, ms.value


def store_bandwidth(n_bytes: int = 2 << 30, n_rep: int = 10, stream=None):
    """(GB/s, best ms): pure-store stream of n_bytes, 16-byte streaming stores, best of n_rep."""
    return _bandwidth(load_library().gw_probe_store_bandwidth, n_bytes, n_rep, stream)


def load_bandwidth(n_bytes: int = 2 << 30, n_rep: int = 10, stream=None):
    """(GB/s, best ms): pure-load stream of n_bytes, 16-byte streaming loads, best of n_rep."""
    return _bandwidth(load_library().gw_probe_load_bandwidth, n_bytes, n_rep, stream)


def main():
    fp64_fma_rate(1 << 13, 0)                             # clock ramp
    out = {}
    for mode, what in MODES.items():
        best = max(fp64_fma_rate(1 << 13, mode)[0] for _ in range(3))
        out[f"fp64_mode_{mode}"] = {"pattern": what, "fma_per_s": best, "tflops": 2 * best / 1e12}
        print(f"mode {mode}: {best / 1e12:6.2f} T-FMA/s = {2 * best / 1e12:6.2f} TFLOP/s   {what}")
    out["sm_clock_after_fp64_probe_mhz"] = sm_clock_mhz()
    print(f"SM clock right after the fp64 probes: {out['sm_clock_after_fp64_probe_mhz']:.0f} MHz")
    out["launch_floor_us"] = 1e3 * launch_floor_ms()
    print(f"empty kernel between two events: {out['launch_floor_us']:.2f} us")
    for name, fn in (("store", store_bandwidth), ("load", load_bandwidth)):
        gbs, ms = fn()
        out[f"hbm_{name}_GBps"] = gbs
        print(f"pure {name:5s}: {gbs:7.1f} GB/s ({ms:.3f} ms for 2 GiB)")
    print(json.dumps(out))


if __name__ == "__main__":
    main()
