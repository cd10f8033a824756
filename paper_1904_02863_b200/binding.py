"""Thin Python binding of the C-ABI library ``csrc/libgwlnl.so`` (include/gwlnl.h).

Argument marshalling only: every step of the path runs in the CUDA kernels.  PyTorch appears for device
buffers (``tensor.data_ptr()``) and streams (``torch.cuda.current_stream().cuda_stream``) and nothing else.
There is no CPU fallback: if the extension is missing or cannot be loaded, importing this module's
``load_library`` raises ``GwError``.  Nothing here imports ``oracle``.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
NPARAM = 11
MAX_DET = 8
DET_ROW = 13   # inputs.py detector row: kind, vertex[3], xarm[3], yarm[3], fplus, fcross, dt

GW_OK, GW_ERR_INVALID_ARG, GW_ERR_ALLOC, GW_ERR_CUDA, GW_ERR_ARCH = 0, -1, -2, -3, -4

# every symbol include/gwlnl.h declares (tests/test_abi.py checks the library exports each)
EXPORTS = (
    "gw_ctx_create", "gw_ctx_reserve", "gw_waveform_batch", "gw_lnl_batch", "gw_lnl_batch_host",
    "gw_waveform_batch_host", "gw_ctx_destroy", "gw_ctx_info", "gw_ctx_n_param", "gw_ctx_plan", "gw_ctx_norms",
    "gw_ctx_launch_count", "gw_strerror", "gw_last_cuda_error", "gw_abi_version",
)
# include/gwlnl_tuning.h: testing / tuning aids exported by the same library, outside the product boundary
TUNING_EXPORTS = ("gw_ctx_force_plan", "gw_ctx_force_grid", "gw_ctx_cluster_finish", "gw_ctx_host_graph", "gw_ctx_boundary_bins", "gw_ctx_plan_boundary_bins", "gw_plan_cta_segments", "gw_ctx_kernel_timing",
                  "gw_ctx_last_kernel_ms")


class GwError(RuntimeError):
    def __init__(self, code: int, where: str, detail: str = ""):
        self.code = code
        super().__init__(f"{where}: {detail or code}")


class gw_detector(ctypes.Structure):
    _fields_ = [("kind", ctypes.c_int), ("vertex_m", ctypes.c_double * 3), ("xarm", ctypes.c_double * 3),
                ("yarm", ctypes.c_double * 3), ("fplus", ctypes.c_double), ("fcross", ctypes.c_double),
                ("dt_s", ctypes.c_double)]


class gw_options(ctypes.Structure):
    _fields_ = [("spin_order", ctypes.c_int), ("isco_cut", ctypes.c_int), ("max_batch", ctypes.c_int64),
                ("phase_marginal", ctypes.c_int), ("tidal_order", ctypes.c_int)]


def lib_path() -> str:
    """csrc/libgwlnl.so, built in-tree by csrc/build.py (no environment-variable dispatch)."""
    return os.path.join(_HERE, "csrc", "libgwlnl.so")


_lib = None
_lib_file = None


def load_library(variant_path: Optional[str] = None):
    """dlopen csrc/libgwlnl.so and declare the prototypes.  Fails loudly; never falls back.

    ``variant_path`` is for the diagnostic tools of this package only (timeline.py: the same sources built with
    -DGW_TIMELINE): it must be given on the FIRST call of the process, before anything else has loaded the library; a
    process uses one library throughout."""
    global _lib, _lib_file
    if _lib is not None:
        if variant_path is not None and os.path.abspath(variant_path) != _lib_file:
            raise GwError(GW_ERR_INVALID_ARG, "load_library", f"{_lib_file} is already loaded in this process")
        return _lib
    path = os.path.abspath(variant_path) if variant_path is not None else lib_path()
    if not os.path.exists(path):
        raise GwError(GW_ERR_CUDA, "load_library",
                      f"{path} is missing: build it with `python paper_1904_02863_b200/csrc/build.py` "
                      "(there is no CPU fallback)")
    lib = ctypes.CDLL(path)
    vp, i64, ci, dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double
    P = ctypes.POINTER
    lib.gw_ctx_create.argtypes = [P(vp), i64, vp, ci, vp, vp, P(gw_detector), dbl, P(gw_options), vp]
    lib.gw_ctx_reserve.argtypes = [vp, i64]
    lib.gw_waveform_batch.argtypes = [vp, i64, vp, vp, vp]
    lib.gw_lnl_batch.argtypes = [vp, i64, vp, vp, vp, vp]
    lib.gw_lnl_batch_host.argtypes = [vp, i64, vp, vp, vp, vp]
    lib.gw_waveform_batch_host.argtypes = [vp, i64, vp, vp, vp]
    lib.gw_ctx_destroy.argtypes = [vp]
    lib.gw_ctx_info.argtypes = [vp, P(i64), P(ci), P(dbl), P(i64)]
    lib.gw_ctx_n_param.argtypes = [vp]
    lib.gw_ctx_plan.argtypes = [vp, i64, P(ci), P(ci), P(ci), P(i64)]
    lib.gw_ctx_norms.argtypes = [vp, P(dbl)]
    lib.gw_ctx_launch_count.argtypes = [vp]
    lib.gw_ctx_launch_count.restype = i64
    lib.gw_ctx_force_plan.argtypes = [vp, ci, ci]
    lib.gw_ctx_force_grid.argtypes = [vp, ci, i64]
    lib.gw_ctx_cluster_finish.argtypes = [vp, ci]
    lib.gw_ctx_host_graph.argtypes = [vp, ci]
    lib.gw_plan_cta_segments.argtypes = [i64, i64, i64, i64, i64, ci, P(i64)]
    lib.gw_ctx_boundary_bins.argtypes = [vp, ci]
    lib.gw_ctx_plan_boundary_bins.argtypes = [vp, i64, P(ci)]
    lib.gw_ctx_kernel_timing.argtypes = [vp, ci]
    lib.gw_ctx_last_kernel_ms.argtypes = [vp, P(dbl), P(dbl)]
    lib.gw_strerror.argtypes = [ci]
    lib.gw_strerror.restype = ctypes.c_char_p
    lib.gw_last_cuda_error.argtypes = [vp]
    lib.gw_abi_version.argtypes = []
    for name in EXPORTS + TUNING_EXPORTS:
        if name not in ("gw_strerror", "gw_ctx_launch_count"):
            getattr(lib, name).restype = ci
    _lib, _lib_file = lib, path
    return lib


def _check(rc: int, where: str, ctx=None):
    if rc != GW_OK:
        lib = load_library()
        detail = lib.gw_strerror(rc).decode()
        if rc == GW_ERR_CUDA and ctx:
            detail += f" (cudaError {lib.gw_last_cuda_error(ctx)})"
        raise GwError(rc, where, detail)


def detector_structs(det_rows: np.ndarray):
    """inputs.py rows [n_det][13] -> ctypes array of gw_detector."""
    rows = np.ascontiguousarray(det_rows, dtype=np.float64).reshape(-1, DET_ROW)
    arr = (gw_detector * rows.shape[0])()
    for i, r in enumerate(rows):
        arr[i].kind = int(r[0])
        arr[i].vertex_m[:] = r[1:4]
        arr[i].xarm[:] = r[4:7]
        arr[i].yarm[:] = r[7:10]
        arr[i].fplus, arr[i].fcross, arr[i].dt_s = float(r[10]), float(r[11]), float(r[12])
    return arr


def _stream_ptr(stream) -> int:
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def _host_ptr(a: np.ndarray) -> int:
    return a.ctypes.data


class GwContext:
    """One analysis segment: frequency grid, per-detector data and PSD, detector geometry (gw_ctx).

    ``freqs`` [M], ``data`` [n_det][M] complex128, ``psd`` [n_det][M]: numpy arrays (host) or torch CUDA
    tensors (device; data as complex128 or [...,2] float64).  ``det_rows``: inputs.py rows [n_det][13].
    """

    def __init__(self, freqs, data, psd, det_rows, gmst: float, spin_order: int = 1,
                 max_batch: int = 4096, stream=None, isco_cut: int = 0, phase_marginal: int = 0,
                 tidal_order: int = 0):
        self._h = ctypes.c_void_p()
        self._lib = load_library()
        self._keep = []
        f_ptr, n_bins = self._as_ptr(freqs, np.float64)
        dets = detector_structs(det_rows)
        self.n_det = len(dets)
        d_ptr, n_d = self._as_ptr(data, np.complex128)
        s_ptr, n_s = self._as_ptr(psd, np.float64)
        if n_d != self.n_det * n_bins or n_s != self.n_det * n_bins:
            raise GwError(GW_ERR_INVALID_ARG, "GwContext", "data/psd must be [n_det][n_bins]")
        opt = gw_options(int(spin_order), int(isco_cut), int(max_batch), int(phase_marginal), int(tidal_order))
        rc = self._lib.gw_ctx_create(ctypes.byref(self._h), n_bins, f_ptr, self.n_det, d_ptr, s_ptr, dets,
                                     float(gmst), ctypes.byref(opt), _stream_ptr(stream))
        self._keep = []
        _check(rc, "gw_ctx_create")
        self.n_bins = int(n_bins)
        self.n_param = int(self._lib.gw_ctx_n_param(self._h))     # 11, or 13 with the tidal option

    def _as_ptr(self, a, dtype) -> Tuple[int, int]:
        """(pointer, element count in units of dtype) for a numpy array or a torch CUDA tensor."""
        try:
            import torch
            if isinstance(a, torch.Tensor):
                t = a.contiguous()
                if dtype is np.complex128 and not t.is_complex():
                    n = t.numel() // 2
                else:
                    n = t.numel()
                want = torch.complex128 if (dtype is np.complex128 and t.is_complex()) else torch.float64
                if t.dtype != want:
                    raise GwError(GW_ERR_INVALID_ARG, "GwContext", f"tensor dtype {t.dtype}, want {want}")
                self._keep.append(t)
                return t.data_ptr(), n
        except ImportError:
            pass
        arr = np.ascontiguousarray(a, dtype=dtype)
        self._keep.append(arr)
        return _host_ptr(arr), arr.size

    # ---- lifetime ----
    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            self._lib.gw_ctx_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # ---- introspection ----
    def info(self):
        nb, nd, df, mb = ctypes.c_int64(), ctypes.c_int(), ctypes.c_double(), ctypes.c_int64()
        _check(self._lib.gw_ctx_info(self._h, ctypes.byref(nb), ctypes.byref(nd), ctypes.byref(df),
                                     ctypes.byref(mb)), "gw_ctx_info")
        return {"n_bins": nb.value, "n_det": nd.value, "delta_f": df.value, "max_batch": mb.value}

    def plan(self, n_prop: int):
        lpp, ppc, nc, ctas = ctypes.c_int(), ctypes.c_int(), ctypes.c_int(), ctypes.c_int64()
        _check(self._lib.gw_ctx_plan(self._h, int(n_prop), ctypes.byref(lpp), ctypes.byref(ppc),
                                     ctypes.byref(nc), ctypes.byref(ctas)), "gw_ctx_plan")
        return {"lanes_per_prop": lpp.value, "props_per_cta": ppc.value, "n_chunks": nc.value, "n_ctas": ctas.value}

    def norms(self) -> np.ndarray:
        out = (ctypes.c_double * MAX_DET)()
        _check(self._lib.gw_ctx_norms(self._h, out), "gw_ctx_norms")
        return np.array(out[: self.n_det])

    def launch_count(self) -> int:
        return int(self._lib.gw_ctx_launch_count(self._h))

    def force_plan(self, lanes_per_prop: int = 0, n_chunks: int = 0):
        """Pin the launch shape of lnl_batch (0 = planner's choice); a testing / tuning aid."""
        _check(self._lib.gw_ctx_force_plan(self._h, int(lanes_per_prop), int(n_chunks)), "gw_ctx_force_plan", self._h)

    def force_grid(self, lanes_per_prop: int = 0, n_ctas: int = 0):
        """Pin the grid of lnl_batch: n_ctas CTAs share the (tile, bin) space equally (0 = planner's choice)."""
        _check(self._lib.gw_ctx_force_grid(self._h, int(lanes_per_prop), int(n_ctas)), "gw_ctx_force_grid", self._h)

    def cluster_finish(self, enable: bool):
        """Tuning aid: cluster / distributed-shared-memory finish of small multi-lane grids on (default) or off."""
        _check(self._lib.gw_ctx_cluster_finish(self._h, int(bool(enable))), "gw_ctx_cluster_finish", self._h)

    def host_graph(self, enable: bool):
        """Tuning aid: small lnl_batch_host calls through the library-owned CUDA graph (default) or launch by launch."""
        _check(self._lib.gw_ctx_host_graph(self._h, int(bool(enable))), "gw_ctx_host_graph", self._h)

    def boundary_bins(self, bins: int):
        """Tuning aid: bins (per lane) by which a range that crosses a tile boundary is shortened on balanced grids."""
        _check(self._lib.gw_ctx_boundary_bins(self._h, int(bins)), "gw_ctx_boundary_bins", self._h)

    def plan_boundary_bins(self, n_prop: int) -> int:
        v = ctypes.c_int()
        _check(self._lib.gw_ctx_plan_boundary_bins(self._h, int(n_prop), ctypes.byref(v)), "gw_ctx_plan_boundary_bins", self._h)
        return v.value

    def kernel_timing(self, enable: bool):
        _check(self._lib.gw_ctx_kernel_timing(self._h, int(bool(enable))), "gw_ctx_kernel_timing", self._h)

    def last_kernel_ms(self):
        """(setup kernel ms, main kernel ms) of the most recent *_batch call made with kernel_timing(True)."""
        a, b = ctypes.c_double(), ctypes.c_double()
        _check(self._lib.gw_ctx_last_kernel_ms(self._h, ctypes.byref(a), ctypes.byref(b)), "gw_ctx_last_kernel_ms", self._h)
        return a.value, b.value

    def reserve(self, max_batch: int):
        _check(self._lib.gw_ctx_reserve(self._h, int(max_batch)), "gw_ctx_reserve", self._h)

    # ---- device-pointer entry points ----
    def _theta_dev(self, theta):
        import torch
        if not (isinstance(theta, torch.Tensor) and theta.is_cuda and theta.dtype == torch.float64
                and theta.is_contiguous() and theta.dim() == 2 and theta.shape[1] == self.n_param):
            raise GwError(GW_ERR_INVALID_ARG, "theta",
                          f"want a contiguous CUDA float64 tensor [n_prop][{self.n_param}]")
        return theta

    @staticmethod
    def _out_dev(t, n_elem, like, what, dtype=None):
        """A caller-supplied output tensor must be CUDA, contiguous, of the right dtype and at least n_elem long,
        on theta's device: the kernels store through its raw pointer."""
        import torch
        dtype = dtype or torch.float64
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()
                and t.numel() >= n_elem and t.device == like.device):
            raise GwError(GW_ERR_INVALID_ARG, what,
                          f"want a contiguous CUDA {dtype} tensor of at least {n_elem} elements on {like.device}")
        return t

    @staticmethod
    def _out_host(a, n_elem, what, dtype=np.float64):
        """A caller-supplied host output must be a C-contiguous, writeable numpy array of the right dtype and size."""
        if not (isinstance(a, np.ndarray) and a.dtype == dtype and a.flags["C_CONTIGUOUS"] and a.flags["WRITEABLE"]
                and a.size >= n_elem):
            raise GwError(GW_ERR_INVALID_ARG, what,
                          f"want a C-contiguous writeable numpy {np.dtype(dtype).name} array of at least {n_elem} elements")
        return a

    def lnl_batch(self, theta, out=None, parts=None, want_parts: bool = False, stream=None):
        """gw_lnl_batch: theta [B][11] CUDA f64 -> lnL [B] (and parts [B][n_det][3]).  Asynchronous."""
        import torch
        th = self._theta_dev(theta)
        n = th.shape[0]
        if out is None:
            out = torch.empty(n, dtype=torch.float64, device=th.device)
        else:
            self._out_dev(out, n, th, "lnl_batch out")
        if parts is None and want_parts:
            parts = torch.empty((n, self.n_det, 3), dtype=torch.float64, device=th.device)
        elif parts is not None:
            self._out_dev(parts, n * self.n_det * 3, th, "lnl_batch parts")
        rc = self._lib.gw_lnl_batch(self._h, n, th.data_ptr(), out.data_ptr(),
                                    parts.data_ptr() if parts is not None else None, _stream_ptr(stream))
        _check(rc, "gw_lnl_batch", self._h)
        return (out, parts) if (want_parts or parts is not None) else out

    def waveform_batch(self, theta, out=None, stream=None):
        """gw_waveform_batch: theta [B][11] CUDA f64 -> h [B][n_det][M] complex128.  Asynchronous."""
        import torch
        th = self._theta_dev(theta)
        n = th.shape[0]
        if out is None:
            out = torch.empty((n, self.n_det, self.n_bins), dtype=torch.complex128, device=th.device)
        else:
            self._out_dev(out, n * self.n_det * self.n_bins, th, "waveform_batch out", torch.complex128)
        rc = self._lib.gw_waveform_batch(self._h, n, th.data_ptr(), out.data_ptr(), _stream_ptr(stream))
        _check(rc, "gw_waveform_batch", self._h)
        return out

    # ---- host-buffer entry points (copies inside the call; synchronises) ----
    def lnl_batch_host(self, theta: np.ndarray, out: Optional[np.ndarray] = None,
                       parts: Optional[np.ndarray] = None, want_parts: bool = False, stream=None):
        th = np.ascontiguousarray(theta, dtype=np.float64).reshape(-1, self.n_param)
        n = th.shape[0]
        if out is None:
            out = np.empty(n)
        else:
            self._out_host(out, n, "lnl_batch_host out")
        if parts is None and want_parts:
            parts = np.empty((n, self.n_det, 3))
        elif parts is not None:
            self._out_host(parts, n * self.n_det * 3, "lnl_batch_host parts")
        rc = self._lib.gw_lnl_batch_host(self._h, n, _host_ptr(th), _host_ptr(out),
                                         _host_ptr(parts) if parts is not None else None, _stream_ptr(stream))
        _check(rc, "gw_lnl_batch_host", self._h)
        return (out, parts) if (want_parts or parts is not None) else out

    def waveform_batch_host(self, theta: np.ndarray, out: Optional[np.ndarray] = None, stream=None):
        th = np.ascontiguousarray(theta, dtype=np.float64).reshape(-1, self.n_param)
        n = th.shape[0]
        if out is None:
            out = np.empty((n, self.n_det, self.n_bins), dtype=np.complex128)
        else:
            self._out_host(out, n * self.n_det * self.n_bins, "waveform_batch_host out", np.complex128)
        rc = self._lib.gw_waveform_batch_host(self._h, n, _host_ptr(th), _host_ptr(out), _stream_ptr(stream))
        _check(rc, "gw_waveform_batch_host", self._h)
        return out


def plan_cta_segments(n_tiles: int, n_bins: int, n_ctas: int, cta: int, max_rows: int = 64, boundary_bins: int = 0) -> np.ndarray:
    """gw_plan_cta_segments (host only): rows (tile, j0, j1, index, count, slot) of the segments one CTA sweeps."""
    lib = load_library()
    rows = np.zeros((max_rows, 6), dtype=np.int64)
    n = lib.gw_plan_cta_segments(int(n_tiles), int(n_bins), int(boundary_bins), int(n_ctas), int(cta), int(max_rows),
                                 rows.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)))
    if n < 0:
        raise GwError(n, "gw_plan_cta_segments", "invalid argument")
    if n > max_rows:
        return plan_cta_segments(n_tiles, n_bins, n_ctas, cta, n, boundary_bins)
    return rows[:n]


def waveform_for_inputs(freqs, det_rows, gmst, theta, spin_order):
    """Adapter with the ``inputs.make_data`` callable signature, computing the injection with the library's
    own gw_waveform_batch (used by bench.py so that its timed path never touches the oracle)."""
    f = np.asarray(freqs, dtype=np.float64)
    rows = np.asarray(det_rows, dtype=np.float64).reshape(-1, DET_ROW)
    n_det = rows.shape[0]
    zeros = np.zeros((n_det, f.size), dtype=np.complex128)
    ones = np.ones((n_det, f.size))
    with GwContext(f, zeros, ones, rows, gmst, spin_order=spin_order, max_batch=max(1, len(theta))) as ctx:
        return ctx.waveform_batch_host(np.asarray(theta, dtype=np.float64))
