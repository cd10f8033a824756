"""Thin Python binding of the population-likelihood entry points of ``csrc/libgwlnl.so`` (include/gwpop.h; PAPER.md
Eq. 3).  Argument marshalling only: every step runs in the CUDA kernels of csrc/gw_pop.cu.  There is no CPU fallback and
nothing here imports ``oracle``.
"""
from __future__ import annotations

import ctypes
from typing import Optional

import numpy as np

from .binding import GW_ERR_INVALID_ARG, GwError, _check, _stream_ptr, load_library

NTHETA = 6      # m1, q, a1, a2, cos tilt_1, cos tilt_2
NLAMBDA = 12    # alpha, m_min, m_max, lam, m_pp, sig_pp, beta_q, alpha_chi, beta_chi, xi, sig_1, sig_2

# every symbol include/gwpop.h declares (tests/test_abi.py checks the library exports each)
EXPORTS = ("gw_pop_ctx_create", "gw_pop_lnl_batch", "gw_pop_lnl_batch_host", "gw_pop_ctx_destroy", "gw_pop_ctx_info",
           "gw_pop_ctx_launch_count", "gw_pop_ctx_kernel_timing", "gw_pop_ctx_last_kernel_ms",
           "gw_pop_lnl_static", "gw_pop_static_need", "gw_pop_static_last_cuda_error")

STATIC_SCRATCH_DOUBLES = 2097152    # GW_POP_STATIC_SCRATCH_DOUBLES: the static device array of gw_pop_lnl_static (16 MiB)
GW_POP_ERR_TOO_LARGE = -16

_declared = False


def _lib():
    global _declared
    lib = load_library()
    if not _declared:
        vp, i64, ci, dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double
        P = ctypes.POINTER
        lib.gw_pop_ctx_create.argtypes = [P(vp), i64, i64, vp, vp, i64, vp]
        lib.gw_pop_lnl_batch.argtypes = [vp, i64, vp, vp, vp]
        lib.gw_pop_lnl_batch_host.argtypes = [vp, i64, vp, vp, vp]
        lib.gw_pop_ctx_destroy.argtypes = [vp]
        lib.gw_pop_ctx_info.argtypes = [vp, P(i64), P(i64), P(i64), P(ci)]
        lib.gw_pop_ctx_launch_count.argtypes = [vp]
        lib.gw_pop_ctx_launch_count.restype = i64
        lib.gw_pop_ctx_kernel_timing.argtypes = [vp, ci]
        lib.gw_pop_ctx_last_kernel_ms.argtypes = [vp, P(dbl), P(dbl), P(dbl)]
        lib.gw_pop_lnl_static.argtypes = [i64, i64, vp, vp, i64, vp, vp, vp]
        lib.gw_pop_static_need.argtypes = [i64, i64, i64]
        lib.gw_pop_static_need.restype = i64
        lib.gw_pop_static_last_cuda_error.argtypes = []
        for name in EXPORTS:
            if name not in ("gw_pop_ctx_launch_count", "gw_pop_static_need"):
                getattr(lib, name).restype = ci
        _declared = True
    return lib


class GwPopContext:
    """Posterior samples of N events (gw_pop_ctx): ``samples`` [N][n][6] and ``prior`` [N][n], numpy arrays (host) or
    torch CUDA float64 tensors (device)."""

    def __init__(self, samples, prior, max_batch: int = 64, stream=None):
        self._h = ctypes.c_void_p()
        self._lib = _lib()
        keep = []

        def ptr(a, shape_tail):
            try:
                import torch
                if isinstance(a, torch.Tensor):
                    t = a.contiguous()
                    if t.dtype != torch.float64:
                        raise GwError(GW_ERR_INVALID_ARG, "GwPopContext", "tensors must be float64")
                    keep.append(t)
                    return t.data_ptr(), tuple(t.shape)
            except ImportError:
                pass
            arr = np.ascontiguousarray(a, dtype=np.float64)
            keep.append(arr)
            return arr.ctypes.data, arr.shape

        s_ptr, s_shape = ptr(samples, (NTHETA,))
        p_ptr, p_shape = ptr(prior, ())
        if len(s_shape) != 3 or s_shape[2] != NTHETA or tuple(p_shape) != tuple(s_shape[:2]):
            raise GwError(GW_ERR_INVALID_ARG, "GwPopContext", "samples must be [N][n][6] and prior [N][n]")
        self.n_events, self.n_samples = int(s_shape[0]), int(s_shape[1])
        rc = self._lib.gw_pop_ctx_create(ctypes.byref(self._h), self.n_events, self.n_samples, s_ptr, p_ptr,
                                         int(max_batch), _stream_ptr(stream))
        _check(rc, "gw_pop_ctx_create")

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            self._lib.gw_pop_ctx_destroy(self._h)
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

    def info(self):
        ne, ns, mb, cpe = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int()
        _check(self._lib.gw_pop_ctx_info(self._h, ctypes.byref(ne), ctypes.byref(ns), ctypes.byref(mb), ctypes.byref(cpe)),
               "gw_pop_ctx_info")
        return {"n_events": ne.value, "n_samples": ns.value, "max_batch": mb.value, "chunks_per_event": cpe.value}

    def launch_count(self) -> int:
        return int(self._lib.gw_pop_ctx_launch_count(self._h))

    def kernel_timing(self, enable: bool):
        _check(self._lib.gw_pop_ctx_kernel_timing(self._h, int(bool(enable))), "gw_pop_ctx_kernel_timing")

    def last_kernel_ms(self):
        """(setup, main, finish) kernel ms of the most recent lnl_batch call made with kernel_timing(True)."""
        a, b, c = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
        _check(self._lib.gw_pop_ctx_last_kernel_ms(self._h, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)),
               "gw_pop_ctx_last_kernel_ms")
        return a.value, b.value, c.value

    def lnl_batch(self, lambdas, out=None, stream=None):
        """gw_pop_lnl_batch: Lambda [B][12] CUDA f64 -> lnL [B].  Asynchronous."""
        import torch
        lam = lambdas
        if not (isinstance(lam, torch.Tensor) and lam.is_cuda and lam.dtype == torch.float64 and lam.is_contiguous()
                and lam.dim() == 2 and lam.shape[1] == NLAMBDA):
            raise GwError(GW_ERR_INVALID_ARG, "lambdas", "want a contiguous CUDA float64 tensor [B][12]")
        n = lam.shape[0]
        if out is None:
            out = torch.empty(n, dtype=torch.float64, device=lam.device)
        elif not (isinstance(out, torch.Tensor) and out.is_cuda and out.dtype == torch.float64 and out.is_contiguous()
                  and out.numel() >= n and out.device == lam.device):
            raise GwError(GW_ERR_INVALID_ARG, "lnl_batch out", f"want a contiguous CUDA float64 tensor of at least {n} elements")
        _check(self._lib.gw_pop_lnl_batch(self._h, n, lam.data_ptr(), out.data_ptr(), _stream_ptr(stream)), "gw_pop_lnl_batch")
        return out

    def lnl_batch_host(self, lambdas: np.ndarray, out: Optional[np.ndarray] = None, stream=None) -> np.ndarray:
        lam = np.ascontiguousarray(lambdas, dtype=np.float64).reshape(-1, NLAMBDA)
        n = lam.shape[0]
        if out is None:
            out = np.empty(n)
        elif not (isinstance(out, np.ndarray) and out.dtype == np.float64 and out.flags["C_CONTIGUOUS"] and out.size >= n):
            raise GwError(GW_ERR_INVALID_ARG, "lnl_batch_host out", f"want a C-contiguous float64 array of at least {n} elements")
        _check(self._lib.gw_pop_lnl_batch_host(self._h, n, lam.ctypes.data, out.ctypes.data, _stream_ptr(stream)),
               "gw_pop_lnl_batch_host")
        return out


def static_need(n_events: int, n_samples: int, n_lambda: int) -> int:
    """gw_pop_static_need: doubles of static scratch gw_pop_lnl_static needs for this size (-1: a size it rejects)."""
    return int(_lib().gw_pop_static_need(int(n_events), int(n_samples), int(n_lambda)))


def lnl_static(samples, prior, lambdas, out=None, stream=None):
    """gw_pop_lnl_static, the entry point that allocates nothing: samples [N][n][6], prior [N][n], Lambda [B][12], all
    contiguous CUDA float64 tensors on the current device -> lnL [B] (``out`` or a new tensor -- pass ``out`` where
    torch must not allocate either).  No context; the scratch is a static device array inside the library, shared by
    every call: calls that overlap on the GPU race.  Asynchronous.  A problem beyond the array raises GwError with
    code GW_POP_ERR_TOO_LARGE."""
    import torch
    for name, t, nd in (("samples", samples, 3), ("prior", prior, 2), ("lambdas", lambdas, 2)):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.dim() == nd):
            raise GwError(GW_ERR_INVALID_ARG, f"lnl_static {name}", f"want a contiguous CUDA float64 tensor with {nd} dimensions")
    if samples.shape[2] != NTHETA or tuple(prior.shape) != tuple(samples.shape[:2]) or lambdas.shape[1] != NLAMBDA:
        raise GwError(GW_ERR_INVALID_ARG, "lnl_static", "samples must be [N][n][6], prior [N][n] and lambdas [B][12]")
    n_events, n_samples, n = int(samples.shape[0]), int(samples.shape[1]), int(lambdas.shape[0])
    if out is None:
        out = torch.empty(n, dtype=torch.float64, device=lambdas.device)
    elif not (isinstance(out, torch.Tensor) and out.is_cuda and out.dtype == torch.float64 and out.is_contiguous()
              and out.numel() >= n and out.device == lambdas.device):
        raise GwError(GW_ERR_INVALID_ARG, "lnl_static out", f"want a contiguous CUDA float64 tensor of at least {n} elements")
    lib = _lib()
    rc = lib.gw_pop_lnl_static(n_events, n_samples, samples.data_ptr(), prior.data_ptr(), n, lambdas.data_ptr(),
                               out.data_ptr(), _stream_ptr(stream))
    if rc == GW_POP_ERR_TOO_LARGE:
        raise GwError(rc, "gw_pop_lnl_static",
                      f"{n_events} x {n_samples} samples with {n} Lambda need {static_need(n_events, n_samples, n)} doubles of "
                      f"scratch, the static array holds {STATIC_SCRATCH_DOUBLES}: use a GwPopContext")
    if rc == -3:
        raise GwError(rc, "gw_pop_lnl_static", f"CUDA runtime error (cudaError {lib.gw_pop_static_last_cuda_error()})")
    _check(rc, "gw_pop_lnl_static")
    return out
