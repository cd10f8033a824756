"""CPU oracle -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Thin ctypes loader for ``oracle/gw_oracle.c`` (plain C, fp64, libm), the slow and
obviously-correct statement of what the hot path computes (Eq. 1,
PAPER.md:69 time shift; waveform per BASELINE.json north_star, written out in
SURVEY.md 8(c) O1..O7).  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` leg of ``bench.py`` may import this
package.  It imports nothing from ``paper_1904_02863_b200`` and shares no code
with the CUDA path.  All marshalling below is argument plumbing: every number is
computed inside ``gw_oracle.c``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gw_oracle.c")
_LIB = os.path.join(_HERE, "libgw_oracle.so")

NPARAM = 11          # Mc, q, chi1, chi2, DL, tc, phic, cos(iota), ra, dec, psi
DET_ROW = 13         # kind, vertex[3], xarm[3], yarm[3], fplus, fcross, dt

_POP_SRC = os.path.join(_HERE, "gw_pop_oracle.c")
_POP_LIB = os.path.join(_HERE, "libgw_pop_oracle.so")
POP_NTHETA = 6       # m1, q, a1, a2, cos tilt1, cos tilt2
POP_NLAMBDA = 12     # alpha, m_min, m_max, lam, m_pp, sig_pp, beta_q, alpha_chi, beta_chi, xi, sig_1, sig_2

_lib = None
_pop_lib = None


def _compile(src: str, lib: str, force: bool) -> str:
    if force or not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(src):
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
               "-Wall", "-Wextra", "-o", lib, src, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return lib


def build(force: bool = False) -> str:
    """Compile gw_oracle.c and gw_pop_oracle.c with gcc (-O2, no fast-math, OpenMP over proposals / events)."""
    _compile(_POP_SRC, _POP_LIB, force)
    return _compile(_SRC, _LIB, force)


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build()
    lib = ctypes.CDLL(_LIB)
    dp = ctypes.POINTER(ctypes.c_double)
    i64, cint, dbl = ctypes.c_int64, ctypes.c_int, ctypes.c_double
    lib.gwo_constants.argtypes = [dp]
    lib.gwo_masses.argtypes = [dbl, dbl, dp, dp, dp, dp]
    lib.gwo_phase_coefficients.argtypes = [dbl, dbl, dbl, dbl, dbl, cint, dp, dp]
    lib.gwo_phase.argtypes = [dbl, dp, cint]
    lib.gwo_phase.restype = dbl
    lib.gwo_amplitude.argtypes = [dbl, dbl]
    lib.gwo_amplitude.restype = dbl
    lib.gwo_antenna.argtypes = [dp, dbl, dbl, dbl, dbl, dp, dp, dp]
    lib.gwo_sky_frame.argtypes = [dbl, dbl, dbl, dbl, dp, dp, dp]
    lib.gwo_waveform.argtypes = [i64, dp, cint, dp, dbl, i64, dp, cint, dp]
    lib.gwo_waveform_opt.argtypes = [i64, dp, cint, dp, dbl, i64, dp, cint, cint, dp]
    lib.gwo_lnl_opt.argtypes = [i64, dp, dbl, cint, dp, dp, dp, dbl, i64, dp, cint, cint, cint, dp, dp]
    lib.gwo_lnl_opt.restype = cint
    lib.gwo_tidal_coefficients.argtypes = [dbl, dbl, dbl, cint, dp, dp]
    lib.gwo_phase_tidal.argtypes = [dbl, dp, cint, dp, cint]
    lib.gwo_phase_tidal.restype = dbl
    lib.gwo_waveform_tidal.argtypes = [i64, dp, cint, dp, dbl, i64, dp, cint, cint, dp, cint, dp]
    lib.gwo_lnl_tidal.argtypes = [i64, dp, dbl, cint, dp, dp, dp, dbl, i64, dp, cint, cint, dp, cint, cint, dp, dp]
    lib.gwo_lnl_tidal.restype = cint
    lib.gwo_f_isco.argtypes = [dbl, dbl]
    lib.gwo_f_isco.restype = dbl
    lib.gwo_log_bessel_i0.argtypes = [dbl]
    lib.gwo_log_bessel_i0.restype = dbl
    lib.gwo_lnl_phase_marginal.argtypes = [i64, cint, dp, dp]
    lib.gwo_lnl.argtypes = [i64, dp, dbl, cint, dp, dp, dp, dbl, i64, dp, cint, cint, dp, dp]
    lib.gwo_lnl.restype = cint
    lib.gwo_inner.argtypes = [i64, dbl, dp, dp, dp, dp, dp]
    lib.gwo_norm_i7.argtypes = [i64, dp, dbl, dp]
    lib.gwo_norm_i7.restype = dbl
    _lib = lib
    return lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _f64(a, shape=None) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        a = a.reshape(shape)
    return a


def _ri(z) -> np.ndarray:
    """complex128 array -> contiguous float64 view with trailing (re, im)."""
    z = np.ascontiguousarray(z, dtype=np.complex128)
    return z.view(np.float64).reshape(z.shape + (2,))


def constants() -> dict:
    out = np.zeros(4)
    _load().gwo_constants(_p(out))
    return {"tsun_s": out[0], "mpc_s": out[1], "c_si": out[2], "euler_gamma": out[3]}


def masses(mc: float, q: float):
    """O1 -> (eta, M_s [s], mu1, mu2)."""
    vals = [ctypes.c_double() for _ in range(4)]
    _load().gwo_masses(mc, q, *[ctypes.byref(v) for v in vals])
    return tuple(v.value for v in vals)


def phase_coefficients(eta, mu1, mu2, chi1=0.0, chi2=0.0, spin_order=1):
    """O2 -> (phi[8], phil[8])."""
    phi, phil = np.zeros(8), np.zeros(8)
    _load().gwo_phase_coefficients(eta, mu1, mu2, chi1, chi2, spin_order, _p(phi), _p(phil))
    return phi, phil


def phase(freqs, theta, spin_order=1, lambdas=None, tidal_order=0) -> np.ndarray:
    """O3: Psi(f) for one theta[11] at each frequency (tidal option: lambdas = (Lambda_1, Lambda_2))."""
    lib = _load()
    th = _f64(theta, (NPARAM,))
    if lambdas is None or tidal_order == 0:
        return np.array([lib.gwo_phase(float(f), _p(th), spin_order) for f in np.atleast_1d(freqs)])
    lam = _f64(lambdas, (2,))
    return np.array([lib.gwo_phase_tidal(float(f), _p(th), spin_order, _p(lam), int(tidal_order))
                     for f in np.atleast_1d(freqs)])


def tidal_coefficients(eta, lambda1, lambda2, tidal_order=2):
    """NEXT-1 option -> (phi_10, phi_12) in units of 3/(128 eta) v^(k-5)."""
    a, b = ctypes.c_double(), ctypes.c_double()
    _load().gwo_tidal_coefficients(eta, lambda1, lambda2, int(tidal_order), ctypes.byref(a), ctypes.byref(b))
    return a.value, b.value


def amplitude(mc: float, dl: float) -> float:
    """O4: A0."""
    return _load().gwo_amplitude(mc, dl)


def antenna(det_row, ra, dec, psi, gmst):
    """O6 -> (F+, Fx, dt_s) for one detector row."""
    d = _f64(det_row, (DET_ROW,))
    vals = [ctypes.c_double() for _ in range(3)]
    _load().gwo_antenna(_p(d), ra, dec, psi, gmst, *[ctypes.byref(v) for v in vals])
    return tuple(v.value for v in vals)


def sky_frame(ra, dec, psi, gmst):
    """O6 -> (X, Y, n) unit vectors."""
    X, Y, n = np.zeros(3), np.zeros(3), np.zeros(3)
    _load().gwo_sky_frame(ra, dec, psi, gmst, _p(X), _p(Y), _p(n))
    return X, Y, n


def _lambdas(lambdas, n_prop, tidal_order):
    if lambdas is None or tidal_order == 0:
        return None, None, 0
    lam = _f64(lambdas).reshape(n_prop, 2)
    return lam, _p(lam), int(tidal_order)


def waveform(freqs, dets, gmst, theta, spin_order=1, isco_cut=0, lambdas=None, tidal_order=0) -> np.ndarray:
    """O4..O6: h[n_prop][n_det][n_bins] complex128 (isco_cut=1: zero above f_ISCO; lambdas[n_prop][2] with
    tidal_order 1 | 2: 5PN | 5PN + 6PN tidal phase terms -- NEXT-1 options)."""
    f = _f64(freqs)
    d = _f64(dets).reshape(-1, DET_ROW)
    th = _f64(theta).reshape(-1, NPARAM)
    out = np.empty((th.shape[0], d.shape[0], f.shape[0], 2))
    lam, lam_p, order = _lambdas(lambdas, th.shape[0], tidal_order)
    _load().gwo_waveform_tidal(f.shape[0], _p(f), d.shape[0], _p(d), gmst, th.shape[0], _p(th),
                               spin_order, int(isco_cut), lam_p, order, _p(out))
    return out.view(np.complex128)[..., 0]


def lnl(freqs, delta_f, data, psd, dets, gmst, theta, spin_order=1, n_threads=0, isco_cut=0,
        lambdas=None, tidal_order=0):
    """O7 -> (lnL[n_prop], parts[n_prop][n_det][3], threads_used)."""
    f = _f64(freqs)
    d = _f64(dets).reshape(-1, DET_ROW)
    n_det, n_bins = d.shape[0], f.shape[0]
    dat = _ri(np.asarray(data).reshape(n_det, n_bins))
    S = _f64(psd, (n_det, n_bins))
    th = _f64(theta).reshape(-1, NPARAM)
    out = np.empty(th.shape[0])
    parts = np.empty((th.shape[0], n_det, 3))
    lam, lam_p, order = _lambdas(lambdas, th.shape[0], tidal_order)
    used = _load().gwo_lnl_tidal(n_bins, _p(f), float(delta_f), n_det, _p(dat), _p(S), _p(d), gmst,
                                 th.shape[0], _p(th), spin_order, int(isco_cut), lam_p, order, int(n_threads),
                                 _p(out), _p(parts))
    return out, parts, used


def inner(delta_f, a, b, psd) -> complex:
    """<a|b> = 4 df sum a conj(b)/S for one detector."""
    a_, b_, S = _ri(np.ravel(a)), _ri(np.ravel(b)), _f64(np.ravel(psd))
    re, im = ctypes.c_double(), ctypes.c_double()
    _load().gwo_inner(S.shape[0], float(delta_f), _p(a_), _p(b_), _p(S), ctypes.byref(re), ctypes.byref(im))
    return complex(re.value, im.value)


def norm_i7(freqs, delta_f, psd) -> float:
    """I7 = 4 df sum f^(-7/3)/S."""
    f, S = _f64(freqs), _f64(psd)
    return _load().gwo_norm_i7(f.shape[0], _p(f), float(delta_f), _p(S))


def f_isco(mc: float, q: float) -> float:
    """NEXT-1 option: 1/(6^(3/2) pi M_s)."""
    return _load().gwo_f_isco(mc, q)


def log_bessel_i0(x: float) -> float:
    """ln I0(x) from the integral definition (trapezoid rule)."""
    return _load().gwo_log_bessel_i0(float(x))


def lnl_phase_marginal(parts) -> np.ndarray:
    """NEXT-1 option: ln I0(|sum_I <d|h>_I|) - 1/2 sum_I <h|h>_I per proposal, from parts[n_prop][n_det][3]."""
    p = _f64(parts)
    out = np.empty(p.shape[0])
    _load().gwo_lnl_phase_marginal(p.shape[0], p.shape[1], _p(p), _p(out))
    return out


# ---- population likelihood, Eq. 3 (gw_pop_oracle.c) ------------------------------------------------------
def _pop():
    global _pop_lib
    if _pop_lib is None:
        build()
        lib = ctypes.CDLL(_POP_LIB)
        dp, i64, cint, dbl = ctypes.POINTER(ctypes.c_double), ctypes.c_int64, ctypes.c_int, ctypes.c_double
        for name, args in (("gwpo_powerlaw_pdf", [dbl] * 4), ("gwpo_truncnorm_pdf", [dbl] * 5),
                           ("gwpo_mass_pdf", [dbl, dp]), ("gwpo_ratio_pdf", [dbl, dbl, dp]),
                           ("gwpo_beta_pdf", [dbl] * 3), ("gwpo_tilt_pdf", [dbl, dbl, dp]),
                           ("gwpo_population_pdf", [dp, dp])):
            f = getattr(lib, name)
            f.argtypes, f.restype = args, dbl
        lib.gwpo_lambda_valid.argtypes, lib.gwpo_lambda_valid.restype = [dp], cint
        lib.gwpo_lnl.argtypes = [i64, i64, dp, dp, i64, dp, cint, dp, dp]
        lib.gwpo_lnl.restype = cint
        _pop_lib = lib
    return _pop_lib


def pop_powerlaw_pdf(x, alpha, lo, hi) -> float:
    return _pop().gwpo_powerlaw_pdf(float(x), float(alpha), float(lo), float(hi))


def pop_truncnorm_pdf(x, mu, sigma, lo, hi) -> float:
    return _pop().gwpo_truncnorm_pdf(float(x), float(mu), float(sigma), float(lo), float(hi))


def pop_mass_pdf(m1, lam) -> float:
    return _pop().gwpo_mass_pdf(float(m1), _p(_f64(lam, (POP_NLAMBDA,))))


def pop_ratio_pdf(q, m1, lam) -> float:
    return _pop().gwpo_ratio_pdf(float(q), float(m1), _p(_f64(lam, (POP_NLAMBDA,))))


def pop_beta_pdf(a, alpha_chi, beta_chi) -> float:
    return _pop().gwpo_beta_pdf(float(a), float(alpha_chi), float(beta_chi))


def pop_tilt_pdf(c1, c2, lam) -> float:
    return _pop().gwpo_tilt_pdf(float(c1), float(c2), _p(_f64(lam, (POP_NLAMBDA,))))


def pop_pdf(theta, lam) -> float:
    """p(theta | Lambda) for one theta[6] and one Lambda[12]."""
    return _pop().gwpo_population_pdf(_p(_f64(theta, (POP_NTHETA,))), _p(_f64(lam, (POP_NLAMBDA,))))


def pop_lambda_valid(lam) -> bool:
    return bool(_pop().gwpo_lambda_valid(_p(_f64(lam, (POP_NLAMBDA,)))))


def pop_lnl(samples, prior, lambdas, n_threads=0):
    """Eq. 3 without its prefactor -> (lnL[B], inner sums [B][N], threads used).
    samples [N][n][6], prior [N][n], lambdas [B][12]."""
    s = _f64(samples)
    n_events, n_samples = s.shape[0], s.shape[1]
    s = s.reshape(n_events, n_samples, POP_NTHETA)
    p0 = _f64(prior, (n_events, n_samples))
    lam = _f64(lambdas).reshape(-1, POP_NLAMBDA)
    out = np.empty(lam.shape[0])
    inner = np.empty((lam.shape[0], n_events))
    used = _pop().gwpo_lnl(n_events, n_samples, _p(s), _p(p0), lam.shape[0], _p(lam), int(n_threads), _p(out), _p(inner))
    if used < 0:
        raise MemoryError("gwpo_lnl")
    return out, inner, used
