"""Pins for the NEXT-1 options of the oracle:
inspiral cut-off at f_ISCO and the likelihood marginalised over the coalescence phase."""
import math

import numpy as np
import pytest
from scipy import special

from paper_1904_02863_b200 import inputs

C_SI, GMSUN = 299792458.0, 1.3271244e20


def _case(f_max=2048.0, batch=24, name="C1"):
    cfg = inputs.CONFIGS[name].reduced(f_max=f_max, batch=batch)
    return cfg, inputs.frequency_grid(cfg), inputs.psd(cfg), inputs.detectors(cfg), inputs.proposals(cfg)


# ------------------------------------------------------------------------------------------ f_ISCO
def test_f_isco_anchors_and_closed_form(oracle):
    """SURVEY.md scale table: Mc=40, q=0.5 (M = 98.6 Msun) -> 44.6 Hz; Mc=1.3, q=0.7 (M = 3.04 Msun) -> 1445 Hz.
    Closed form from SI quantities: c^3 / (6^(3/2) pi G M)."""
    assert oracle.f_isco(40.0, 0.5) == pytest.approx(44.6, abs=0.05)
    assert oracle.f_isco(1.3, 0.7) == pytest.approx(1445.0, abs=0.5)
    for mc, q in [(28.0, 0.8), (1.2, 0.9), (35.0, 1.0)]:
        eta = q / (1 + q) ** 2
        m_si = mc * eta ** -0.6                                         # Msun
        want = C_SI ** 3 / (6 ** 1.5 * math.pi * GMSUN * m_si)
        assert oracle.f_isco(mc, q) == pytest.approx(want, rel=1e-14)
    # scales as 1/M: doubling the chirp mass at fixed q halves it
    assert oracle.f_isco(20.0, 0.7) / oracle.f_isco(40.0, 0.7) == pytest.approx(2.0, rel=1e-15)


def test_isco_cut_is_a_mask_on_the_uncut_waveform(oracle):
    cfg, f, S, dets, th = _case(batch=12)
    h0 = oracle.waveform(f, dets, cfg.gmst, th)
    h1 = oracle.waveform(f, dets, cfg.gmst, th, isco_cut=1)
    for b in range(len(th)):
        fi = oracle.f_isco(th[b, inputs.P_MC], th[b, inputs.P_Q])
        keep = f <= fi
        assert 0 < keep.sum() < f.size                                  # BBH: the cut falls inside 20-2048 Hz
        assert np.array_equal(h1[b][:, keep], h0[b][:, keep])
        assert np.all(h1[b][:, ~keep] == 0)


def test_isco_cut_hh_closed_form_and_zero_data(oracle):
    """<h|h>_I = |C_I|^2 A0^2 4 df sum_{f_j <= f_ISCO} f_j^(-7/3)/S_j; with d = 0, lnL = -1/2 sum_I <h|h>_I."""
    cfg, f, S, dets, th = _case(batch=16)
    zero = np.zeros((cfg.n_det, f.size), complex)
    lnl, parts, _ = oracle.lnl(f, cfg.delta_f, zero, S, dets, cfg.gmst, th, isco_cut=1)
    _, parts_full, _ = oracle.lnl(f, cfg.delta_f, zero, S, dets, cfg.gmst, th)
    cum = np.cumsum(f ** (-7.0 / 3.0) / S[0])
    for b in range(len(th)):
        fi = oracle.f_isco(th[b, inputs.P_MC], th[b, inputs.P_Q])
        j = np.searchsorted(f, fi, side="right") - 1
        ratio = cum[j] / cum[-1]
        np.testing.assert_allclose(parts[b, :, 2], parts_full[b, :, 2] * ratio, rtol=1e-12)
    np.testing.assert_allclose(lnl, -0.5 * parts[..., 2].sum(axis=1), rtol=1e-15)
    assert np.all(parts[..., :2] == 0)


def test_isco_cut_above_band_changes_nothing(oracle):
    """BNS: f_ISCO (~1500 Hz) above a 20-512 Hz band: identical to the uncut result."""
    cfg, f, S, dets, th = _case(f_max=100.0, batch=6, name="C2")
    d = inputs.make_data(cfg, oracle.waveform)
    a = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th)
    b = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, isco_cut=1)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


# ------------------------------------------------------------------------------------------ ln I0
def test_log_bessel_i0_against_library_and_limits(oracle):
    for x in [0.0, 1e-4, 0.3, 1.0, 7.5, 42.0, 300.0, 5e3, 2e5]:
        want = math.log(special.ive(0, x)) + x
        assert oracle.log_bessel_i0(x) == pytest.approx(want, rel=2e-14, abs=1e-15)
    assert oracle.log_bessel_i0(1e-3) == pytest.approx(math.log1p(1e-6 / 4 + 1e-12 / 64), rel=1e-9)     # series
    x = 1e4                                                                                              # asymptotic
    assert oracle.log_bessel_i0(x) == pytest.approx(x - 0.5 * math.log(2 * math.pi * x) + math.log1p(1 / (8 * x) + 9 / (128 * x * x)), rel=1e-14)
    assert oracle.log_bessel_i0(-3.0) == oracle.log_bessel_i0(3.0)


# ------------------------------------------------------------------------------------------ marginalisation
def test_phase_marginal_equals_quadrature_over_phic(oracle):
    """ln[(1/2pi) int exp(lnL(phi_c)) dphi_c] by brute force (512-point periodic trapezoid over phi_c, each point a
    full oracle lnL) equals ln I0(|sum <d|h>|) - 1/2 sum <h|h>."""
    cfg, f, S, dets, th = _case(f_max=128.0, batch=6)
    d = inputs.make_data(cfg, oracle.waveform)
    n = 512
    phis = 2 * math.pi * np.arange(n) / n
    for b in range(len(th)):
        rows = np.tile(th[b], (n, 1))
        rows[:, inputs.P_PHIC] = phis
        lnl, parts, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, rows)
        m = lnl.max()
        brute = m + math.log(np.mean(np.exp(lnl - m)))
        marg = oracle.lnl_phase_marginal(parts)
        assert np.ptp(marg) <= 1e-10 * max(1.0, abs(marg[0]))            # independent of the phi_c it is evaluated at
        assert marg[0] == pytest.approx(brute, rel=1e-11, abs=1e-11)
        assert marg[0] <= lnl.max() + 1e-12 and marg[0] >= lnl.min() - 1e-12   # a mean lies between the extremes


def test_phase_marginal_zero_data(oracle):
    cfg, f, S, dets, th = _case(f_max=64.0, batch=4)
    zero = np.zeros((cfg.n_det, f.size), complex)
    lnl, parts, _ = oracle.lnl(f, cfg.delta_f, zero, S, dets, cfg.gmst, th)
    np.testing.assert_array_equal(oracle.lnl_phase_marginal(parts), lnl)     # I0(0) = 1
