"""Pins for the oracle's inner products and lnL (SURVEY.md 8(c) pins P3, P4, P8; reading A2).

The paper's Eq. 1 fixes the normalisation: exponent -(2/T)|d-h|^2/S.
"""
import math

import numpy as np
import pytest

from paper_1904_02863_b200 import inputs


def _small(name="C1", f_max=96.0, batch=6):
    cfg = inputs.CONFIGS[name].reduced(f_max=f_max, batch=batch)
    return cfg, inputs.frequency_grid(cfg), inputs.psd(cfg), inputs.detectors(cfg)


def test_p3_zero_data_gives_minus_half_hh(oracle):
    cfg, f, S, dets = _small()
    th = inputs.proposals(cfg)
    zero = np.zeros((cfg.n_det, cfg.n_bins), complex)
    lnl, parts, _ = oracle.lnl(f, cfg.delta_f, zero, S, dets, cfg.gmst, th)
    assert np.all(parts[..., 0] == 0) and np.all(parts[..., 1] == 0)
    np.testing.assert_allclose(lnl, -0.5 * parts[..., 2].sum(axis=1), rtol=1e-15)
    assert np.all(lnl < 0)


def test_p3_noiseless_data_at_truth_gives_plus_half_hh(oracle):
    cfg, f, S, dets = _small()
    th = inputs.proposals(cfg)
    d = oracle.waveform(f, dets, cfg.gmst, th[:1])[0]
    lnl, parts, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th)
    hh = parts[0, :, 2].sum()
    assert lnl[0] == pytest.approx(0.5 * hh, rel=1e-13)
    assert np.abs(parts[0, :, 1]).max() < 1e-12 * hh          # Im<d|h> = 0 at the truth
    np.testing.assert_allclose(parts[0, :, 0], parts[0, :, 2], rtol=1e-13)
    # Cauchy-Schwarz: lnL(theta) <= 1/2 <d|d>, equality only at h = d
    dd = sum(oracle.inner(cfg.delta_f, d[i], d[i], S[i]).real for i in range(cfg.n_det))
    assert dd == pytest.approx(hh, rel=1e-13)
    assert np.all(lnl[1:] < 0.5 * dd)


def test_p3_cauchy_schwarz_with_noise(oracle):
    cfg, f, S, dets = _small(batch=32)
    th = inputs.proposals(cfg)
    d = inputs.make_data(cfg, oracle.waveform)
    lnl, parts, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th)
    dd = sum(oracle.inner(cfg.delta_f, d[i], d[i], S[i]).real for i in range(cfg.n_det))
    assert np.all(lnl <= 0.5 * dd)
    for i in range(cfg.n_det):
        ddi = oracle.inner(cfg.delta_f, d[i], d[i], S[i]).real
        assert np.all(parts[:, i, 0] ** 2 + parts[:, i, 1] ** 2 <= ddi * parts[:, i, 2] * (1 + 1e-12))


def test_eq1_log_likelihood_ratio(oracle):
    """lnL = ln L_Eq1(d|theta) - ln L_Eq1(d|h=0), with Eq. 1 typed as printed:
    ln L_Eq1 = sum_ij [ -ln(2 pi S_ij) - (2/T) |d_ij - h_ij|^2 / S_ij ]."""
    cfg, f, S, dets = _small("C1", 80.0, 5)
    th = inputs.proposals(cfg)
    d = inputs.make_data(cfg, oracle.waveform)
    h = oracle.waveform(f, dets, cfg.gmst, th)
    T = cfg.duration_s

    def ln_eq1(model):
        return np.sum(-np.log(2 * np.pi * S) - (2.0 / T) * np.abs(d - model) ** 2 / S)

    lnl, _, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th)
    noise_only = ln_eq1(np.zeros_like(d))
    for b in range(th.shape[0]):
        assert lnl[b] == pytest.approx(ln_eq1(h[b]) - noise_only, rel=1e-9, abs=1e-9)


def test_inner_product_normalisation_matches_noise_recipe(oracle):
    """BASELINE.json configs[0]: noise variance S/(4 df) per component  <=>  Var Re<n|h> = <h|h>
    (the 4 df of the inner product and the noise recipe are one convention; reading A2)."""
    cfg, f, S, dets = _small("C0", 148.0, 1)
    th = inputs.proposals(cfg)
    h = oracle.waveform(f, dets, cfg.gmst, th, cfg.spin_order)[0, 0]
    hh = oracle.inner(cfg.delta_f, h, h, S[0]).real
    rng = np.random.default_rng(11)
    sig = np.sqrt(S[0] / (4 * cfg.delta_f))
    n_real = 4000
    z = (rng.standard_normal((n_real, cfg.n_bins)) + 1j * rng.standard_normal((n_real, cfg.n_bins))) * sig
    nh = 4 * cfg.delta_f * np.sum(z * np.conj(h) / S[0], axis=1)
    assert nh.real.var() == pytest.approx(hh, rel=0.08)      # 4000 draws: sigma(var)/var = sqrt(2/4000) = 2.2 %
    assert nh.imag.var() == pytest.approx(hh, rel=0.08)
    assert abs(nh.real.mean()) < 5 * math.sqrt(hh / n_real)


def test_p4_lnl_invariant_when_data_and_tc_shift_together(oracle):
    cfg, f, S, dets = _small()
    th = inputs.proposals(cfg)
    d = inputs.make_data(cfg, oracle.waveform)
    tau = 0.004
    d_shift = d * np.exp(-2j * np.pi * f * tau)[None, :]
    th_shift = th.copy(); th_shift[:, inputs.P_TC] += tau
    a, pa, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th)
    b, pb, _ = oracle.lnl(f, cfg.delta_f, d_shift, S, dets, cfg.gmst, th_shift)
    scale = np.abs(pa[..., 0]).sum(axis=1) + pa[..., 2].sum(axis=1)
    assert np.all(np.abs(a - b) < 1e-10 * scale)


def test_parts_sum_to_lnl_and_detectors_add(oracle):
    cfg, f, S, dets = _small()
    th = inputs.proposals(cfg)
    d = inputs.make_data(cfg, oracle.waveform)
    lnl, parts, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th)
    np.testing.assert_allclose(lnl, (parts[..., 0] - 0.5 * parts[..., 2]).sum(axis=1), rtol=1e-14)
    single = sum(oracle.lnl(f, cfg.delta_f, d[i:i + 1], S[i:i + 1], dets[i:i + 1], cfg.gmst, th)[0] for i in range(3))
    np.testing.assert_allclose(lnl, single, rtol=1e-13, atol=1e-12)


def test_p8_tiny_case_by_brute_force(oracle):
    """M = 4 bins, B = 2, one FIXED detector: <d|h> and <h|h> expanded term by term in Python complex
    arithmetic from the oracle's own h (pins the conjugation side, the 4 df factor and the output layout)."""
    f = np.array([30.0, 30.5, 31.0, 31.5])
    df = 0.5
    S = np.array([[2e-46, 3e-46, 2.5e-46, 4e-46]])
    det = inputs.fixed_detector(0.6, -0.3, 0.002)[None]
    th = np.array([[25.0, 0.7, 0.1, -0.3, 400.0, 0.02, 0.5, 0.4, 0, 0, 0],
                   [35.0, 0.9, 0.0, 0.2, 900.0, -0.03, 2.5, -0.8, 0, 0, 0]])
    d = np.array([[1e-23 + 2e-23j, -3e-23 + 1e-23j, 2e-23 - 2e-23j, -1e-23 - 1e-23j]])
    h = oracle.waveform(f, det, 0.0, th)
    lnl, parts, _ = oracle.lnl(f, df, d, S, det, 0.0, th)
    for b in range(2):
        dh = sum(4 * df * d[0, j] * h[b, 0, j].conjugate() / S[0, j] for j in range(4))
        hh = sum(4 * df * abs(h[b, 0, j]) ** 2 / S[0, j] for j in range(4))
        assert parts[b, 0, 0] == pytest.approx(dh.real, rel=1e-14)
        assert parts[b, 0, 1] == pytest.approx(dh.imag, rel=1e-14)
        assert parts[b, 0, 2] == pytest.approx(hh, rel=1e-14)
        assert lnl[b] == pytest.approx(dh.real - 0.5 * hh, rel=1e-13)


def test_openmp_thread_count_does_not_change_results(oracle):
    cfg, f, S, dets = _small(batch=16)
    th = inputs.proposals(cfg)
    d = inputs.make_data(cfg, oracle.waveform)
    a, pa, used1 = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, n_threads=1)
    b, pb, usedn = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, n_threads=4)
    assert used1 == 1 and usedn >= 1
    assert np.array_equal(a, b) and np.array_equal(pa, pb)
