"""Pins for the oracle's amplitude, detector response and waveform
(SURVEY.md 8(c) pins P2, P4, P5, P6, P9; readings A3, A12, A13 of DESIGN.md).
"""
import math

import numpy as np
import pytest
from scipy import integrate

from paper_1904_02863_b200 import inputs

C_SI = 299792458.0


def _theta(**kw):
    th = dict(mc=28.0, q=0.8, chi1=0.3, chi2=-0.2, dl=500.0, tc=0.01, phic=1.3, cosi=0.8, ra=1.0, dec=-0.5, psi=0.7)
    th.update(kw)
    return np.array([th[k] for k in ("mc", "q", "chi1", "chi2", "dl", "tc", "phic", "cosi", "ra", "dec", "psi")])


# ----------------------------------------------------------------------------- constants / amplitude
def test_constants_from_exact_definitions(oracle):
    c = oracle.constants()
    assert c["tsun_s"] == pytest.approx(4.9254909476412675e-6, rel=1e-15)
    assert c["mpc_s"] == pytest.approx(1.02927125054339e14, rel=1e-14)


def test_amplitude_anchor_and_scaling(oracle):
    """A0(28, 500) = 2.5087222601e-21 (SURVEY.md scale table); A0 ~ Mc^(5/6) / D."""
    assert oracle.amplitude(28.0, 500.0) == pytest.approx(2.5087222601e-21, rel=1e-10)
    assert oracle.amplitude(1.2, 100.0) == pytest.approx(9.0874e-22, rel=1e-4)
    assert oracle.amplitude(28.0, 1000.0) == pytest.approx(oracle.amplitude(28.0, 500.0) / 2, rel=1e-15)
    assert oracle.amplitude(56.0, 500.0) / oracle.amplitude(28.0, 500.0) == pytest.approx(2 ** (5 / 6), rel=1e-14)
    # closed form from SI quantities: sqrt(5/24) pi^(-2/3) c (G Mc/c^3)^(5/6) / D
    gm, mpc = 1.3271244e20, 1e6 * 648000 / math.pi * 149597870700.0
    a0 = math.sqrt(5 / 24) * math.pi ** (-2 / 3) * C_SI * (gm * 28 / C_SI ** 3) ** (5 / 6) / (500 * mpc)
    assert oracle.amplitude(28.0, 500.0) == pytest.approx(a0, rel=1e-14)


# ----------------------------------------------------------------------------- P2
@pytest.mark.parametrize("name", ["C0", "C1"])
def test_p2_hh_closed_form(oracle, name):
    """<h|h>_I = |C_I|^2 A0^2 I7_I exactly (phase-independent), and the optimal SNR anchor 108.05 (C0)."""
    cfg = inputs.CONFIGS[name]
    f, S, dets = inputs.frequency_grid(cfg), inputs.psd(cfg), inputs.detectors(cfg)
    th = np.array(cfg.theta_inj)
    zero = np.zeros((cfg.n_det, cfg.n_bins), complex)
    _, parts, _ = oracle.lnl(f, cfg.delta_f, zero, S, dets, cfg.gmst, th[None], cfg.spin_order)
    a0 = oracle.amplitude(th[0], th[4])
    i7 = oracle.norm_i7(f, cfg.delta_f, S[0])
    for i in range(cfg.n_det):
        fp, fc, _ = oracle.antenna(dets[i], th[8], th[9], th[10], cfg.gmst)
        c2 = (fp * 0.5 * (1 + th[7] ** 2)) ** 2 + (fc * th[7]) ** 2
        assert parts[0, i, 2] == pytest.approx(c2 * a0 * a0 * i7, rel=1e-12)
    if name == "C0":
        assert math.sqrt(parts[0, 0, 2]) == pytest.approx(108.05, abs=0.01)


@pytest.mark.parametrize("name,i7_printed,cont_printed", [
    ("C0", 1.854949528061384e45, 1.854819320630977e45),
    ("C1", 1.862160879773427e45, 1.8619081818397986e45),
    ("C3", 1.8742017960336145e45, 1.8742012400193934e45),
])
def test_p2_i7_against_quadrature(oracle, name, i7_printed, cont_printed):
    """I7 = 4 df sum f^(-7/3)/S against adaptive quadrature of 4 int f^(-7/3)/S df (trapezoid-corrected, 1e-6)."""
    cfg = inputs.CONFIGS[name]
    f = inputs.frequency_grid(cfg)
    S = inputs.analytic_psd(f)
    i7 = oracle.norm_i7(f, cfg.delta_f, S)
    assert i7 == pytest.approx(i7_printed, rel=1e-13)
    integrand = lambda x: x ** (-7.0 / 3.0) / inputs.analytic_psd(np.array([x]))[0]
    # break the interval so that the steep low-frequency end is resolved
    edges = [cfg.f_min, 30, 60, 120, 250, 500, 1000, cfg.f_max]
    edges = [e for e in edges if cfg.f_min <= e <= cfg.f_max]
    cont = 4 * sum(integrate.quad(integrand, a, b, epsabs=0, epsrel=1e-12, limit=200)[0]
                   for a, b in zip(edges[:-1], edges[1:]))
    assert cont == pytest.approx(cont_printed, rel=1e-9)
    ends = 0.5 * 4 * cfg.delta_f * (integrand(f[0]) + integrand(f[-1]))
    assert (i7 - ends) == pytest.approx(cont, rel=1e-6)


# ----------------------------------------------------------------------------- P4
def test_p4_modulus_and_shift_identities(oracle):
    cfg = inputs.CONFIGS["C1"].reduced(f_max=256.0)
    f, dets = inputs.frequency_grid(cfg), inputs.detectors(cfg)
    th = _theta()
    h = oracle.waveform(f, dets, cfg.gmst, th[None])[0]
    a0 = oracle.amplitude(th[0], th[4])
    for i in range(3):
        fp, fc, _ = oracle.antenna(dets[i], th[8], th[9], th[10], cfg.gmst)
        cmod = math.hypot(fp * 0.5 * (1 + th[7] ** 2), fc * th[7])
        np.testing.assert_allclose(np.abs(h[i]), cmod * a0 * f ** (-7 / 6), rtol=1e-13)
    tau, alpha = 0.003, 0.9
    h_t = oracle.waveform(f, dets, cfg.gmst, _theta(tc=0.01 + tau)[None])[0]
    h_p = oracle.waveform(f, dets, cfg.gmst, _theta(phic=1.3 + alpha)[None])[0]
    scale = np.abs(h).max()
    # h(tc + tau) = h(tc) exp(-2 pi i f tau)   (PAPER.md:69 sign), h(phic + a) = h(phic) exp(+i a)
    assert np.abs(h_t - h * np.exp(-2j * np.pi * f * tau)).max() < 1e-11 * scale
    assert np.abs(h_p - h * np.exp(1j * alpha)).max() < 1e-12 * scale


def test_p4_tc_and_fixed_delay_are_interchangeable(oracle):
    """A FIXED detector with dt = tau equals t_c -> t_c + tau (reading A3: the shifts add)."""
    f = np.linspace(20, 200, 721)
    th = _theta(cosi=1.0)
    tau = 0.0123
    h_a = oracle.waveform(f, inputs.fixed_detector(1.0, 0.0, tau)[None], 0.0, th[None], 0)[0, 0]
    h_b = oracle.waveform(f, inputs.fixed_detector(1.0, 0.0, 0.0)[None], 0.0, _theta(cosi=1.0, tc=0.01 + tau)[None], 0)[0, 0]
    assert np.abs(h_a - h_b).max() < 1e-11 * np.abs(h_a).max()


def test_polarisation_content(oracle):
    """O5: h+ = (1+cos^2 i)/2 h0, hx = -i cos i h0, read off with FIXED detectors (F+,Fx) = (1,0), (0,1)."""
    f = np.linspace(20, 100, 161)
    th = _theta(cosi=0.37)
    hp = oracle.waveform(f, inputs.fixed_detector(1, 0, 0)[None], 0.0, th[None])[0, 0]
    hc = oracle.waveform(f, inputs.fixed_detector(0, 1, 0)[None], 0.0, th[None])[0, 0]
    h0 = hp / (0.5 * (1 + 0.37 ** 2))
    np.testing.assert_allclose(hc, -1j * 0.37 * h0, rtol=1e-13)
    # h0 = A0 f^(-7/6) exp(-i Psi)
    psi = oracle.phase(f, th)
    want = oracle.amplitude(th[0], th[4]) * f ** (-7 / 6) * np.exp(-1j * psi)
    np.testing.assert_allclose(h0, want, rtol=1e-12)


# ----------------------------------------------------------------------------- P5
def test_p5_sky_frame_is_orthonormal_and_left_handed_about_n(oracle):
    rng = np.random.default_rng(5)
    for _ in range(50):
        ra, dec, psi, gmst = rng.uniform(0, 2 * np.pi), np.arcsin(rng.uniform(-1, 1)), rng.uniform(0, np.pi), rng.uniform(0, 2 * np.pi)
        X, Y, n = oracle.sky_frame(ra, dec, psi, gmst)
        for a in (X, Y, n):
            assert np.dot(a, a) == pytest.approx(1.0, abs=1e-14)
        assert abs(np.dot(X, Y)) < 1e-14 and abs(np.dot(X, n)) < 1e-14 and abs(np.dot(Y, n)) < 1e-14
        np.testing.assert_allclose(np.cross(X, Y), -n, atol=1e-14)   # X x Y = propagation direction


def test_p5_antenna_invariants(oracle):
    rng = np.random.default_rng(6)
    for name in ("H1", "L1", "V1"):
        det = inputs.geometric_detector(name)
        for _ in range(20):
            ra, dec, psi, gmst = rng.uniform(0, 2 * np.pi), np.arcsin(rng.uniform(-1, 1)), rng.uniform(0, np.pi), rng.uniform(0, 2 * np.pi)
            fp, fc, _ = oracle.antenna(det, ra, dec, psi, gmst)
            fp2, fc2, _ = oracle.antenna(det, ra, dec, psi + 0.4, gmst)
            assert fp * fp + fc * fc == pytest.approx(fp2 * fp2 + fc2 * fc2, abs=1e-14)   # psi-independent
            assert fp * fp + fc * fc <= 1.0 + 1e-6
            fp3, fc3, _ = oracle.antenna(det, ra, dec, psi + np.pi / 2, gmst)
            assert fp3 == pytest.approx(-fp, abs=1e-14) and fc3 == pytest.approx(-fc, abs=1e-14)
            # rotating psi by a rotates (F+, Fx) by 2a
            a = 0.4
            assert fp2 == pytest.approx(fp * math.cos(2 * a) + fc * math.sin(2 * a), abs=1e-13) or \
                   fp2 == pytest.approx(fp * math.cos(2 * a) - fc * math.sin(2 * a), abs=1e-13)
            # only gmst - ra matters
            fp4, fc4, dt4 = oracle.antenna(det, ra + 0.3, dec, psi, gmst + 0.3)
            assert (fp4, fc4) == (pytest.approx(fp, abs=1e-13), pytest.approx(fc, abs=1e-13))


def test_p5_closed_form_overhead_source(oracle):
    """Arms x=(1,0,0), y=(0,1,0), dec = pi/2:  F+ = -cos 2(psi+gmst-ra),  Fx = sin 2(psi+gmst-ra)."""
    det = np.zeros(13)
    det[4:7], det[7:10] = (1, 0, 0), (0, 1, 0)
    for ra, psi, gmst in ((0.3, 0.2, 1.1), (2.0, 1.3, 0.4), (5.5, 2.9, 6.0)):
        fp, fc, dt = oracle.antenna(det, ra, np.pi / 2, psi, gmst)
        a = psi + gmst - ra
        assert fp == pytest.approx(-math.cos(2 * a), abs=1e-14)
        assert fc == pytest.approx(math.sin(2 * a), abs=1e-14)
        assert dt == 0.0


def test_p5_h1_anchor(oracle):
    """SURVEY.md scale table: H1, ra=1, dec=-0.5, psi=0.7, gmst=2."""
    fp, fc, dt = oracle.antenna(inputs.geometric_detector("H1"), 1.0, -0.5, 0.7, 2.0)
    assert fp == pytest.approx(0.408881419111625, abs=1e-14)
    assert fc == pytest.approx(0.151248654198486, abs=1e-14)
    assert dt == pytest.approx(1.32962525135725e-3, rel=1e-13)


# ----------------------------------------------------------------------------- P6
def test_p6_delays_bounded_by_light_travel_times(oracle):
    dets = {n: inputs.geometric_detector(n) for n in ("H1", "L1", "V1")}
    rng = np.random.default_rng(8)
    for _ in range(200):
        ra, dec = rng.uniform(0, 2 * np.pi), np.arcsin(rng.uniform(-1, 1))
        dt = {n: oracle.antenna(d, ra, dec, 0.3, 1.0)[2] for n, d in dets.items()}
        for n, d in dets.items():
            assert abs(dt[n]) <= np.linalg.norm(d[1:4]) / C_SI * (1 + 1e-14)
        for a, b in (("H1", "L1"), ("H1", "V1"), ("L1", "V1")):
            base = np.linalg.norm(dets[a][1:4] - dets[b][1:4]) / C_SI
            assert abs(dt[a] - dt[b]) <= base * (1 + 1e-13)
    # equality when n is parallel to the baseline; the detector nearer the source hears it first (A13)
    base = dets["H1"][1:4] - dets["L1"][1:4]
    n = base / np.linalg.norm(base)            # source in the direction from L1 towards H1
    dec, ra = math.asin(n[2]), math.atan2(n[1], n[0])
    d_h = oracle.antenna(dets["H1"], ra, dec, 0.0, 0.0)[2]
    d_l = oracle.antenna(dets["L1"], ra, dec, 0.0, 0.0)[2]
    assert d_l - d_h == pytest.approx(np.linalg.norm(base) / C_SI, rel=1e-12)
    assert d_h < d_l


# ----------------------------------------------------------------------------- P9
def test_p9_bin_independence(oracle):
    """'the value at each frequency can be evaluated independently' -- bitwise in the oracle."""
    cfg = inputs.CONFIGS["C1"].reduced(f_max=128.0)
    f, dets = inputs.frequency_grid(cfg), inputs.detectors(cfg)
    th = inputs.proposals(cfg, 3)
    full = oracle.waveform(f, dets, cfg.gmst, th)
    sub = oracle.waveform(f[100:150], dets, cfg.gmst, th)
    assert np.array_equal(full[:, :, 100:150], sub)
    perm = np.random.default_rng(1).permutation(f.shape[0])
    assert np.array_equal(oracle.waveform(f[perm], dets, cfg.gmst, th), full[:, :, perm])
