"""P10: pins of the oracle's tidal option (NEXT-1, reading A21).

The tidal phase terms are not in PAPER.md (the paper's motivation names the neutron-star equation of state,
PAPER.md:11); the oracle codes the literature closed form in the (Lambda~, dLambda~) variables.  The pins reach
the same numbers by routes that share nothing with that coding:
  P10a  the per-body form of the same terms (another algebraic coding, exact rationals),
  P10b  a stationary-phase re-derivation from the tidal corrections to the binding energy and the flux,
  P10c  equal masses, equal Lambda: Lambda~ = Lambda, dLambda~ = 0,
  P10d  Lambda = 0 and tidal_order = 0 reduce to the point-mass results bit for bit,
  P10e  the phase with tidal terms against 40-digit arithmetic on the per-body form,
  P10f  waveform / lnL entry points: the tidal terms change the phase only (|h| unchanged, <h|h> unchanged).
"""
import math
from fractions import Fraction as Fr

import mpmath as mp
import numpy as np
import pytest
import sympy as sp

from paper_1904_02863_b200 import inputs


def _per_body(q, lam1, lam2):
    """phi_10, phi_12 as exact rationals: sum over bodies with X_A = m_A/M,
    phi_10 = -24 (12 - 11 X) X^4 Lambda,  phi_12 = -(5/28)(3179 - 919 X - 2286 X^2 + 260 X^3) X^4 Lambda."""
    q, lam1, lam2 = Fr(q), Fr(lam1), Fr(lam2)
    p10 = p12 = Fr(0)
    for x, lam in ((1 / (1 + q), lam1), (q / (1 + q), lam2)):
        p10 += -24 * (12 - 11 * x) * x ** 4 * lam
        p12 += -Fr(5, 28) * (3179 - 919 * x - 2286 * x ** 2 + 260 * x ** 3) * x ** 4 * lam
    return p10, p12


@pytest.mark.parametrize("q,lam1,lam2", [(Fr(1), 400, 400), (Fr(7, 10), 300, 900), (Fr(1, 2), 100, 2500),
                                         (Fr(9, 10), 0, 1000), (Fr(4, 5), 5000, 0), (Fr(3, 4), 1, 1)])
def test_p10a_two_codings(oracle, q, lam1, lam2):
    eta = float(q / (1 + q) ** 2)
    got10, got12 = oracle.tidal_coefficients(eta, lam1, lam2, 2)
    want10, want12 = _per_body(q, lam1, lam2)
    assert got10 == pytest.approx(float(want10), rel=1e-13)
    assert got12 == pytest.approx(float(want12), rel=1e-13)
    only5 = oracle.tidal_coefficients(eta, lam1, lam2, 1)
    assert only5[0] == got10 and only5[1] == 0.0


# ----------------------------------------------------------------------------- P10b
def _spa_tidal_from_energy_flux():
    """Stationary-phase tidal coefficients from the tidal corrections to E(v) and F(v), one body of mass
    fraction X and deformability Lambda (the companion's contribution follows by X -> 1 - X).

    E = -(eta/2) v^2 [1 + e2 v^2 + e10 v^10 + e12 v^12],  F = (32/5) eta^2 v^10 [1 + f2 v^2 + f10 v^10 + f12 v^12],
    with lam = Lambda X^5 (= lambda_A/M^5) and X_B = 1 - X:
      e10 = -9 (X_B/X) lam                       e12 = -(11/2)(X_B/X)(3 + 2 X + 3 X^2) lam
      f10 = (18 - 12 X)/X lam                    f12 = -(704 + 1803 X - 4501 X^2 + 2170 X^3)/(28 X) lam
    Same integral as tests/test_oracle_phase.py P1b: a term r_n v^n of (E'/F)/(its Newtonian value) gives
    phi_n = 40 r_n / ((n-5)(n-8)) in units of 3/(128 eta) v^(n-5)  (n != 5, 8).  Returns (phi_10, phi_12, X, Lambda).
    """
    X, Lam = sp.symbols("X Lambda", positive=True)
    R = sp.Rational
    eta = X * (1 - X)
    lam = Lam * X ** 5
    xb = 1 - X
    e = {0: sp.Integer(1), 2: -(R(3, 4) + eta / 12),
         10: -9 * xb / X * lam, 12: -R(11, 2) * xb / X * (3 + 2 * X + 3 * X ** 2) * lam}
    f = {0: sp.Integer(1), 2: -(R(1247, 336) + R(35, 12) * eta),
         10: (18 - 12 * X) / X * lam, 12: -(704 + 1803 * X - 4501 * X ** 2 + 2170 * X ** 3) / (28 * X) * lam}
    N = 13
    de = [sp.expand(R(k + 2, 2) * e.get(k, 0)) for k in range(N)]        # E' = -eta v sum (k+2)/2 e_k v^k
    fs = [f.get(k, 0) for k in range(N)]
    inv = [sp.Integer(1)] + [sp.Integer(0)] * (N - 1)                     # 1 / sum f_k v^k
    for n in range(1, N):
        inv[n] = sp.expand(-sum(fs[k] * inv[n - k] for k in range(1, n + 1)))
    r = [sp.expand(sum(de[k] * inv[n - k] for k in range(n + 1))) for n in range(N)]
    lin = lambda expr: sp.expand(expr).coeff(Lam, 1) * Lam                 # the part linear in Lambda
    phi10 = sp.simplify(R(40, (10 - 5) * (10 - 8)) * lin(r[10]))
    phi12 = sp.simplify(R(40, (12 - 5) * (12 - 8)) * lin(r[12]))
    return phi10, phi12, X, Lam


def test_p10b_rederivation_from_tidal_energy_and_flux(oracle):
    phi10, phi12, X, Lam = _spa_tidal_from_energy_flux()
    # the closed forms the two codings of P10a state, now as polynomial identities in X
    assert sp.simplify(phi10 + 24 * (12 - 11 * X) * X ** 4 * Lam) == 0
    assert sp.simplify(phi12 + sp.Rational(5, 28) * (3179 - 919 * X - 2286 * X ** 2 + 260 * X ** 3) * X ** 4 * Lam) == 0
    # and numerically against the oracle, both bodies
    for q, lam1, lam2 in ((0.8, 500.0, 800.0), (0.55, 90.0, 3000.0), (1.0, 250.0, 750.0)):
        eta = q / (1 + q) ** 2
        x1, x2 = 1 / (1 + q), q / (1 + q)
        want10 = float(phi10.subs({X: x1, Lam: lam1}) + phi10.subs({X: x2, Lam: lam2}))
        want12 = float(phi12.subs({X: x1, Lam: lam1}) + phi12.subs({X: x2, Lam: lam2}))
        got10, got12 = oracle.tidal_coefficients(eta, lam1, lam2, 2)
        assert got10 == pytest.approx(want10, rel=1e-12)
        assert got12 == pytest.approx(want12, rel=1e-12)


# ----------------------------------------------------------------------------- P10c / P10d
def test_p10c_equal_mass_equal_lambda(oracle):
    """Lambda~ = Lambda and dLambda~ = 0: phi_10 = -(39/2) Lambda, phi_12 = -(3115/64) Lambda."""
    for lam in (1.0, 400.0, 5000.0):
        p10, p12 = oracle.tidal_coefficients(0.25, lam, lam, 2)
        assert p10 == pytest.approx(-19.5 * lam, rel=1e-15)
        assert p12 == pytest.approx(-3115.0 / 64.0 * lam, rel=1e-15)


def test_p10c_sign_and_size(oracle):
    """Tides speed the inspiral up: the tidal phase is negative, grows as f^(5/3) at 5PN, and for Lambda~ = 400,
    M = 2.7 Msun at 1 kHz it is -(3/32)(39/2) 400 v^5 = a few radians."""
    th = np.array([2.7 * 0.25 ** 0.6, 1.0, 0, 0, 100.0, 0, 0, 1, 0, 0, 0])
    f = np.array([500.0, 1000.0])
    d5 = oracle.phase(f, th, 0, lambdas=[400, 400], tidal_order=1) - oracle.phase(f, th, 0)
    assert np.all(d5 < 0)
    assert d5[1] / d5[0] == pytest.approx(2 ** (5 / 3), rel=1e-9)
    v = (math.pi * 2.7 * oracle.constants()["tsun_s"] * 1000.0) ** (1 / 3)
    assert d5[1] == pytest.approx(-(3 / 32) * 19.5 * 400 * v ** 5, rel=1e-9)
    assert -10 < d5[1] < -1


def test_p10d_reduces_to_point_mass(oracle):
    cfg = inputs.CONFIGS["C2"]
    th = inputs.proposals(cfg, 4)
    f = np.linspace(20, 2048, 257)
    for b in range(4):
        base = oracle.phase(f, th[b], 1)
        assert np.array_equal(base, oracle.phase(f, th[b], 1, lambdas=[0.0, 0.0], tidal_order=2))
        assert np.array_equal(base, oracle.phase(f, th[b], 1, lambdas=[300.0, 500.0], tidal_order=0))


# ----------------------------------------------------------------------------- P10e
def _mp_tidal_phase(f, theta, lam1, lam2):
    """Tidal part of the phase in 40-digit arithmetic from the per-body form (not the oracle's coding)."""
    mp.mp.dps = 40
    mc, q = mp.mpf(float(theta[0])), mp.mpf(float(theta[1]))
    tsun = mp.mpf("1.3271244e20") / mp.mpf(299792458) ** 3
    eta = q / (1 + q) ** 2
    ms = mc * eta ** (mp.mpf(-3) / 5) * tsun
    v = mp.cbrt(mp.pi * ms * mp.mpf(float(f)))
    p10 = p12 = mp.mpf(0)
    for x, lam in ((1 / (1 + q), mp.mpf(float(lam1))), (q / (1 + q), mp.mpf(float(lam2)))):
        p10 += -24 * (12 - 11 * x) * x ** 4 * lam
        p12 += -mp.mpf(5) / 28 * (3179 - 919 * x - 2286 * x ** 2 + 260 * x ** 3) * x ** 4 * lam
    return 3 / (128 * eta) * (p10 * v ** 5 + p12 * v ** 7)


def test_p10e_phase_against_40_digits(oracle):
    """Oracle phase with tidal terms minus its point-mass phase vs the 40-digit tidal part.  The difference of two
    phases of size |Psi| carries their rounding (a few ulp of |Psi|, see P7), so that is the bound."""
    rng = np.random.default_rng(11)
    for _ in range(100):
        theta = np.array([rng.uniform(1.1, 1.3), rng.uniform(0.7, 1), rng.uniform(-0.05, 0.05),
                          rng.uniform(-0.05, 0.05), 100.0, rng.uniform(-0.1, 0.1), rng.uniform(0, 6.28),
                          0.3, 0, 0, 0])
        lam = rng.uniform(0, 5000, 2)
        f = float(rng.uniform(10, 2048))
        full = oracle.phase([f], theta, 1, lambdas=lam, tidal_order=2)[0]
        base = oracle.phase([f], theta, 1)[0]
        want = _mp_tidal_phase(f, theta, lam[0], lam[1])
        err = abs(float(mp.mpf(full) - mp.mpf(base) - want))
        assert err < 32 * np.spacing(abs(base)) + 1e-13, (theta, lam, f, err)
        assert abs(float(want)) > 1e-4          # not vacuous


# ----------------------------------------------------------------------------- P10f
def test_p10f_tides_change_the_phase_only(oracle):
    """|h(f)| and <h|h> do not depend on Lambda; h picks up exactly exp(-i dPsi_tidal); <d|h> changes."""
    cfg = inputs.CONFIGS["C2"].reduced(f_max=276.0, duration_s=2.0, batch=6)
    f = inputs.frequency_grid(cfg)
    dets = inputs.detectors(cfg)
    th = inputs.proposals(cfg)
    lam = inputs.tidal_lambdas(cfg)
    h0 = oracle.waveform(f, dets, cfg.gmst, th, 1)
    h2 = oracle.waveform(f, dets, cfg.gmst, th, 1, lambdas=lam, tidal_order=2)
    assert np.allclose(np.abs(h2), np.abs(h0), rtol=1e-13, atol=0)
    for b in range(th.shape[0]):
        dpsi = np.array([float(_mp_tidal_phase(fj, th[b], lam[b, 0], lam[b, 1])) for fj in f[::37]])
        ratio = h2[b, :, ::37] / h0[b, :, ::37]
        assert np.allclose(ratio, np.exp(-1j * dpsi)[None, :], rtol=0, atol=2e-11)
    data = inputs.make_data(cfg, oracle.waveform)
    S = inputs.psd(cfg)
    l0, p0, _ = oracle.lnl(f, cfg.delta_f, data, S, dets, cfg.gmst, th, 1)
    l2, p2, _ = oracle.lnl(f, cfg.delta_f, data, S, dets, cfg.gmst, th, 1, lambdas=lam, tidal_order=2)
    assert np.allclose(p2[..., 2], p0[..., 2], rtol=1e-13)
    # definition check: lnL from the tidal waveform by the plain inner product
    for b in (0, 3):
        tot = 0.0
        for i in range(cfg.n_det):
            dh = oracle.inner(cfg.delta_f, data[i], h2[b, i], S[i])
            hh = oracle.inner(cfg.delta_f, h2[b, i], h2[b, i], S[i])
            assert p2[b, i, 0] == pytest.approx(dh.real, rel=1e-12, abs=1e-12 * abs(hh.real))
            tot += dh.real - 0.5 * hh.real
        assert l2[b] == pytest.approx(tot, rel=1e-12)
    # lambdas = 0 reproduces the point-mass numbers bit for bit
    lz, pz, _ = oracle.lnl(f, cfg.delta_f, data, S, dets, cfg.gmst, th, 1, lambdas=np.zeros_like(lam), tidal_order=2)
    assert np.array_equal(lz, l0) and np.array_equal(pz, p0)
