"""P11: pins of the oracle's spin_order = 2 option (NEXT-1, reading A22): the
spin-orbit phase terms linear in the spins at 2.5PN, 3PN and 3.5PN.  They are not in PAPER.md (literature closed
forms); the pins reach them by routes that share nothing with the oracle's coding in (S_l, dS_l):
  P11a  stationary-phase re-derivation from the spin-orbit terms of the binding energy and of the flux through
        3.5PN (the route of P1b), as symbolic identities and numerically,
  P11b  the same coefficients in the (chi_s, chi_a) coding, exact rationals,
  P11c  equal masses / equal spins and single-spin special cases,
  P11d  zero spins: spin_order 2 == spin_order 0 bit for bit; spin_order 2 leaves phi_0..phi_4 of spin_order 1 alone,
  P11e  the phase against 40-digit arithmetic.
"""
import math
from fractions import Fraction as Fr

import mpmath as mp
import numpy as np
import pytest
import sympy as sp


# ----------------------------------------------------------------------------- P11a
def _so_phase_terms_from_energy_flux():
    """phi_k (constant part, ln v part) linear in the spins for k = 3, 5, 6, 7, from
         E = -(eta/2) v^2 sum e_k v^k,  F = (32/5) eta^2 v^10 sum f_k v^k
    with the non-spinning e_k, f_k of P1b and the spin-orbit pieces (S = S_l, D = delta Sigma_l):
      e3 = 14/3 S + 2 D          e5 = (11 - 61/9 eta) S + (3 - 10/3 eta) D
      e7 = (135/4 - 367/4 eta + 29/12 eta^2) S + (27/4 - 39 eta + 5/4 eta^2) D
      f3 = 4 pi - 4 S - 5/4 D    f5 += (-9/2 + 272/9 eta) S + (-13/16 + 43/4 eta) D
      f6 += -16 pi S - 31/6 pi D
      f7 += (476645/6804 + 6172/189 eta - 2810/27 eta^2) S + (9535/336 + 1849/126 eta - 1501/36 eta^2) D
    Psi = ... + (2/M) int_{v_f}^{v_c} (v_f^3 - v^3) E'(v)/F(v) dv; only the lower limit carries f-dependence."""
    R, pi, g = sp.Rational, sp.pi, sp.EulerGamma
    eta, S, D, lnv = sp.symbols("eta S D lnv")
    e = {0: 1, 2: -(R(3, 4) + eta / 12), 4: -(R(27, 8) - R(19, 8) * eta + eta ** 2 / 24),
         6: -(R(675, 64) - (R(34445, 576) - R(205, 96) * pi ** 2) * eta + R(155, 96) * eta ** 2 + R(35, 5184) * eta ** 3),
         3: R(14, 3) * S + 2 * D,
         5: (11 - R(61, 9) * eta) * S + (3 - R(10, 3) * eta) * D,
         7: (R(135, 4) - R(367, 4) * eta + R(29, 12) * eta ** 2) * S + (R(27, 4) - 39 * eta + R(5, 4) * eta ** 2) * D}
    f = {0: 1, 2: -(R(1247, 336) + R(35, 12) * eta),
         3: 4 * pi - 4 * S - R(5, 4) * D,
         4: -R(44711, 9072) + R(9271, 504) * eta + R(65, 18) * eta ** 2,
         5: -(R(8191, 672) + R(583, 24) * eta) * pi + (-R(9, 2) + R(272, 9) * eta) * S + (-R(13, 16) + R(43, 4) * eta) * D,
         6: (R(6643739519, 69854400) + R(16, 3) * pi ** 2 - R(1712, 105) * g
             + (-R(134543, 7776) + R(41, 48) * pi ** 2) * eta - R(94403, 3024) * eta ** 2 - R(775, 324) * eta ** 3
             - R(856, 105) * (sp.log(16) + 2 * lnv)) - 16 * pi * S - R(31, 6) * pi * D,
         7: (-R(16285, 504) + R(214745, 1728) * eta + R(193385, 3024) * eta ** 2) * pi
            + (R(476645, 6804) + R(6172, 189) * eta - R(2810, 27) * eta ** 2) * S
            + (R(9535, 336) + R(1849, 126) * eta - R(1501, 36) * eta ** 2) * D}
    N = 8
    de = [sp.expand(R(k + 2, 2) * e.get(k, 0)) for k in range(N)]
    fs = [f.get(k, 0) for k in range(N)]
    inv = [sp.Integer(1)] + [sp.Integer(0)] * (N - 1)
    for n in range(1, N):
        inv[n] = sp.expand(-sum(fs[k] * inv[n - k] for k in range(1, n + 1)))
    r = [sp.expand(sum(de[k] * inv[n - k] for k in range(n + 1))) for n in range(N)]

    def linear_in_spin(x):
        x = sp.expand(x)
        return sp.expand(x.coeff(S, 1).subs(D, 0) * S + x.coeff(D, 1).subs(S, 0) * D)

    def prim_at_vf(n, c, l):
        if n == -1:
            return sp.Integer(0), c
        m = R(1, n + 1)
        return c * m - l * m * m, l * m

    scale = 2 * (-R(5, 32)) / R(3, 128)
    out = {}
    for k in (3, 5, 6, 7):
        rk = linear_in_spin(r[k])
        c, l = rk.coeff(lnv, 0), rk.coeff(lnv, 1)
        a, b = prim_at_vf(k - 9, c, l), prim_at_vf(k - 6, c, l)
        out[k] = (sp.expand(scale * -(a[0] - b[0])), sp.expand(scale * -(a[1] - b[1])))
    return out, (eta, S, D)


@pytest.fixture(scope="module")
def so_terms():
    return _so_phase_terms_from_energy_flux()


def test_p11a_symbolic_identities(so_terms):
    out, (eta, S, D) = so_terms
    R, pi = sp.Rational, sp.pi
    gamma = (R(554345, 1134) + R(110, 9) * eta) * S + (R(13915, 84) - R(10, 3) * eta) * D
    assert sp.expand(out[3][0] - (R(188, 3) * S + 25 * D)) == 0 and out[3][1] == 0          # 4 beta
    assert sp.expand(out[5][0] + gamma) == 0 and sp.expand(out[5][1] + 3 * gamma) == 0
    assert sp.expand(out[6][0] - pi * (3760 * S + 1490 * D) / 3) == 0 and out[6][1] == 0
    want7 = ((-R(8980424995, 762048) + R(6586595, 756) * eta - R(305, 36) * eta ** 2) * S
             - (R(170978035, 48384) - R(2876425, 672) * eta - R(4735, 144) * eta ** 2) * D)
    assert sp.expand(out[7][0] - want7) == 0 and out[7][1] == 0


@pytest.mark.parametrize("q,chi1,chi2", [(0.8, 0.3, -0.2), (0.5, -0.7, 0.6), (1.0, 0.8, 0.8), (0.3, 0.0, 0.9)])
def test_p11a_oracle_against_the_rederivation(oracle, so_terms, q, chi1, chi2):
    out, (eta_s, S_s, D_s) = so_terms
    eta, mu1, mu2 = q / (1 + q) ** 2, 1 / (1 + q), q / (1 + q)
    subs = {eta_s: sp.Float(eta, 30), S_s: sp.Float(mu1 ** 2 * chi1 + mu2 ** 2 * chi2, 30),
            D_s: sp.Float((mu1 - mu2) * (mu2 * chi2 - mu1 * chi1), 30)}
    p1, l1 = oracle.phase_coefficients(eta, mu1, mu2, chi1, chi2, 1)
    p2, l2 = oracle.phase_coefficients(eta, mu1, mu2, chi1, chi2, 2)
    for k in (5, 6, 7):
        c = float(sp.N(out[k][0].subs(subs), 25))
        l = float(sp.N(out[k][1].subs(subs), 25))
        assert p2[k] - p1[k] == pytest.approx(c, rel=1e-12, abs=1e-12), k
        assert l2[k] - l1[k] == pytest.approx(l, rel=1e-12, abs=1e-12), k
    # the 1.5PN term the default already has follows from the same series (cross-check of the variables)
    p0, _ = oracle.phase_coefficients(eta, mu1, mu2, 0, 0, 0)
    assert p1[3] - p0[3] == pytest.approx(float(sp.N(out[3][0].subs(subs), 25)), rel=1e-12, abs=1e-12)


# ----------------------------------------------------------------------------- P11b
def _chis_chia_coding(q, chi1, chi2):
    """S_l = (1 - 2 eta) chi_s + delta chi_a,  dS_l = -(1 - 4 eta) chi_s - delta chi_a  (exact rationals)."""
    q, chi1, chi2 = Fr(q), Fr(chi1), Fr(chi2)
    eta, delta = q / (1 + q) ** 2, (1 - q) / (1 + q)
    xs, xa = (chi1 + chi2) / 2, (chi1 - chi2) / 2
    S = (1 - 2 * eta) * xs + delta * xa
    D = -(1 - 4 * eta) * xs - delta * xa
    gamma = (Fr(554345, 1134) + Fr(110, 9) * eta) * S + (Fr(13915, 84) - Fr(10, 3) * eta) * D
    six = (3760 * S + 1490 * D) / 3                                           # times pi
    seven = ((-Fr(8980424995, 762048) + Fr(6586595, 756) * eta - Fr(305, 36) * eta ** 2) * S
             - (Fr(170978035, 48384) - Fr(2876425, 672) * eta - Fr(4735, 144) * eta ** 2) * D)
    return float(-gamma), float(six) * math.pi, float(seven)


@pytest.mark.parametrize("q,chi1,chi2", [(Fr(4, 5), Fr(3, 10), Fr(-1, 5)), (Fr(1, 2), Fr(-7, 10), Fr(3, 5)),
                                         (Fr(1), Fr(4, 5), Fr(-4, 5)), (Fr(7, 10), Fr(1, 20), Fr(0))])
def test_p11b_two_codings(oracle, q, chi1, chi2):
    eta, mu1, mu2 = float(q / (1 + q) ** 2), float(1 / (1 + q)), float(q / (1 + q))
    p1, l1 = oracle.phase_coefficients(eta, mu1, mu2, float(chi1), float(chi2), 1)
    p2, l2 = oracle.phase_coefficients(eta, mu1, mu2, float(chi1), float(chi2), 2)
    d5, d6, d7 = _chis_chia_coding(q, chi1, chi2)
    assert p2[5] - p1[5] == pytest.approx(d5, rel=1e-12, abs=1e-12)
    assert l2[5] - l1[5] == pytest.approx(3 * d5, rel=1e-12, abs=1e-12)
    assert p2[6] - p1[6] == pytest.approx(d6, rel=1e-12, abs=1e-12)
    assert p2[7] - p1[7] == pytest.approx(d7, rel=1e-12, abs=1e-12)


# ----------------------------------------------------------------------------- P11c / P11d
def test_p11c_equal_mass_equal_spin(oracle):
    """eta = 1/4, chi1 = chi2 = chi: S_l = chi/2, dS_l = 0."""
    chi = 0.6
    p1, l1 = oracle.phase_coefficients(0.25, 0.5, 0.5, chi, chi, 1)
    p2, l2 = oracle.phase_coefficients(0.25, 0.5, 0.5, chi, chi, 2)
    g = (554345 / 1134 + 110 / 36) * chi / 2
    assert p2[5] - p1[5] == pytest.approx(-g, rel=1e-13)
    assert p2[6] - p1[6] == pytest.approx(math.pi * 3760 / 3 * chi / 2, rel=1e-13)
    assert p2[7] - p1[7] == pytest.approx((-8980424995 / 762048 + 6586595 / 3024 - 305 / 576) * chi / 2, rel=1e-13)
    # antisymmetric spins on equal masses: S_l = 0 and delta = 0, nothing changes
    a1 = oracle.phase_coefficients(0.25, 0.5, 0.5, chi, -chi, 1)
    a2 = oracle.phase_coefficients(0.25, 0.5, 0.5, chi, -chi, 2)
    assert np.allclose(a1[0], a2[0], rtol=0, atol=1e-12) and np.allclose(a1[1], a2[1], rtol=0, atol=1e-12)


def test_p11d_reductions(oracle):
    for q in (1.0, 0.6, 0.25):
        eta, mu1, mu2 = q / (1 + q) ** 2, 1 / (1 + q), q / (1 + q)
        z0 = oracle.phase_coefficients(eta, mu1, mu2, 0.0, 0.0, 0)
        z2 = oracle.phase_coefficients(eta, mu1, mu2, 0.0, 0.0, 2)
        assert np.array_equal(z0[0], z2[0]) and np.array_equal(z0[1], z2[1])
        s1 = oracle.phase_coefficients(eta, mu1, mu2, 0.4, -0.3, 1)
        s2 = oracle.phase_coefficients(eta, mu1, mu2, 0.4, -0.3, 2)
        assert np.array_equal(s1[0][:5], s2[0][:5]) and np.array_equal(s1[1][:5], s2[1][:5])
        assert s2[1][5] - s1[1][5] == pytest.approx(3 * (s2[0][5] - s1[0][5]), rel=1e-13)
        assert s2[1][6] == s1[1][6] and s2[1][7] == s1[1][7] == 0.0


# ----------------------------------------------------------------------------- P11e
def test_p11e_phase_against_40_digits(oracle):
    """Psi(spin_order 2) - Psi(spin_order 1) vs the (chi_s, chi_a) coding evaluated in 40-digit arithmetic."""
    mp.mp.dps = 40
    rng = np.random.default_rng(12)
    tsun = mp.mpf("1.3271244e20") / mp.mpf(299792458) ** 3
    for i in range(100):
        bns = i % 2 == 0
        theta = np.array([rng.uniform(1.1, 1.3) if bns else rng.uniform(20, 40), rng.uniform(0.5, 1),
                          rng.uniform(-0.8, 0.8), rng.uniform(-0.8, 0.8), 100.0, rng.uniform(-0.1, 0.1),
                          rng.uniform(0, 6.28), 0.3, 0, 0, 0])
        f = float(rng.uniform(10, 2048))
        mc, q, chi1, chi2 = [mp.mpf(float(x)) for x in theta[:4]]
        eta, delta = q / (1 + q) ** 2, (1 - q) / (1 + q)
        xs, xa = (chi1 + chi2) / 2, (chi1 - chi2) / 2
        S = (1 - 2 * eta) * xs + delta * xa
        D = -(1 - 4 * eta) * xs - delta * xa
        r = lambda a, b: mp.mpf(a) / mp.mpf(b)
        gamma = (r(554345, 1134) + r(110, 9) * eta) * S + (r(13915, 84) - r(10, 3) * eta) * D
        six = mp.pi * (3760 * S + 1490 * D) / 3
        seven = ((-r(8980424995, 762048) + r(6586595, 756) * eta - r(305, 36) * eta ** 2) * S
                 - (r(170978035, 48384) - r(2876425, 672) * eta - r(4735, 144) * eta ** 2) * D)
        v = mp.cbrt(mp.pi * mc * eta ** (mp.mpf(-3) / 5) * tsun * mp.mpf(f))
        want = 3 / (128 * eta) * (-gamma * (1 + 3 * mp.log(v)) + six * v + seven * v ** 2)
        full = oracle.phase([f], theta, 2)[0]
        base = oracle.phase([f], theta, 1)[0]
        err = abs(float(mp.mpf(full) - mp.mpf(base) - want))
        assert err < 32 * np.spacing(abs(base)) + 1e-13, (theta, f, err)
        assert abs(float(want)) > 1e-6
