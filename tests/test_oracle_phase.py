"""Pins for the oracle's TaylorF2 phase (SURVEY.md 8(c) pins P1a-P1d, P7).

PAPER.md gives no waveform formula (PAPER.md:43 names TaylorF2 only); BASELINE.json's
north_star fixes "TaylorF2 3.5PN phase, Newtonian amplitude, 1.5PN spin-orbit, 2PN
spin-spin".  These tests pin oracle/gw_oracle.c to things other than itself:
exact rationals, an independent stationary-phase derivation from the 3.5PN energy and
flux series, the Newtonian chirp time, two further codings of the spin terms, and
40-digit arithmetic.
"""
import math
from fractions import Fraction as Fr

import mpmath as mp
import numpy as np
import pytest
import sympy as sp


# ----------------------------------------------------------------------------- P1a
def test_p1a_anchor_values(oracle):
    """30-digit anchors printed in SURVEY.md 8(c) scale table (eta = 1/4 and 1/5, no spin)."""
    phi, phil = oracle.phase_coefficients(0.25, 0.5, 0.5, 0, 0, 0)
    want = [1.0, 0.0, 6.4417989417989418, -50.265482457436692, 46.245886085915848,
            154.91874884368716, -1104.1231610823976, 1130.8942020382669]
    np.testing.assert_allclose(phi, want, rtol=2e-15, atol=0)
    np.testing.assert_allclose(phil, [0, 0, 0, 0, 0, 464.75624653106148, -326.09523809523810, 0],
                               rtol=2e-15, atol=0)
    # eta = 0.2  <=>  q = (3 - sqrt 5)/2
    q = (3 - math.sqrt(5)) / 2
    phi, phil = oracle.phase_coefficients(0.2, 1 / (1 + q), q / (1 + q), 0, 0, 0)
    want = [1.0, 0.0, 6.1362433862433862, -50.265482457436692, 42.588867236709499,
            156.05321285748347, -938.94537636835636, 1098.4939825262963]
    np.testing.assert_allclose(phi, want, rtol=2e-15, atol=0)
    np.testing.assert_allclose(phil[5], 468.15963857245042, rtol=2e-15)


def test_p1a_exact_rationals(oracle):
    """The rational parts, in exact arithmetic, at a rational eta."""
    eta = Fr(2, 9)  # q = 1/2
    q = 0.5
    phi, phil = oracle.phase_coefficients(float(eta), 1 / (1 + q), q / (1 + q), 0, 0, 0)
    assert phi[0] == 1.0 and phi[1] == 0.0
    assert phi[2] == pytest.approx(float(Fr(3715, 756) + Fr(55, 9) * eta), rel=2e-16)
    assert phi[4] == pytest.approx(float(Fr(15293365, 508032) + Fr(27145, 504) * eta + Fr(3085, 72) * eta ** 2),
                                   rel=4e-16)
    assert phi[5] / math.pi == pytest.approx(float(Fr(38645, 756) - Fr(65, 9) * eta), rel=4e-16)
    assert phil[5] == pytest.approx(3 * phi[5], rel=2e-16)
    assert phi[7] / math.pi == pytest.approx(
        float(Fr(77096675, 254016) + Fr(378515, 1512) * eta - Fr(74045, 756) * eta ** 2), rel=4e-16)
    assert phil[6] == pytest.approx(float(Fr(-6848, 21)), rel=2e-16)


# ----------------------------------------------------------------------------- P1b
def _spa_coefficients_from_energy_flux(with_spin_orbit=False):
    """Stationary-phase phasing derived from the 3.5PN binding energy E(v) and flux F(v).

    Psi(f) = 2 pi f t_c - phi_c - pi/4 + (2/M) int_{v_f}^{v_c} (v_f^3 - v^3) E'(v)/F(v) dv
    (G = c = 1, v_f = (pi M f)^(1/3)).  Only the lower limit contributes f-dependence beyond
    terms absorbed by t_c (prop. to v_f^3) and phi_c (constants).  Returns sympy expressions
    {k: (phi_k, phil_k)} in units of 3/(128 eta) v_f^(k-5).
    """
    v, vf, eta = sp.symbols("v v_f eta", positive=True)
    chis, chia, delta = sp.symbols("chi_s chi_a delta", real=True)
    g = sp.EulerGamma
    pi = sp.pi
    R = sp.Rational
    # binding energy per unit total mass M (3PN; no 3.5PN term)
    e2 = -(R(3, 4) + eta / 12)
    e4 = -(R(27, 8) - R(19, 8) * eta + eta ** 2 / 24)
    e6 = -(R(675, 64) - (R(34445, 576) - R(205, 96) * pi ** 2) * eta + R(155, 96) * eta ** 2
           + R(35, 5184) * eta ** 3)
    e3 = (R(8, 3) * delta * chia + (R(8, 3) - R(4, 3) * eta) * chis) if with_spin_orbit else 0
    E = -(eta / 2) * v ** 2 * (1 + e2 * v ** 2 + e3 * v ** 3 + e4 * v ** 4 + e6 * v ** 6)
    # gravitational-wave flux (3.5PN)
    f2 = -(R(1247, 336) + R(35, 12) * eta)
    f3 = 4 * pi - ((R(11, 4) * delta * chia + (R(11, 4) - 3 * eta) * chis) if with_spin_orbit else 0)
    f4 = -R(44711, 9072) + R(9271, 504) * eta + R(65, 18) * eta ** 2
    f5 = -(R(8191, 672) + R(583, 24) * eta) * pi
    lnv = sp.Symbol("lnv")  # stands for log(v); kept symbolic so that series() treats it as a coefficient
    f6 = (R(6643739519, 69854400) + R(16, 3) * pi ** 2 - R(1712, 105) * g
          + (-R(134543, 7776) + R(41, 48) * pi ** 2) * eta - R(94403, 3024) * eta ** 2
          - R(775, 324) * eta ** 3 - R(856, 105) * (sp.log(16) + 2 * lnv))
    f7 = (-R(16285, 504) + R(214745, 1728) * eta + R(193385, 3024) * eta ** 2) * pi
    flux = R(32, 5) * eta ** 2 * v ** 10 * (1 + f2 * v ** 2 + f3 * v ** 3 + f4 * v ** 4 + f5 * v ** 5
                                             + f6 * v ** 6 + f7 * v ** 7)
    # E'/F = -(5/(32 eta)) v^-9 * (1 + r2 v^2 + ... + r7 v^7): truncated power-series arithmetic
    e_ser = [1, 0, e2, e3, e4, 0, e6, 0]                        # E = -(eta/2) v^2 sum e_k v^k
    de_ser = [sp.expand(sp.Rational(k + 2, 2) * e_ser[k]) for k in range(8)]   # E' = -eta v sum (k+2)/2 e_k v^k
    f_ser = [1, 0, f2, f3, f4, f5, f6, f7]
    inv = [sp.Integer(1)] + [0] * 7                            # 1/(sum f_k v^k)
    for n in range(1, 8):
        inv[n] = sp.expand(-sum(f_ser[k] * inv[n - k] for k in range(1, n + 1)))
    r_ser = [sp.expand(sum(de_ser[k] * inv[n - k] for k in range(n + 1))) for n in range(8)]
    # lower-limit value of  -int (v_f^3 v^(k-9) - v^(k-6)) (c + l ln v) dv, in units of v_f^(k-5):
    # elementary primitives  int v^n = v^(n+1)/(n+1),  int v^n ln v = v^(n+1) [ln v/(n+1) - 1/(n+1)^2],
    # int v^-1 = ln v  (k = 5 only; its log-coefficient r5_l is zero).
    def prim_at_vf(n, c, l):
        """(constant part, ln v_f part) of [int v^n (c + l ln v) dv](v_f) / v_f^(n+1)"""
        if n == -1:
            assert l == 0
            return sp.Integer(0), c          # ln v_f  (times v_f^0)
        m = R(1, n + 1)
        return c * m - l * m * m, l * m

    out = {}
    for k in range(8):
        rk = r_ser[k]
        rk_c, rk_l = rk.coeff(lnv, 0), rk.coeff(lnv, 1)
        a_c, a_l = prim_at_vf(k - 9, rk_c, rk_l)          # times v_f^3 * v_f^(k-8) = v_f^(k-5)
        b_c, b_l = prim_at_vf(k - 6, rk_c, rk_l)          # times v_f^(k-5)
        lower_c, lower_l = -(a_c - b_c), -(a_l - b_l)     # lower limit enters with a minus sign
        scale = 2 * (-R(5, 32)) / R(3, 128)               # (2/M) * [E'/F prefactor] / [3/(128 eta)], eta cancels
        out[k] = (sp.expand(scale * lower_c), sp.expand(scale * lower_l))
    return out, eta, (chis, chia, delta)


@pytest.fixture(scope="module")
def spa_nonspinning():
    return _spa_coefficients_from_energy_flux(False)


def test_p1b_stationary_phase_rederivation(oracle, spa_nonspinning):
    """All phi_k, phil_k (non-spinning) from E(v), F(v): an independent route to the O2 table."""
    derived, eta_s, _ = spa_nonspinning
    for q in (1.0, 0.8, 0.5, 0.3):
        eta = q / (1 + q) ** 2
        phi, phil = oracle.phase_coefficients(eta, 1 / (1 + q), q / (1 + q), 0, 0, 0)
        for k in range(8):
            c = float(sp.N(derived[k][0].subs(eta_s, sp.Float(eta, 30)), 25))
            l = float(sp.N(derived[k][1].subs(eta_s, sp.Float(eta, 30)), 25))
            assert phi[k] == pytest.approx(c, rel=1e-14, abs=1e-14), (k, q)
            assert phil[k] == pytest.approx(l, rel=1e-14, abs=1e-14), (k, q)


def test_p1b_spin_orbit_from_energy_flux(oracle):
    """1.5PN spin-orbit term from the spin-orbit pieces of E and F: phi_3 = -16 pi + 4 beta."""
    derived, eta_s, (chis_s, chia_s, delta_s) = _spa_coefficients_from_energy_flux(True)
    for q, chi1, chi2 in ((0.8, 0.3, -0.2), (0.5, -0.7, 0.6), (1.0, 0.8, 0.8)):
        eta = q / (1 + q) ** 2
        mu1, mu2 = 1 / (1 + q), q / (1 + q)
        # sigma off: compare k=3 only (sigma enters k=4)
        phi, _ = oracle.phase_coefficients(eta, mu1, mu2, chi1, chi2, 1)
        subs = {eta_s: eta, chis_s: (chi1 + chi2) / 2, chia_s: (chi1 - chi2) / 2, delta_s: mu1 - mu2}
        assert phi[3] == pytest.approx(float(sp.N(derived[3][0].subs(subs), 20)), rel=1e-13)
        assert float(sp.N(derived[3][1].subs(subs), 20)) == pytest.approx(0.0, abs=1e-14)


# ----------------------------------------------------------------------------- P1c
def test_p1c_newtonian_chirp_time_and_tc_sign(oracle):
    """d Psi / d f = 2 pi t(f), with t_c - t(f) = (5/256) M_s/eta (pi M_s f)^(-8/3) [1 + (4/3)(743/336 + 11 eta/4) v^2 + O(v^3)].
    Fixes the overall 3/(128 eta) v^-5 normalisation and the sign of the 2 pi f t_c term (reading A3)."""
    mc, q, tc = 0.01, 0.7, 0.37           # tiny masses: v ~ 0.02, PN corrections are small
    theta = np.array([mc, q, 0, 0, 100.0, tc, 0.4, 1.0, 0, 0, 0])
    eta, ms, _, _ = oracle.masses(mc, q)
    f, df = 15.0, 1e-3
    dpsi = (oracle.phase([f + df], theta, 0)[0] - oracle.phase([f - df], theta, 0)[0]) / (2 * df)
    t_of_f = dpsi / (2 * math.pi)
    v = (math.pi * ms * f) ** (1 / 3)
    tau0 = 5.0 / 256.0 * ms / eta * (math.pi * ms * f) ** (-8.0 / 3.0)
    tau1 = tau0 * (1 + 4.0 / 3.0 * (743.0 / 336.0 + 11.0 / 4.0 * eta) * v * v)
    assert tau0 > 1e3 * abs(tc)
    assert (tc - t_of_f) == pytest.approx(tau0, rel=5e-3)      # Newtonian
    assert (tc - t_of_f) == pytest.approx(tau1, rel=20 * v ** 3)  # with the 1PN correction
    # the t_c term alone: Psi(tc + tau) - Psi(tc) = 2 pi f tau
    th2 = theta.copy(); th2[5] += 0.125
    d = oracle.phase([f], th2, 0)[0] - oracle.phase([f], theta, 0)[0]
    assert d == pytest.approx(2 * math.pi * f * 0.125, abs=1e-6)
    # phi_c enters once with a minus sign (reading A4)
    th3 = theta.copy(); th3[6] += 0.5
    assert oracle.phase([f], th3, 0)[0] - oracle.phase([f], theta, 0)[0] == pytest.approx(-0.5, abs=1e-6)


# ----------------------------------------------------------------------------- P1d
@pytest.mark.parametrize("q,chi1,chi2", [(1.0, 0.5, 0.5), (0.8, 0.3, -0.2), (0.5, -0.8, 0.8), (0.31, 0.77, 0.1)])
def test_p1d_spin_terms_two_codings(oracle, q, chi1, chi2):
    """beta/sigma form (oracle) vs the chi_s/chi_a form of SURVEY.md O2, to 1e-14."""
    eta = q / (1 + q) ** 2
    mu1, mu2 = 1 / (1 + q), q / (1 + q)
    delta = mu1 - mu2
    phi_s, _ = oracle.phase_coefficients(eta, mu1, mu2, chi1, chi2, 1)
    phi_0, _ = oracle.phase_coefficients(eta, mu1, mu2, chi1, chi2, 0)
    cs, ca = (chi1 + chi2) / 2, (chi1 - chi2) / 2
    four_beta = (113 / 3 - 76 * eta / 3) * cs + 113 / 3 * delta * ca
    m10sigma = (-405 / 8 + 5 * eta / 2) * cs ** 2 + (-405 / 8 + 200 * eta) * ca ** 2 - 405 / 4 * delta * cs * ca
    assert phi_s[3] - phi_0[3] == pytest.approx(four_beta, rel=1e-13, abs=1e-13)
    assert phi_s[4] - phi_0[4] == pytest.approx(m10sigma, rel=1e-13, abs=1e-13)
    for k in (0, 1, 2, 5, 6, 7):      # reading A8: no spin terms at 2.5PN and above
        assert phi_s[k] == phi_0[k]


def test_p1d_equal_mass_equal_spin_special_case(oracle):
    """eta = 1/4, chi1 = chi2 = chi: 4 beta = (94/3) chi, -10 sigma = -50 chi^2."""
    for chi in (0.1, -0.6, 0.9):
        phi_s, _ = oracle.phase_coefficients(0.25, 0.5, 0.5, chi, chi, 1)
        phi_0, _ = oracle.phase_coefficients(0.25, 0.5, 0.5, chi, chi, 0)
        assert phi_s[3] - phi_0[3] == pytest.approx(94 / 3 * chi, rel=1e-13)
        assert phi_s[4] - phi_0[4] == pytest.approx(-50 * chi * chi, rel=1e-13)


@pytest.mark.parametrize("q,chi1,chi2", [(0.8, 0.3, -0.2), (0.5, -0.8, 0.8)])
def test_p1d_sigma_from_its_three_physical_pieces(oracle, q, chi1, chi2):
    """Reading A7: sigma = S1S2 cross term + quadrupole-monopole (kappa=1) + self-spin, aligned spins:
    eta/48 (-247 + 721) chi1 chi2  +  sum_i (5/2)(3-1) mu_i^2 chi_i^2  +  sum_i (1/96)(7-1) mu_i^2 chi_i^2."""
    eta = q / (1 + q) ** 2
    mu1, mu2 = 1 / (1 + q), q / (1 + q)
    s12 = eta / 48 * (-247 + 721) * chi1 * chi2
    qm = 2.5 * (3 - 1) * (mu1 ** 2 * chi1 ** 2 + mu2 ** 2 * chi2 ** 2)
    ss = (7 - 1) / 96 * (mu1 ** 2 * chi1 ** 2 + mu2 ** 2 * chi2 ** 2)
    phi_s, _ = oracle.phase_coefficients(eta, mu1, mu2, chi1, chi2, 1)
    phi_0, _ = oracle.phase_coefficients(eta, mu1, mu2, chi1, chi2, 0)
    assert phi_s[4] - phi_0[4] == pytest.approx(-10 * (s12 + qm + ss), rel=1e-13)


# ----------------------------------------------------------------------------- P7
def _mp_phase(f, theta, spin_order, consts):
    """The O3 formula in 40-digit arithmetic, from the exact rationals (checks fp64 rounding, not the formula)."""
    mp.mp.dps = 40
    mc, q, chi1, chi2, dl, tc, phic = [mp.mpf(float(x)) for x in theta[:7]]
    tsun = mp.mpf("1.3271244e20") / mp.mpf(299792458) ** 3
    eta = q / (1 + q) ** 2
    ms = mc * eta ** (mp.mpf(-3) / 5) * tsun
    mu1, mu2 = 1 / (1 + q), q / (1 + q)
    beta = sigma = mp.mpf(0)
    if spin_order:
        beta = (mp.mpf(113) / 12 * mu1 ** 2 + mp.mpf(25) / 4 * eta) * chi1 + (mp.mpf(113) / 12 * mu2 ** 2 + mp.mpf(25) / 4 * eta) * chi2
        sigma = mp.mpf(79) / 8 * eta * chi1 * chi2 + mp.mpf(81) / 16 * (mu1 ** 2 * chi1 ** 2 + mu2 ** 2 * chi2 ** 2)
    pi, g = mp.pi, mp.euler
    r = lambda a, b: mp.mpf(a) / mp.mpf(b)
    p = [mp.mpf(0)] * 8
    pl = [mp.mpf(0)] * 8
    p[0] = mp.mpf(1)
    p[2] = r(3715, 756) + r(55, 9) * eta
    p[3] = -16 * pi + 4 * beta
    p[4] = r(15293365, 508032) + r(27145, 504) * eta + r(3085, 72) * eta ** 2 - 10 * sigma
    p[5] = pi * (r(38645, 756) - r(65, 9) * eta)
    pl[5] = 3 * p[5]
    p[6] = (r(11583231236531, 4694215680) - r(640, 3) * pi ** 2 - r(6848, 21) * g
            + eta * (-r(15737765635, 3048192) + r(2255, 12) * pi ** 2) + r(76055, 1728) * eta ** 2
            - r(127825, 1296) * eta ** 3 - r(6848, 21) * mp.log(4))
    pl[6] = -r(6848, 21)
    p[7] = pi * (r(77096675, 254016) + r(378515, 1512) * eta - r(74045, 756) * eta ** 2)
    f = mp.mpf(float(f))
    v = mp.cbrt(pi * ms * f)
    series = sum((p[k] + pl[k] * mp.log(v)) * v ** k for k in range(8))
    return 2 * pi * f * tc - phic - pi / 4 + 3 / (128 * eta) * v ** -5 * series


def test_p7_fp64_accuracy_of_the_phase(oracle):
    """Oracle phase vs 40-digit arithmetic at random (theta, f): error below 16 ulp of |Psi| (+1e-13): Psi ~ M_s^(-5/3), so the
    roundings of eta^(-3/5), cbrt and pow(v,-5) are amplified by 5/3..5.
    The bound is ulp-relative because |Psi| reaches 4.5e4 rad (C3, Mc = 1.1 at 10 Hz): 1 ulp = 7e-12 rad."""
    rng = np.random.default_rng(7)
    worst = 0.0
    for i in range(200):
        bns = i % 2 == 0
        mc = rng.uniform(1.1, 1.3) if bns else rng.uniform(20, 40)
        theta = np.array([mc, rng.uniform(0.5, 1), rng.uniform(-0.8, 0.8), rng.uniform(-0.8, 0.8), 100.0,
                          rng.uniform(-0.1, 0.1), rng.uniform(0, 2 * math.pi), 0.3, 0, 0, 0])
        f = float(rng.uniform(10, 2048)) if i % 4 else 10.0
        got = oracle.phase([f], theta, 1)[0]
        want = _mp_phase(f, theta, 1, None)
        err = abs(float(mp.mpf(got) - want))
        bound = 16 * np.spacing(abs(got)) + 1e-13
        worst = max(worst, err / bound)
        assert err < bound, (theta, f, err, bound)
    assert worst > 0  # the comparison was not vacuous
