"""`-m "not gpu"`: pins of the population-likelihood oracle (oracle/gw_pop_oracle.c; Eq. 3, data flow
PAPER.md:109).  PAPER.md prints no population model (PAPER.md:117 cites them), so the densities are DESIGN.md reading P1
and are pinned by what mathematics fixes: each integrates to one (adaptive quadrature), each reduces to a library
density (scipy.stats, an independent implementation) or to a closed form in a special case, the joint ratio obeys the
importance-sampling identity, and Eq. 3 itself is checked on a hand-expanded 2 x 3 case and by its invariances."""
import math

import numpy as np
import pytest
from scipy import integrate, stats

from paper_1904_02863_b200 import inputs

LAM0 = np.array([2.35, 5.0, 70.0, 0.1, 33.0, 5.0, 1.3, 2.0, 4.0, 0.6, 1.0, 1.5])


def _random_lambdas(n, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    lo = np.array([-1.0, 3.0, 40.0, 0.0, 20.0, 1.0, -3.0, 0.6, 0.6, 0.0, 0.2, 0.2])
    hi = np.array([4.0, 9.0, 95.0, 1.0, 45.0, 9.0, 5.0, 6.0, 6.0, 1.0, 4.0, 4.0])
    return lo + (hi - lo) * rng.random((n, 12))


# ---- P12a: every factor integrates to one over its support ---------------------------------------------------------
@pytest.mark.parametrize("lam", list(_random_lambdas(6, 1)) + [LAM0])
def test_each_density_integrates_to_one(oracle, lam):
    mmin, mmax = lam[1], lam[2]
    pts = [lam[4]] if mmin < lam[4] < mmax else None
    val, _ = integrate.quad(lambda m: oracle.pop_mass_pdf(m, lam), mmin, mmax, points=pts, epsabs=0, epsrel=1e-11, limit=400)
    assert abs(val - 1.0) < 1e-9
    for m1 in (mmin * 1.05, 0.5 * (mmin + mmax), mmax):
        val, _ = integrate.quad(lambda q: oracle.pop_ratio_pdf(q, m1, lam), mmin / m1, 1.0, epsabs=0, epsrel=1e-11, limit=400)
        assert abs(val - 1.0) < 1e-9
    if lam[7] >= 1.0 and lam[8] >= 1.0:             # integrable end-point singularities otherwise: checked via scipy below
        val, _ = integrate.quad(lambda a: oracle.pop_beta_pdf(a, lam[7], lam[8]), 0.0, 1.0, epsabs=0, epsrel=1e-11, limit=400)
        assert abs(val - 1.0) < 1e-9
    # the tilt mixture is separable term by term: integrate over c2 analytically-free by nesting quadratures
    inner = lambda c1: integrate.quad(lambda c2: oracle.pop_tilt_pdf(c1, c2, lam), -1.0, 1.0, epsabs=0, epsrel=1e-10)[0]
    val, _ = integrate.quad(inner, -1.0, 1.0, epsabs=0, epsrel=1e-9)
    assert abs(val - 1.0) < 1e-7


# ---- P12b: library densities (independent implementations) ---------------------------------------------------------
def test_factors_against_scipy_stats(oracle):
    rng = np.random.Generator(np.random.PCG64(2))
    for lam in _random_lambdas(20, 3):
        a, b = lam[7], lam[8]
        for x in rng.random(5):
            assert oracle.pop_beta_pdf(x, a, b) == pytest.approx(stats.beta.pdf(x, a, b), rel=1e-12)
        mu, sg, lo, hi = lam[4], lam[5], lam[1], lam[2]
        tn = stats.truncnorm((lo - mu) / sg, (hi - mu) / sg, loc=mu, scale=sg)
        for x in lo + (hi - lo) * rng.random(5):
            assert oracle.pop_truncnorm_pdf(x, mu, sg, lo, hi) == pytest.approx(tn.pdf(x), rel=1e-11)
        # power law as a scipy "powerlaw"-free closed form: pdf ratio and normalisation by quadrature
        al = lam[0]
        x1, x2 = lo + (hi - lo) * rng.random(2)
        assert oracle.pop_powerlaw_pdf(x1, al, lo, hi) / oracle.pop_powerlaw_pdf(x2, al, lo, hi) == pytest.approx((x1 / x2) ** -al, rel=1e-12)
    # outside the support every factor is exactly zero
    assert oracle.pop_powerlaw_pdf(4.99, 2.0, 5.0, 50.0) == 0.0 and oracle.pop_powerlaw_pdf(50.01, 2.0, 5.0, 50.0) == 0.0
    assert oracle.pop_truncnorm_pdf(-1.01, 1.0, 1.0, -1.0, 1.0) == 0.0 and oracle.pop_beta_pdf(1.01, 2.0, 2.0) == 0.0
    assert oracle.pop_ratio_pdf(0.09, 50.0, LAM0) == 0.0 and oracle.pop_ratio_pdf(0.11, 50.0, LAM0) > 0.0   # q_min = 5/50
    assert oracle.pop_ratio_pdf(0.9, 4.0, LAM0) == 0.0                                                      # m1 < m_min


# ---- P12c: closed-form special cases -------------------------------------------------------------------------------
def test_special_cases_reduce_to_closed_forms(oracle):
    # alpha = 0, lam = 0: uniform in m1; alpha = 1 (removable singularity of the normalisation): 1 / (m ln(hi/lo))
    flat = LAM0.copy(); flat[0] = 0.0; flat[3] = 0.0
    assert oracle.pop_mass_pdf(20.0, flat) == pytest.approx(1.0 / 65.0, rel=1e-14)
    assert oracle.pop_powerlaw_pdf(20.0, 1.0, 5.0, 70.0) == pytest.approx(1.0 / (20.0 * math.log(14.0)), rel=1e-14)
    assert oracle.pop_powerlaw_pdf(20.0, 1.0 + 1e-9, 5.0, 70.0) == pytest.approx(oracle.pop_powerlaw_pdf(20.0, 1.0, 5.0, 70.0), rel=1e-7)
    # alpha = 2: x^-2 / (1/lo - 1/hi)
    assert oracle.pop_powerlaw_pdf(10.0, 2.0, 5.0, 50.0) == pytest.approx(0.01 / (0.2 - 0.02), rel=1e-14)
    # lam = 1: the pure truncated Gaussian peak
    peak = LAM0.copy(); peak[3] = 1.0
    assert oracle.pop_mass_pdf(30.0, peak) == pytest.approx(oracle.pop_truncnorm_pdf(30.0, 33.0, 5.0, 5.0, 70.0), rel=1e-15)
    # beta_q = 0: uniform on [m_min/m1, 1]; beta_q = 1: 2 q / (1 - (m_min/m1)^2); beta_q = -1: 1 / (q ln(m1/m_min))
    l0 = LAM0.copy(); l0[6] = 0.0
    assert oracle.pop_ratio_pdf(0.7, 50.0, l0) == pytest.approx(1.0 / 0.9, rel=1e-14)
    l1 = LAM0.copy(); l1[6] = 1.0
    assert oracle.pop_ratio_pdf(0.7, 50.0, l1) == pytest.approx(1.4 / 0.99, rel=1e-14)
    lm = LAM0.copy(); lm[6] = -1.0
    assert oracle.pop_ratio_pdf(0.7, 50.0, lm) == pytest.approx(1.0 / (0.7 * math.log(10.0)), rel=1e-14)
    # Beta(1,1) is uniform, Beta(2,1) = 2a; xi = 0 is isotropic: 1/4; sigma -> large: the aligned part tends to 1/4 too
    assert oracle.pop_beta_pdf(0.37, 1.0, 1.0) == pytest.approx(1.0, rel=1e-15)
    assert oracle.pop_beta_pdf(0.37, 2.0, 1.0) == pytest.approx(0.74, rel=1e-14)
    iso = LAM0.copy(); iso[9] = 0.0
    assert oracle.pop_tilt_pdf(0.3, -0.8, iso) == pytest.approx(0.25, rel=1e-15)
    wide = LAM0.copy(); wide[9] = 1.0; wide[10] = wide[11] = 1e4
    assert oracle.pop_tilt_pdf(0.3, -0.8, wide) == pytest.approx(0.25, rel=1e-7)
    # the aligned component prefers cos tilt = 1 and is symmetric in exchanging the two bodies' widths and arguments
    al = LAM0.copy(); al[9] = 1.0
    assert oracle.pop_tilt_pdf(0.9, 0.9, al) > oracle.pop_tilt_pdf(0.0, 0.0, al) > oracle.pop_tilt_pdf(-0.9, -0.9, al)
    sw = al.copy(); sw[10], sw[11] = al[11], al[10]
    assert oracle.pop_tilt_pdf(0.2, 0.7, al) == pytest.approx(oracle.pop_tilt_pdf(0.7, 0.2, sw), rel=1e-15)


def test_joint_density_is_the_product_of_its_factors(oracle):
    rng = np.random.Generator(np.random.PCG64(4))
    for lam in _random_lambdas(10, 5):
        th = np.array([lam[1] + (lam[2] - lam[1]) * rng.random(), 0.0, rng.random(), rng.random(),
                       2 * rng.random() - 1, 2 * rng.random() - 1])
        th[1] = lam[1] / th[0] + (1 - lam[1] / th[0]) * rng.random()
        want = (oracle.pop_mass_pdf(th[0], lam) * oracle.pop_ratio_pdf(th[1], th[0], lam) *
                oracle.pop_beta_pdf(th[2], lam[7], lam[8]) * oracle.pop_beta_pdf(th[3], lam[7], lam[8]) *
                oracle.pop_tilt_pdf(th[4], th[5], lam))
        assert want > 0 and oracle.pop_pdf(th, lam) == pytest.approx(want, rel=1e-15)


# ---- P12d: Eq. 3 on a hand-expanded 2 x 3 case, literal numbers ----------------------------------------------------
def test_eq3_hand_expanded_two_events_three_samples(oracle):
    """Flat model: alpha = 0, lam = 0 on [5, 55] -> p(m1) = 1/50; beta_q = 0 -> p(q|m1) = 1/(1 - 5/m1); Beta(1,1) = 1;
    xi = 0 -> 1/4.  So w_ij = (1/50) / (1 - 5/m1_ij) / 4 / prior_ij, typed out below."""
    lam = np.array([0.0, 5.0, 55.0, 0.0, 30.0, 5.0, 0.0, 1.0, 1.0, 0.0, 1.0, 1.0])
    s = np.array([[[10.0, 0.8, 0.1, 0.2, 0.3, -0.4], [25.0, 0.6, 0.5, 0.5, 0.0, 0.0], [50.0, 0.2, 0.9, 0.3, -0.9, 0.9]],
                  [[20.0, 0.5, 0.2, 0.2, 0.5, 0.5], [60.0, 0.9, 0.2, 0.2, 0.5, 0.5], [40.0, 0.1, 0.7, 0.1, 0.1, 0.2]]])
    p0 = np.array([[0.01, 0.02, 0.005], [0.004, 0.01, 0.02]])
    w = [[(1 / 50) / (1 - 5 / 10) / 4 / 0.01, (1 / 50) / (1 - 5 / 25) / 4 / 0.02, (1 / 50) / (1 - 5 / 50) / 4 / 0.005],
         [(1 / 50) / (1 - 5 / 20) / 4 / 0.004, 0.0,                          # m1 = 60 > m_max: no support
          0.0]]                                                             # q = 0.1 < m_min/m1 = 0.125: no support
    want = math.log(sum(w[0])) + math.log(sum(w[1]))
    lnl, inner, _ = oracle.pop_lnl(s, p0, lam[None])
    assert inner[0] == pytest.approx([sum(w[0]), sum(w[1])], rel=1e-14)
    assert lnl[0] == pytest.approx(want, rel=1e-14)


# ---- P12e: invariances and limits of Eq. 3 -------------------------------------------------------------------------
def test_eq3_invariances_and_flat_model(oracle):
    cfg = inputs.POP_CONFIGS["P0"]
    s, p0 = inputs.pop_samples(cfg)
    lam = inputs.pop_lambdas(cfg)[:8]
    lnl, inner, _ = oracle.pop_lnl(s, p0, lam)
    assert np.all(np.isfinite(lnl))
    rng = np.random.Generator(np.random.PCG64(6))
    pj = rng.permutation(cfg.n_samples)
    pi = rng.permutation(cfg.n_events)
    lnl_j, _, _ = oracle.pop_lnl(s[:, pj], p0[:, pj], lam)           # order of the samples within an event
    lnl_i, inner_i, _ = oracle.pop_lnl(s[pi], p0[pi], lam)           # order of the events
    assert np.allclose(lnl_j, lnl, rtol=1e-13, atol=0) and np.allclose(lnl_i, lnl, rtol=1e-13, atol=0)
    assert np.allclose(inner_i, inner[:, pi], rtol=1e-13)
    # doubling every prior value subtracts N ln 2; duplicating every sample adds N ln 2
    lnl_2, _, _ = oracle.pop_lnl(s, 2.0 * p0, lam)
    assert np.allclose(lnl_2, lnl - cfg.n_events * math.log(2.0), rtol=1e-13)
    lnl_d, _, _ = oracle.pop_lnl(np.concatenate([s, s], axis=1), np.concatenate([p0, p0], axis=1), lam)
    assert np.allclose(lnl_d, lnl + cfg.n_events * math.log(2.0), rtol=1e-13)
    # the population equal to the sampling prior (on the samples' support): every weight is 1, ln L = N ln n.
    # prior = flat in (m1, q, a1, a2, c1, c2) on [5,55] x [5/m1,1] x [0,1]^2 x [-1,1]^2 = model with alpha=0, beta_q=0
    flat = np.array([0.0, 5.0, 55.0, 0.0, 30.0, 5.0, 0.0, 1.0, 1.0, 0.0, 1.0, 1.0])
    m1 = 6.0 + 48.0 * rng.random((3, 500))
    q = 5.0 / m1 + (1 - 5.0 / m1) * rng.random((3, 500))
    th = np.stack([m1, q, rng.random((3, 500)), rng.random((3, 500)), 2 * rng.random((3, 500)) - 1, 2 * rng.random((3, 500)) - 1], axis=-1)
    prior = (1 / 50.0) / (1 - 5.0 / m1) * 0.25
    lnl_f, inner_f, _ = oracle.pop_lnl(th, prior, flat[None])
    assert np.allclose(inner_f, 500.0, rtol=1e-13) and lnl_f[0] == pytest.approx(3 * math.log(500.0), rel=1e-13)


def test_eq3_degenerate_inputs(oracle):
    cfg = inputs.POP_CONFIGS["P0"]
    s, p0 = inputs.pop_samples(cfg)
    s, p0 = s[:3, :50], p0[:3, :50]
    bad = LAM0.copy(); bad[2] = bad[1] - 1.0                        # m_max < m_min
    neg = LAM0.copy(); neg[5] = -1.0                                # sigma < 0
    nan = LAM0.copy(); nan[0] = np.nan
    narrow = LAM0.copy(); narrow[1], narrow[2] = 90.0, 94.0         # no sample of event 0 lies in [90, 94]
    lnl, inner, _ = oracle.pop_lnl(s, p0, np.stack([LAM0, bad, neg, nan, narrow]))
    assert np.isfinite(lnl[0]) and np.all(np.isnan(lnl[1:4])) and lnl[4] == -np.inf and np.any(inner[4] == 0.0)
    assert not oracle.pop_lambda_valid(bad) and oracle.pop_lambda_valid(LAM0)


# ---- P12f: the importance-sampling identity pins the normalisation of the JOINT ratio -------------------------------
def test_importance_sampling_identity(oracle):
    """theta_j ~ p0 (a flat proposal that covers the model's support) => (1/n) sum_j p(theta_j | Lambda) / p0 -> 1, for
    any Lambda, because both densities integrate to one.  n = 4e5: the mean must sit within 5 standard errors."""
    rng = np.random.Generator(np.random.PCG64(7))
    n = 400000
    lam = np.array([1.8, 6.0, 60.0, 0.2, 30.0, 6.0, 0.7, 1.5, 2.5, 0.5, 1.2, 0.8])
    m1 = 6.0 + 54.0 * rng.random(n)
    q = rng.random(n)                                                # flat on [0,1] (covers [m_min/m1, 1])
    th = np.stack([m1, q, rng.random(n), rng.random(n), 2 * rng.random(n) - 1, 2 * rng.random(n) - 1], axis=-1)
    p0 = np.full(n, (1 / 54.0) * 0.25)
    _, inner, _ = oracle.pop_lnl(th[None], p0[None], lam[None])
    w = np.array([oracle.pop_pdf(t, lam) for t in th[:20000]]) / p0[0]
    se = w.std() / math.sqrt(n)
    assert abs(inner[0, 0] / n - 1.0) < 5 * se, (inner[0, 0] / n, se)
