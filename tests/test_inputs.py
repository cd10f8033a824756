"""The seeded input recipe: shapes, PSD values, geometry invariants.

The H1/L1/V1 digits are input data; the source document is not available, so they are pinned
by invariants only (unit arms, orthogonality, Earth radius, 10/27/26 ms baselines).
"""
import numpy as np
import pytest

from paper_1904_02863_b200 import inputs

C_SI = 299792458.0


@pytest.mark.parametrize("name,n_det,n_bins,batch", [
    ("C0", 1, 3937, 256), ("C1", 3, 8113, 4096), ("C2", 3, 259585, 1024),
    ("C3", 3, 1043457, 256), ("C4", 3, 8113, 65536)])
def test_config_shapes(name, n_det, n_bins, batch):
    cfg = inputs.CONFIGS[name]
    assert (cfg.n_det, cfg.n_bins, cfg.batch) == (n_det, n_bins, batch)
    f = inputs.frequency_grid(cfg)
    assert f.shape == (n_bins,) and f[0] == cfg.f_min and f[-1] == pytest.approx(cfg.f_max, rel=1e-15)
    assert np.all(np.diff(f) > 0)
    assert (f[-1] - f[0]) / (n_bins - 1) == pytest.approx(cfg.delta_f, rel=1e-14)


def test_psd_printed_values():
    """SURVEY.md scale table: min 3.2414e-48 at ~228.3 Hz; S(20), S(10), S(2048); positive on [10, 2048]."""
    f = np.linspace(10, 2048, 200001)
    S = inputs.analytic_psd(f)
    assert np.all(S > 0)
    assert S.min() == pytest.approx(3.2414e-48, rel=1e-4)
    assert f[S.argmin()] == pytest.approx(228.3, abs=0.2)
    assert inputs.analytic_psd(np.array([20.0]))[0] == pytest.approx(1.8154e-45, rel=1e-4)
    assert inputs.analytic_psd(np.array([10.0]))[0] == pytest.approx(3.2612e-44, rel=1e-4)
    assert inputs.analytic_psd(np.array([2048.0]))[0] == pytest.approx(9.64e-46, rel=1e-3)
    # the formula at x = 1 (f = 215 Hz): 1e-49 [1 - 5 + 111 (1/2)/(3/2)] = 33e-49
    assert inputs.analytic_psd(np.array([215.0]))[0] == pytest.approx(33e-49, rel=1e-14)


def test_detector_geometry_invariants():
    rows = {n: inputs.geometric_detector(n) for n in ("H1", "L1", "V1")}
    for n, r in rows.items():
        x, y, v = r[4:7], r[7:10], r[1:4]
        assert abs(np.linalg.norm(x) - 1) < 5e-12 and abs(np.linalg.norm(y) - 1) < 5e-12
        assert abs(np.dot(x, y)) < 2e-7
        up = v / np.linalg.norm(v)
        assert abs(np.dot(x, up)) < np.sin(np.radians(0.2)) and abs(np.dot(y, up)) < np.sin(np.radians(0.2))
    assert np.linalg.norm(rows["H1"][1:4]) / 1e3 == pytest.approx(6367.1, abs=0.1)
    assert np.linalg.norm(rows["L1"][1:4]) / 1e3 == pytest.approx(6372.6, abs=0.1)
    assert np.linalg.norm(rows["V1"][1:4]) / 1e3 == pytest.approx(6368.1, abs=0.1)
    lt = lambda a, b: np.linalg.norm(rows[a][1:4] - rows[b][1:4]) / C_SI * 1e3
    assert lt("H1", "L1") == pytest.approx(10.013, abs=1e-3)
    assert lt("H1", "V1") == pytest.approx(27.288, abs=1e-3)
    assert lt("L1", "V1") == pytest.approx(26.448, abs=1e-3)


def test_proposals_ranges_seeding_and_prefixes():
    for name in ("C0", "C1", "C2", "C3"):
        cfg = inputs.CONFIGS[name]
        th = inputs.proposals(cfg)
        assert th.shape == (cfg.batch, 11)
        assert np.array_equal(th, inputs.proposals(cfg))                 # seeded
        assert np.array_equal(th[0], np.array(cfg.theta_inj))           # row 0 = injection
        body = th[1:]
        for col, (lo, hi) in ((inputs.P_MC, cfg.mc_range), (inputs.P_Q, cfg.q_range), (inputs.P_DL, cfg.dl_range)):
            assert body[:, col].min() >= lo and body[:, col].max() <= hi
        assert np.abs(body[:, inputs.P_TC]).max() <= 0.1
        assert body[:, inputs.P_PHIC].min() >= 0 and body[:, inputs.P_PHIC].max() < 2 * np.pi
        if name == "C0":
            assert np.all(body[:, [inputs.P_CHI1, inputs.P_CHI2]] == 0) and np.all(body[:, inputs.P_COSI] == 1)
        else:
            assert np.abs(body[:, inputs.P_COSI]).max() <= 1 and np.abs(body[:, inputs.P_DEC]).max() <= np.pi / 2
            assert body[:, inputs.P_CHI1].min() >= cfg.chi_range[0] and body[:, inputs.P_CHI1].max() <= cfg.chi_range[1]
    c4 = inputs.CONFIGS["C4"]
    assert np.array_equal(inputs.proposals(c4, 16), inputs.proposals(c4, 256)[:16])
    # distinct configs draw distinct streams
    assert not np.array_equal(inputs.proposals(inputs.CONFIGS["C1"], 8)[1:], inputs.proposals(c4, 8)[1:])


def test_noise_statistics_and_data_assembly():
    cfg = inputs.CONFIGS["C1"]
    n = inputs.noise(cfg)
    assert n.shape == (3, cfg.n_bins) and np.array_equal(n, inputs.noise(cfg))
    w = n / np.sqrt(inputs.psd(cfg) / (4 * cfg.delta_f))
    assert w.real.var() == pytest.approx(1.0, rel=0.03) and w.imag.var() == pytest.approx(1.0, rel=0.03)
    assert abs(np.mean(w.real * w.imag)) < 0.02
    calls = []

    def fake_waveform(f, dets, gmst, theta, spin_order):
        calls.append((f.shape, dets.shape, gmst, theta.shape, spin_order))
        return np.ones((1, 3, f.shape[0]), complex)

    d = inputs.make_data(cfg, fake_waveform)
    assert calls == [((cfg.n_bins,), (3, 13), 2.0, (1, 11), 1)]
    assert np.array_equal(d, 1.0 + n)
