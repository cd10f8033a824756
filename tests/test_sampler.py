"""The batched-sampler driver (paper_1904_02863_b200/sampler.py).  `-m "not gpu"`: the host
logic samples a known Gaussian correctly through the same stretch-move code; `-m gpu`: on a C1-shaped event it recovers
the injected chirp mass and mass ratio within the posterior width, every likelihood coming from gw_lnl_batch_host."""
import numpy as np
import pytest

from paper_1904_02863_b200 import sampler


def test_stretch_move_samples_a_known_gaussian():
    mu = np.array([1.0, -2.0, 0.5])
    sg = np.array([0.1, 2.0, 0.01])
    calls = []

    def lnl(th):
        calls.append(len(th))
        return -0.5 * (((th[:, [0, 2, 3]] - mu) / sg) ** 2).sum(axis=1)

    rng = np.random.Generator(np.random.PCG64(3))
    W = 400
    th0 = np.zeros((W, 5))
    th0[:, 1] = 7.0                                           # a fixed column stays untouched
    th0[:, [0, 2, 3]] = mu + 3 * sg * rng.standard_normal((W, 3))
    res = sampler.stretch_ensemble(lnl, th0, [0, 2, 3], np.array([-50.0, -50.0, -50.0]), np.array([50.0, 50.0, 50.0]), 600, seed=5)
    post = res["chain"][200:].reshape(-1, 3)
    assert np.all(np.abs(post.mean(axis=0) - mu) < 0.05 * sg) and np.all(np.abs(post.std(axis=0) / sg - 1.0) < 0.05)
    assert np.all(res["theta"][:, 1] == 7.0) and 0.2 < res["accept"] < 0.9
    assert set(calls) == {W // 2} and len(calls) == 2 * 600 + 2    # two half-ensemble calls per iteration
    # a hard prior wall: walkers that start inside the box never leave it
    inside0 = np.clip(th0[:, [0, 2, 3]], mu - 0.5 * sg, mu + 0.5 * sg)
    th1 = th0.copy(); th1[:, [0, 2, 3]] = inside0
    res = sampler.stretch_ensemble(lnl, th1, [0, 2, 3], mu - 0.5 * sg, mu + 0.5 * sg, 50, seed=6)
    assert np.all(res["chain"] >= mu - 0.5 * sg) and np.all(res["chain"] <= mu + 0.5 * sg)
    with pytest.raises(ValueError):
        sampler.stretch_ensemble(lnl, th0[:5], [0, 2, 3], mu - 1, mu + 1, 1)


@pytest.mark.gpu
def test_sampler_recovers_the_injection_on_a_c1_shaped_event():
    summary, res = sampler.run("C1", walkers=1024, iters=400, seed=11)
    p, inj = summary["posterior"], summary["injected"]
    assert 0.1 < summary["accept_fraction"] < 0.8
    assert p["Mc_std"] < 1.0 and abs(p["Mc_mean"] - inj["Mc"]) < 4 * p["Mc_std"] + 1e-3      # a ~1 % measurement of Mc
    assert abs(p["q_mean"] - inj["q"]) < 4 * p["q_std"] + 0.01
    assert summary["plan"]["n_ctas"] >= 1 and summary["lnl_evals_per_s"] > 1e5
    print(summary)
