"""A minimal batched-sampler driver for the likelihood library (the part that needs one GPU).

The paper's sampler is the serial consumer of ln L ("it is difficult to parallelize the actual
sampling algorithm"); what parallelises is the likelihood of many proposals at once.  This driver is an ensemble sampler
whose walkers ARE the batch: an affine-invariant stretch move (Goodman & Weare 2010) on two half-ensembles, so that one
iteration is two ``gw_lnl_batch_host`` calls of W/2 proposals each -- host parameters in, host ln L out, exactly the
end-to-end path bench.py times.  All of the method's arithmetic (waveform, projection, inner products) runs in the CUDA
library; this module only proposes, accepts and rejects (numpy on the host).

    python -m paper_1904_02863_b200.sampler [--workload C1] [--walkers 4096] [--iters 300]

prints one JSON line: iterations/s, likelihood evaluations/s, the fraction of wall time spent inside the library calls,
and the posterior summary of (Mc, q) against the injected values.
"""
from __future__ import annotations

import argparse
import json
import time
from typing import Optional, Sequence

import numpy as np

from . import inputs


def stretch_ensemble(lnl_fn, theta0: np.ndarray, free: Sequence[int], lo: np.ndarray, hi: np.ndarray, n_iter: int,
                     seed: int = 1, a: float = 2.0, thin: int = 1):
    """Affine-invariant ensemble MCMC with a uniform prior on the box [lo, hi] of the free columns.

    lnl_fn(theta[B][n_param]) -> lnL[B] is called twice per iteration with W/2 rows.  theta0 [W][n_param] holds the
    walkers' start (fixed columns stay as given).  Returns a dict with the thinned chain [n_keep][W][len(free)], the
    ln L of the last state, the acceptance fraction and the time spent inside lnl_fn.
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    free = np.asarray(free)
    W, d = theta0.shape[0], len(free)
    if W % 2 or W < 2 * (d + 1):
        raise ValueError("need an even number of walkers, at least 2 (d + 1)")
    theta = np.ascontiguousarray(theta0, dtype=np.float64).copy()
    half = W // 2
    sets = (np.arange(half), np.arange(half, W))
    t_lib = 0.0
    t0 = time.perf_counter()
    lnl = np.empty(W)
    for s in sets:
        t1 = time.perf_counter(); lnl[s] = lnl_fn(theta[s]); t_lib += time.perf_counter() - t1
    chain = []
    n_acc = 0
    for it in range(n_iter):
        for k in (0, 1):
            s, c = sets[k], sets[1 - k]
            partner = theta[c[rng.integers(0, half, size=half)]][:, free]
            z = ((a - 1.0) * rng.random(half) + 1.0) ** 2 / a
            prop = theta[s].copy()
            prop[:, free] = partner + z[:, None] * (theta[s][:, free] - partner)
            inside = np.all((prop[:, free] >= lo) & (prop[:, free] <= hi), axis=1)
            safe = np.where(inside[:, None], prop, theta[s])          # out-of-box proposals are never evaluated as such
            t1 = time.perf_counter(); new = lnl_fn(safe); t_lib += time.perf_counter() - t1
            log_ratio = (d - 1) * np.log(z) + new - lnl[s]
            accept = inside & (np.log(rng.random(half)) < log_ratio)
            theta[s[accept]] = prop[accept]
            lnl[s[accept]] = new[accept]
            n_acc += int(accept.sum())
        if (it + 1) % thin == 0:
            chain.append(theta[:, free].copy())
    wall = time.perf_counter() - t0
    return {"chain": np.array(chain), "theta": theta, "lnl": lnl, "accept": n_acc / (n_iter * W), "wall_s": wall,
            "library_s": t_lib, "n_eval": W * (n_iter + 1)}


FREE_DEFAULT = (inputs.P_MC, inputs.P_Q, inputs.P_CHI1, inputs.P_CHI2, inputs.P_DL, inputs.P_TC)


def run(workload: str = "C1", walkers: int = 4096, iters: int = 300, burn: Optional[int] = None, seed: int = 7,
        reduced_f_max: Optional[float] = None):
    """Sample (Mc, q, chi1, chi2, D, t_c) of a seeded synthetic event of the given workload shape, phi_c marginalised
    (gw_options.phase_marginal), the remaining extrinsic parameters fixed at the injection.  The injection is computed by
    the library's own waveform kernel, as in bench.py."""
    from .binding import GwContext, waveform_for_inputs
    cfg = inputs.CONFIGS[workload]
    if reduced_f_max is not None:
        cfg = cfg.reduced(f_max=reduced_f_max)
    f, S, dets = inputs.frequency_grid(cfg), inputs.psd(cfg), inputs.detectors(cfg)
    d = inputs.make_data(cfg, waveform_for_inputs)
    inj = np.array(cfg.theta_inj)
    free = np.array(FREE_DEFAULT if cfg.spin_order else (inputs.P_MC, inputs.P_Q, inputs.P_DL, inputs.P_TC))
    lo = np.array([cfg.mc_range[0], cfg.q_range[0], -0.9, -0.9, cfg.dl_range[0], -0.1])
    hi = np.array([cfg.mc_range[1], cfg.q_range[1], 0.9, 0.9, cfg.dl_range[1], 0.1])
    if not cfg.spin_order:
        lo, hi = lo[[0, 1, 4, 5]], hi[[0, 1, 4, 5]]
    rng = np.random.Generator(np.random.PCG64(seed))
    theta0 = np.tile(inj, (walkers, 1))
    scale = np.array([1e-3 * inj[inputs.P_MC], 0.02, 0.05, 0.05, 0.02 * inj[inputs.P_DL], 2e-4])
    if not cfg.spin_order:
        scale = scale[[0, 1, 4, 5]]
    theta0[:, free] = np.clip(inj[free] + scale * rng.standard_normal((walkers, len(free))), lo, hi)
    burn = iters // 2 if burn is None else burn
    with GwContext(f, d, S, dets, cfg.gmst, spin_order=cfg.spin_order, max_batch=walkers // 2, phase_marginal=1) as ctx:
        out = np.empty(walkers // 2)

        def lnl_fn(th):
            return ctx.lnl_batch_host(th, out=out).copy()

        res = stretch_ensemble(lnl_fn, theta0, free, lo, hi, iters, seed=seed + 1)
        plan = ctx.plan(walkers // 2)
    post = res["chain"][burn:].reshape(-1, len(free))
    summary = {"workload": f"{cfg.name}: {cfg.n_det} det x {cfg.n_bins} bins", "walkers": walkers, "iterations": iters,
               "burn_in": burn, "free_parameters": [int(i) for i in free], "accept_fraction": res["accept"],
               "iterations_per_s": iters / res["wall_s"], "lnl_evals_per_s": res["n_eval"] / res["wall_s"],
               "fraction_of_wall_time_in_library": res["library_s"] / res["wall_s"], "wall_s": res["wall_s"],
               "calls_per_iteration": 2, "proposals_per_call": walkers // 2, "plan": plan,
               "injected": {"Mc": float(inj[inputs.P_MC]), "q": float(inj[inputs.P_Q])},
               "posterior": {"Mc_mean": float(post[:, 0].mean()), "Mc_std": float(post[:, 0].std()),
                             "q_mean": float(post[:, 1].mean()), "q_std": float(post[:, 1].std())}}
    return summary, res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="C1")
    ap.add_argument("--walkers", type=int, default=4096)
    ap.add_argument("--iters", type=int, default=300)
    ap.add_argument("--seed", type=int, default=7)
    args = ap.parse_args()
    summary, _ = run(args.workload, args.walkers, args.iters, seed=args.seed)
    print(json.dumps(summary))


if __name__ == "__main__":
    main()
