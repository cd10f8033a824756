"""Helpers shared by the `-m gpu` parity tests: build a GwContext for a (possibly reduced) config with
oracle-injected data, and the two tolerances of BASELINE.json's north_star (reading A16 of DESIGN.md)."""
import numpy as np

from paper_1904_02863_b200 import inputs

H_RTOL = 1e-9        # |dh| <= 1e-9 * max_bins |h|  per (proposal, detector) row
LNL_RTOL = 1e-8      # |dlnL| <= 1e-8 * (|sum_I Re<d|h>_I| + sum_I <h|h>_I)


def make_problem(oracle, cfg):
    """freqs, psd, det rows, data (oracle injection + seeded noise), theta for a config."""
    f = inputs.frequency_grid(cfg)
    S = inputs.psd(cfg)
    dets = inputs.detectors(cfg)
    d = inputs.make_data(cfg, oracle.waveform)
    th = inputs.proposals(cfg)
    return f, S, dets, d, th


def make_ctx(cfg, f, d, S, dets, max_batch=None):
    from paper_1904_02863_b200 import GwContext
    return GwContext(f, d, S, dets, cfg.gmst, spin_order=cfg.spin_order,
                     max_batch=max_batch or max(cfg.batch, 1))


def assert_h_close(h_gpu, h_ref):
    """elementwise, row-wise scale (A16)."""
    scale = np.abs(h_ref).max(axis=-1, keepdims=True)
    err = np.abs(h_gpu - h_ref)
    worst = float((err / scale).max())
    assert worst <= H_RTOL, f"max |dh|/max|h| = {worst:.3e}"
    return worst


def assert_lnl_close(lnl_gpu, parts_gpu, lnl_ref, parts_ref):
    """lnL per proposal against the summed scale; parts per detector against the same bound (A16)."""
    scale = np.abs(parts_ref[..., 0].sum(axis=1)) + parts_ref[..., 2].sum(axis=1)
    worst = float((np.abs(lnl_gpu - lnl_ref) / scale).max())
    assert worst <= LNL_RTOL, f"max |dlnL|/scale = {worst:.3e}"
    if parts_gpu is not None:
        pscale = (np.hypot(parts_ref[..., 0], parts_ref[..., 1]) + parts_ref[..., 2])[..., None]
        pw = float((np.abs(parts_gpu - parts_ref) / pscale).max())
        assert pw <= LNL_RTOL, f"max parts error / scale = {pw:.3e}"
        worst = max(worst, pw)
    return worst
