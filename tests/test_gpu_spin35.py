"""`-m gpu`: spin_order = 2 (NEXT-1): spin-orbit phase terms at 2.5PN, 3PN and 3.5PN through the C-ABI
against the oracle.  Only K1's per-proposal coefficients change; the fused and waveform kernels are the default ones."""
from dataclasses import replace

import numpy as np
import pytest

from paper_1904_02863_b200 import inputs

from gpu_common import assert_h_close, assert_lnl_close, make_ctx, make_problem

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name,red", [
    ("C1", dict(f_max=1024.0, batch=300)),                  # BBH, |chi| up to 0.8: the new terms move the phase by ~10 rad
    ("C2", dict(f_max=500.0, duration_s=4.0, batch=150)),   # BNS, |chi| <= 0.05
    ("C3", dict(f_max=200.0, duration_s=8.0, batch=40)),    # from 10 Hz, multi-lane layout
])
def test_spin_order_2_lnl_and_waveform(oracle, name, red):
    import torch
    cfg = replace(inputs.CONFIGS[name].reduced(**red), spin_order=2)
    f, S, dets, d, th = make_problem(oracle, cfg)           # the injection carries the same terms
    with make_ctx(cfg, f, d, S, dets) as ctx:
        thd = torch.from_numpy(th).cuda()
        lnl, parts = ctx.lnl_batch(thd, want_parts=True)
        h = ctx.waveform_batch(thd[:24].contiguous())
        torch.cuda.synchronize()
        lnl, parts, h = lnl.cpu().numpy(), parts.cpu().numpy(), h.cpu().numpy()
    lnl_ref, parts_ref, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, 2)
    assert_lnl_close(lnl, parts, lnl_ref, parts_ref)
    assert_h_close(h, oracle.waveform(f, dets, cfg.gmst, th[:24], 2))
    assert parts_ref[0, :, 0].sum() > 0.8 * parts_ref[0, :, 2].sum()        # the injection row is recovered
    lnl_1, _, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, 1)
    assert not np.allclose(lnl, lnl_1, rtol=1e-6)                            # the option does something


def test_spin_order_2_zero_spins_equal_spin_order_0_bits(oracle):
    """With chi1 = chi2 = 0 the three spin orders give identical bits (the added terms are exact zeros)."""
    import torch
    from paper_1904_02863_b200 import GwContext
    cfg = inputs.CONFIGS["C1"].reduced(f_max=300.0, batch=200)
    f, S, dets, d, th = make_problem(oracle, cfg)
    th = th.copy(); th[:, inputs.P_CHI1] = 0.0; th[:, inputs.P_CHI2] = 0.0
    outs = []
    for order in (0, 1, 2):
        with GwContext(f, d, S, dets, cfg.gmst, spin_order=order, max_batch=200) as ctx:
            outs.append(ctx.lnl_batch(torch.from_numpy(th).cuda()).cpu().numpy())
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])


def test_spin_order_2_with_all_options(oracle):
    """spin_order 2 + tidal_order 2 + isco_cut + phase_marginal compose."""
    import torch
    from paper_1904_02863_b200 import GwContext
    from gpu_common import LNL_RTOL
    cfg = inputs.CONFIGS["C2"].reduced(f_max=700.0, duration_s=2.0, batch=140)
    f, S, dets, d, th = make_problem(oracle, cfg)
    th = th.copy(); th[:, inputs.P_MC] *= 6.0
    th[:, inputs.P_CHI1] *= 10.0; th[:, inputs.P_CHI2] *= 10.0            # |chi| up to 0.5
    lam = inputs.tidal_lambdas(cfg)
    with GwContext(f, d, S, dets, cfg.gmst, spin_order=2, max_batch=140, tidal_order=2, isco_cut=1,
                   phase_marginal=1) as ctx:
        lnl, parts = ctx.lnl_batch(torch.from_numpy(np.hstack([th, lam])).cuda(), want_parts=True)
        lnl, parts = lnl.cpu().numpy(), parts.cpu().numpy()
    _, parts_ref, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, 2, isco_cut=1, lambdas=lam, tidal_order=2)
    marg_ref = oracle.lnl_phase_marginal(parts_ref)
    scale = np.abs(parts_ref[..., 0].sum(axis=1)) + parts_ref[..., 2].sum(axis=1)
    assert (np.abs(lnl - marg_ref) / scale).max() <= LNL_RTOL
    pscale = (np.hypot(parts_ref[..., 0], parts_ref[..., 1]) + parts_ref[..., 2])[..., None]
    assert (np.abs(parts - parts_ref) / pscale).max() <= LNL_RTOL
