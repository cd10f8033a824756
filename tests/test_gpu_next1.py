"""`-m gpu`: the NEXT-1 options through the C-ABI against the oracle: inspiral cut-off at f_ISCO
(`gw_options.isco_cut`) and the phase-marginalised likelihood (`gw_options.phase_marginal`)."""
import numpy as np
import pytest

from paper_1904_02863_b200 import inputs

from gpu_common import LNL_RTOL, assert_h_close, assert_lnl_close, make_problem

pytestmark = pytest.mark.gpu


def _ctx(cfg, f, d, S, dets, **kw):
    from paper_1904_02863_b200 import GwContext
    return GwContext(f, d, S, dets, cfg.gmst, spin_order=cfg.spin_order, max_batch=max(cfg.batch, 1), **kw)


@pytest.mark.parametrize("name,red", [
    ("C1", dict(f_max=2048.0, batch=300)),        # BBH: f_ISCO 45-110 Hz, deep inside the band; 2 tiles, several chunks
    ("C0", dict(f_max=512.0, batch=256)),         # 1 fixed detector
    ("C2", dict(f_max=40.0, batch=40)),           # BNS: f_ISCO above the band -> identical to the uncut result
])
def test_isco_cut_lnl_and_waveform(oracle, name, red):
    import torch
    cfg = inputs.CONFIGS[name].reduced(**red)
    f, S, dets, d, th = make_problem(oracle, cfg)
    with _ctx(cfg, f, d, S, dets, isco_cut=1) as ctx:
        thd = torch.from_numpy(th).cuda()
        lnl, parts = ctx.lnl_batch(thd, want_parts=True)
        h = ctx.waveform_batch(thd[:24].contiguous())
        torch.cuda.synchronize()
        lnl, parts, h = lnl.cpu().numpy(), parts.cpu().numpy(), h.cpu().numpy()
    lnl_ref, parts_ref, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, cfg.spin_order, isco_cut=1)
    assert_lnl_close(lnl, parts, lnl_ref, parts_ref)
    h_ref = oracle.waveform(f, dets, cfg.gmst, th[:24], cfg.spin_order, isco_cut=1)
    assert np.array_equal(h == 0, h_ref == 0)                     # the same bins are cut (fp64 decision on both sides)
    assert_h_close(h, h_ref)
    if name != "C2":
        uncut, _, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, cfg.spin_order)
        assert not np.allclose(lnl, uncut, rtol=1e-6)              # the option does something


@pytest.mark.parametrize("batch", [1, 7, 33, 300])
def test_isco_cut_all_lane_layouts(oracle, batch):
    import torch
    cfg = inputs.CONFIGS["C1"].reduced(f_max=301.25, batch=300)
    f, S, dets, d, th = make_problem(oracle, cfg)
    with _ctx(cfg, f, d, S, dets, isco_cut=1) as ctx:
        lnl, parts = ctx.lnl_batch(torch.from_numpy(th[:batch]).cuda(), want_parts=True)
        torch.cuda.synchronize()
    ref = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th[:batch], cfg.spin_order, isco_cut=1)
    assert_lnl_close(lnl.cpu().numpy(), parts.cpu().numpy(), ref[0], ref[1])


@pytest.mark.parametrize("lpp,n_chunks", [(1, 1), (1, 7), (1, 40), (4, 3), (8, 40), (32, 11)])
def test_isco_cut_skipped_stages_in_forced_plans(oracle, lpp, n_chunks):
    """Stages (and whole CTAs) above every proposal's cut-off are not swept (fused_kernel, ISCO): BBH proposals cut at
    45-110 Hz in a band up to 1024 Hz, so with 7 or 40 chunks most CTAs sweep nothing and the CTA holding the cut
    sweeps part of its stages; one light proposal (cut above the band) per tile keeps every stage of that tile alive
    in the second half of the batch."""
    import torch
    cfg = inputs.CONFIGS["C1"].reduced(f_max=1024.0, batch=520)
    f, S, dets, d, th = make_problem(oracle, cfg)
    th = th.copy()
    th[300:, inputs.P_MC] = np.where(np.arange(300, 520) % 64 == 0, 1.2, th[300:, inputs.P_MC])   # f_ISCO > 1024 Hz
    with _ctx(cfg, f, d, S, dets, isco_cut=1) as ctx:
        ctx.force_plan(lpp, n_chunks)
        plan = ctx.plan(len(th))
        assert plan["lanes_per_prop"] == lpp and plan["n_chunks"] == n_chunks
        thd = torch.from_numpy(th).cuda()
        lnl, parts = ctx.lnl_batch(thd, want_parts=True)
        again, _ = ctx.lnl_batch(thd, want_parts=True)
        torch.cuda.synchronize()
    ref = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, cfg.spin_order, isco_cut=1)
    assert_lnl_close(lnl.cpu().numpy(), parts.cpu().numpy(), ref[0], ref[1])
    assert torch.equal(lnl, again)


@pytest.mark.parametrize("isco", [0, 1])
def test_phase_marginal(oracle, isco):
    import torch
    cfg = inputs.CONFIGS["C1"].reduced(f_max=400.0, batch=300)
    f, S, dets, d, th = make_problem(oracle, cfg)
    with _ctx(cfg, f, d, S, dets, phase_marginal=1, isco_cut=isco) as ctx:
        lnl, parts = ctx.lnl_batch(torch.from_numpy(th).cuda(), want_parts=True)
        torch.cuda.synchronize()
        lnl, parts = lnl.cpu().numpy(), parts.cpu().numpy()
    _, parts_ref, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, cfg.spin_order, isco_cut=isco)
    marg_ref = oracle.lnl_phase_marginal(parts_ref)
    scale = np.abs(parts_ref[..., 0].sum(axis=1)) + parts_ref[..., 2].sum(axis=1)
    assert (np.abs(lnl - marg_ref) / scale).max() <= LNL_RTOL
    pscale = (np.hypot(parts_ref[..., 0], parts_ref[..., 1]) + parts_ref[..., 2])[..., None]
    assert (np.abs(parts - parts_ref) / pscale).max() <= LNL_RTOL
    # the marginal value does not depend on the proposal's phi_c: shift it and compare
    th2 = th.copy(); th2[:, inputs.P_PHIC] += 1.234
    with _ctx(cfg, f, d, S, dets, phase_marginal=1, isco_cut=isco) as ctx:
        lnl2 = ctx.lnl_batch(torch.from_numpy(th2).cuda()).cpu().numpy()
    assert (np.abs(lnl2 - lnl) / scale).max() <= LNL_RTOL


def test_phase_marginal_large_snr_branch(oracle):
    """C0 at full band: the injection row has <d|h> ~ 1.2e4 > 500, which exercises the asymptotic ln I0 branch."""
    import torch
    cfg = inputs.CONFIGS["C0"]
    f, S, dets, d, th = make_problem(oracle, cfg)
    with _ctx(cfg, f, d, S, dets, phase_marginal=1) as ctx:
        lnl, parts = ctx.lnl_batch(torch.from_numpy(th).cuda(), want_parts=True)
        torch.cuda.synchronize()
        lnl, parts = lnl.cpu().numpy(), parts.cpu().numpy()
    assert np.hypot(parts[0, 0, 0], parts[0, 0, 1]) > 500.0
    _, parts_ref, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, cfg.spin_order)
    marg_ref = oracle.lnl_phase_marginal(parts_ref)
    scale = np.abs(parts_ref[..., 0].sum(axis=1)) + parts_ref[..., 2].sum(axis=1)
    assert (np.abs(lnl - marg_ref) / scale).max() <= LNL_RTOL
