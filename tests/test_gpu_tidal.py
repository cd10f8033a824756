"""`-m gpu`: the tidal option (NEXT-1; `gw_options.tidal_order`, theta rows of 13 columns) through the
C-ABI against the oracle: 5PN and 5PN + 6PN adiabatic tidal phase terms on the neutron-star workloads C2 / C3."""
import numpy as np
import pytest

from paper_1904_02863_b200 import inputs

from gpu_common import LNL_RTOL, assert_h_close, assert_lnl_close

pytestmark = pytest.mark.gpu


def _problem(oracle, cfg, tidal_order):
    """The config's recipe with a tidal injection: data = oracle h(theta_inj, Lambda = (400, 600)) + seeded noise."""
    f = inputs.frequency_grid(cfg)
    S = inputs.psd(cfg)
    dets = inputs.detectors(cfg)
    th = inputs.proposals(cfg)
    lam = inputs.tidal_lambdas(cfg)
    inject = lambda fr, de, gm, t, so: oracle.waveform(fr, de, gm, t, so, lambdas=lam[:1], tidal_order=tidal_order)
    d = inputs.make_data(cfg, inject)
    return f, S, dets, d, th, lam


def _ctx(cfg, f, d, S, dets, **kw):
    from paper_1904_02863_b200 import GwContext
    return GwContext(f, d, S, dets, cfg.gmst, spin_order=cfg.spin_order, max_batch=max(cfg.batch, 1), **kw)


@pytest.mark.parametrize("name,red,order", [
    ("C2", dict(f_max=2048.0, duration_s=2.0, batch=300), 2),     # full band (tides matter above ~400 Hz), 4057 bins
    ("C2", dict(f_max=2048.0, duration_s=2.0, batch=300), 1),     # 5PN only
    ("C3", dict(f_max=1500.0, duration_s=1.0, batch=70), 2),      # from 10 Hz; multi-lane layout
    ("C0", dict(f_max=512.0, batch=256), 2),                      # 1 fixed detector, BBH masses (tides tiny but coded)
])
def test_tidal_lnl_and_waveform(oracle, name, red, order):
    import torch
    cfg = inputs.CONFIGS[name].reduced(**red)
    f, S, dets, d, th, lam = _problem(oracle, cfg, order)
    th13 = np.ascontiguousarray(np.hstack([th, lam]))
    with _ctx(cfg, f, d, S, dets, tidal_order=order) as ctx:
        assert ctx.n_param == 13
        thd = torch.from_numpy(th13).cuda()
        lnl, parts = ctx.lnl_batch(thd, want_parts=True)
        again = ctx.lnl_batch(thd)
        h = ctx.waveform_batch(thd[:24].contiguous())
        torch.cuda.synchronize()
        assert torch.equal(lnl, again)
        lnl, parts, h = lnl.cpu().numpy(), parts.cpu().numpy(), h.cpu().numpy()
        lnl_host, parts_host = ctx.lnl_batch_host(th13, want_parts=True)
    lnl_ref, parts_ref, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, cfg.spin_order,
                                       lambdas=lam, tidal_order=order)
    assert_lnl_close(lnl, parts, lnl_ref, parts_ref)
    assert np.array_equal(lnl_host, lnl) and np.array_equal(parts_host, parts)
    h_ref = oracle.waveform(f, dets, cfg.gmst, th[:24], cfg.spin_order, lambdas=lam[:24], tidal_order=order)
    assert_h_close(h, h_ref)
    if name != "C0":
        # the option does something: the point-mass likelihood of the same proposals differs
        pm, _, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, cfg.spin_order)
        assert not np.allclose(lnl, pm, rtol=1e-6)
        # and the injection row (Lambda = (400, 600), the injected values) recovers <d|h> ~ <h|h>
        assert parts_ref[0, :, 0].sum() > 0.8 * parts_ref[0, :, 2].sum()


@pytest.mark.parametrize("lpp,n_chunks", [(1, 1), (1, 7), (1, 40), (2, 5), (8, 40), (32, 11)])
def test_tidal_forced_plans(oracle, lpp, n_chunks):
    """Every lane layout and the direct, single-level and two-level finish with the TIDAL kernel variant."""
    import torch
    cfg = inputs.CONFIGS["C2"].reduced(f_max=1100.0, duration_s=2.0, batch=290)
    f, S, dets, d, th, lam = _problem(oracle, cfg, 2)
    th13 = np.ascontiguousarray(np.hstack([th, lam]))
    with _ctx(cfg, f, d, S, dets, tidal_order=2) as ctx:
        ctx.force_plan(lpp, n_chunks)
        lnl, parts = ctx.lnl_batch(torch.from_numpy(th13).cuda(), want_parts=True)
        torch.cuda.synchronize()
    ref = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, cfg.spin_order, lambdas=lam, tidal_order=2)
    assert_lnl_close(lnl.cpu().numpy(), parts.cpu().numpy(), ref[0], ref[1])


def test_tidal_zero_lambda_equals_point_mass_context(oracle):
    """Lambda = 0 through the tidal kernels gives the point-mass context's numbers to rounding (the extra terms add
    exact zeros to the phase), and with isco_cut + phase_marginal on top the options compose."""
    import torch
    cfg = inputs.CONFIGS["C2"].reduced(f_max=600.0, duration_s=2.0, batch=130)
    f, S, dets, d, th, lam = _problem(oracle, cfg, 2)
    th13 = np.ascontiguousarray(np.hstack([th, np.zeros_like(lam)]))
    with _ctx(cfg, f, d, S, dets, tidal_order=2) as ctx:
        a = ctx.lnl_batch(torch.from_numpy(th13).cuda()).cpu().numpy()
    with _ctx(cfg, f, d, S, dets) as ctx:
        b = ctx.lnl_batch(torch.from_numpy(th).cuda()).cpu().numpy()
    assert np.array_equal(a, b)
    # composition with the other two options (heavy masses so that the cut-off falls inside the band)
    th = th.copy(); th[:, inputs.P_MC] *= 8.0
    th13 = np.ascontiguousarray(np.hstack([th, lam]))
    with _ctx(cfg, f, d, S, dets, tidal_order=2, isco_cut=1, phase_marginal=1) as ctx:
        lnl, parts = ctx.lnl_batch(torch.from_numpy(th13).cuda(), want_parts=True)
        lnl, parts = lnl.cpu().numpy(), parts.cpu().numpy()
    _, parts_ref, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, cfg.spin_order, isco_cut=1,
                                 lambdas=lam, tidal_order=2)
    marg_ref = oracle.lnl_phase_marginal(parts_ref)
    scale = np.abs(parts_ref[..., 0].sum(axis=1)) + parts_ref[..., 2].sum(axis=1)
    assert (np.abs(lnl - marg_ref) / scale).max() <= LNL_RTOL


def test_tidal_bad_lambda_poisons_only_its_proposal(oracle):
    import torch
    cfg = inputs.CONFIGS["C2"].reduced(f_max=100.0, duration_s=2.0, batch=40)
    f, S, dets, d, th, lam = _problem(oracle, cfg, 2)
    th13 = np.ascontiguousarray(np.hstack([th, lam]))
    bad = th13.copy()
    bad[3, 11] = -1.0
    bad[17, 12] = np.nan
    with _ctx(cfg, f, d, S, dets, tidal_order=2) as ctx:
        good = ctx.lnl_batch(torch.from_numpy(th13).cuda()).cpu().numpy()
        got = ctx.lnl_batch(torch.from_numpy(bad).cuda()).cpu().numpy()
        h = ctx.waveform_batch(torch.from_numpy(bad[:8]).cuda()).cpu().numpy()
        with pytest.raises(Exception):
            ctx.lnl_batch(torch.from_numpy(th).cuda())           # 11 columns on a 13-column context
    assert np.isnan(got[3]) and np.isnan(got[17]) and np.isnan(h[3]).all()
    keep = np.ones(len(got), bool); keep[[3, 17]] = False
    assert np.array_equal(got[keep], good[keep]) and np.isfinite(h[:3]).all()
