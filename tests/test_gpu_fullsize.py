"""`-m gpu`: the five BASELINE.json workloads at FULL size, in the launch configuration bench.py times, against the
oracle on EVERY proposal (SURVEY.md section 9 gate 3: "every proposal, all five configs"; the oracle needs 1-11 s per
workload on the box's host cores).  On top of the element-by-element comparison each run is checked by properties that
hold for every proposal at any size: Cauchy-Schwarz lnL <= 1/2 <d|d>, <h|h> > 0, finite outputs, run-to-run identical
bits.  Waveform parity: all rows of C0; the first 64 and the last 64 rows of C1 and of the C2 / C3 batches (SURVEY.md
8(d): "all of C0; first 64 + last 64 rows elsewhere", which keeps the host buffers at a few GB).  The NEXT-1 options
(isco_cut, phase_marginal, spin_order 2, tidal_order 2) are run at full size on C1 and C2 (tidal: C2 and C3)."""
import numpy as np
import pytest

from paper_1904_02863_b200 import inputs

from gpu_common import LNL_RTOL, assert_h_close, assert_lnl_close, make_problem

pytestmark = pytest.mark.gpu

_cache = {}
_ref_cache = {}


def _problem(oracle, name):
    key = name                                  # C4 is the C1 shape with its own seeds
    if key not in _cache:
        _cache.clear()                          # keep at most one (C3 is ~100 MB of tables)
        _ref_cache.clear()
        _cache[key] = make_problem(oracle, inputs.CONFIGS[name])
    return _cache[key]


def _oracle_lnl(oracle, name, batch, spin_order=None, isco_cut=0, lambdas=None, tidal_order=0):
    """Oracle lnL and parts of the first `batch` proposals of a workload -- every proposal -- cached per option set
    (the C4 sweep reuses prefixes of its 65 536-row run)."""
    cfg = inputs.CONFIGS[name]
    f, S, dets, d, th_all = _problem(oracle, name)
    so = cfg.spin_order if spin_order is None else spin_order
    key = (name, so, isco_cut, tidal_order)
    if key not in _ref_cache or len(_ref_cache[key][0]) < batch:
        kw = dict(lambdas=lambdas[:batch], tidal_order=tidal_order) if tidal_order else {}
        lnl, parts, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th_all[:batch], so, isco_cut=isco_cut, **kw)
        _ref_cache[key] = (lnl, parts)
    lnl, parts = _ref_cache[key]
    return lnl[:batch], parts[:batch]


def _ctx(cfg, f, d, S, dets, batch, **kw):
    from paper_1904_02863_b200 import GwContext
    kw.setdefault("spin_order", cfg.spin_order)
    return GwContext(f, d, S, dets, cfg.gmst, max_batch=batch, **kw)


def _run_twice(ctx, th):
    """lnL and parts of one gw_lnl_batch call in the planner's own launch shape, asserted bit-identical to a repeat."""
    import torch
    thd = torch.from_numpy(np.ascontiguousarray(th)).cuda()
    lnl, parts = ctx.lnl_batch(thd, want_parts=True)
    lnl2, parts2 = ctx.lnl_batch(thd, want_parts=True)
    torch.cuda.synchronize()
    assert torch.equal(lnl, lnl2) and torch.equal(parts, parts2)
    return lnl.cpu().numpy(), parts.cpu().numpy()


# the C4 sweep runs from the largest batch down so that the oracle's 65 536-row pass is computed once
CASES = [("C0", 256), ("C1", 4096), ("C2", 1024), ("C3", 256),
         ("C4", 65536), ("C4", 4096), ("C4", 256), ("C4", 16), ("C4", 1)]


@pytest.mark.parametrize("name,batch", CASES, ids=[f"{c[0]}-B{c[1]}" for c in CASES])
def test_lnl_full_size_every_proposal(oracle, name, batch):
    cfg = inputs.CONFIGS[name]
    f, S, dets, d, th_all = _problem(oracle, name)
    th = th_all[:batch]
    with _ctx(cfg, f, d, S, dets, batch) as ctx:
        lnl, parts = _run_twice(ctx, th)
        plan = ctx.plan(batch)
    assert np.all(np.isfinite(lnl)) and np.all(np.isfinite(parts)) and np.all(parts[..., 2] > 0)
    dd = sum(oracle.inner(cfg.delta_f, d[i], d[i], S[i]).real for i in range(cfg.n_det))
    assert np.all(lnl <= 0.5 * dd)
    lnl_ref, parts_ref = _oracle_lnl(oracle, name, batch)
    worst = assert_lnl_close(lnl, parts, lnl_ref, parts_ref)
    print(f"{name} B={batch} plan={plan} compared={len(lnl)} (every proposal) worst_rel={worst:.2e}")


OPTION_CASES = [("C1", "isco_cut"), ("C2", "isco_cut"), ("C1", "phase_marginal"), ("C2", "phase_marginal"),
                ("C1", "spin_order_2"), ("C2", "spin_order_2")]


@pytest.mark.parametrize("name,option", OPTION_CASES, ids=[f"{c[0]}-{c[1]}" for c in OPTION_CASES])
def test_lnl_full_size_options_every_proposal(oracle, name, option):
    """One NEXT-1 option at a time on the headline workload C1 and the long-signal workload C2, at full size, in the
    planner's launch shape, every proposal against the oracle."""
    cfg = inputs.CONFIGS[name]
    batch = cfg.batch
    f, S, dets, d, th = _problem(oracle, name)
    kw = {"isco_cut": dict(isco_cut=1), "phase_marginal": dict(phase_marginal=1),
          "spin_order_2": dict(spin_order=2)}[option]
    with _ctx(cfg, f, d, S, dets, batch, **kw) as ctx:
        lnl, parts = _run_twice(ctx, th)
    assert np.all(np.isfinite(lnl)) and np.all(np.isfinite(parts))
    lnl_ref, parts_ref = _oracle_lnl(oracle, name, batch, spin_order=kw.get("spin_order"),
                                     isco_cut=kw.get("isco_cut", 0))
    if option == "phase_marginal":
        lnl_ref = oracle.lnl_phase_marginal(parts_ref)
    if option == "isco_cut":            # every proposal keeps some bins (f_ISCO >= 44.6 Hz > f_min), so <h|h> > 0
        assert np.all(parts_ref[..., 2] > 0) and np.all(parts[..., 2] > 0)
    worst = assert_lnl_close(lnl, parts, lnl_ref, parts_ref)
    print(f"{name} {option} B={batch} compared={len(lnl)} worst_rel={worst:.2e}")


@pytest.mark.parametrize("name", ["C2", "C3"], ids=["C2-tidal", "C3-tidal"])
def test_lnl_full_size_tidal_every_proposal(oracle, name):
    """The neutron-star workloads at full size with the tidal option (NEXT-1; 13-column theta, TIDAL kernel variant),
    same data as above (a point-mass injection), every proposal against the oracle + run-to-run identical bits."""
    cfg = inputs.CONFIGS[name]
    batch = cfg.batch
    f, S, dets, d, th = _problem(oracle, name)
    lam = inputs.tidal_lambdas(cfg, batch)
    th13 = np.ascontiguousarray(np.hstack([th[:batch], lam]))
    with _ctx(cfg, f, d, S, dets, batch, tidal_order=2) as ctx:
        lnl, parts = _run_twice(ctx, th13)
    assert np.all(np.isfinite(lnl)) and np.all(parts[..., 2] > 0)
    lnl_ref, parts_ref = _oracle_lnl(oracle, name, batch, lambdas=lam, tidal_order=2)
    worst = assert_lnl_close(lnl, parts, lnl_ref, parts_ref)
    print(f"{name} tidal B={batch} compared={len(lnl)} (every proposal) worst_rel={worst:.2e}")


WCASES = [("C0", 256, 256), ("C1", 4096, 64), ("C2", 1024, 64), ("C3", 256, 64)]


@pytest.mark.parametrize("name,batch,edge", WCASES, ids=[f"{c[0]}-B{c[1]}" for c in WCASES])
def test_waveform_full_size(oracle, name, batch, edge):
    """gw_waveform_batch on the full band, elementwise against the oracle: all rows of C0; the first `edge` and the
    last `edge` rows of the C1, C2 and C3 batches.  C1 is computed on its full 4096-proposal batch (1.6 GB of h) and
    the two row groups are read out of it; the long-signal configs compute each row group with a call of its own
    (their full outputs are 12.8 GB), which uses the same kernel, the same proposal-block size and the same theta."""
    import torch
    cfg = inputs.CONFIGS[name]
    f, S, dets, d, th_all = _problem(oracle, name)
    th = th_all[:batch]
    groups = [np.arange(batch)] if edge >= batch else [np.arange(edge), np.arange(batch - edge, batch)]
    whole = cfg.n_det * cfg.n_bins * batch * 16 <= (2 << 30)
    worst, rows = 0.0, 0
    with _ctx(cfg, f, d, S, dets, batch) as ctx:
        h_all = None
        if whole:
            h_all = ctx.waveform_batch(torch.from_numpy(th).cuda())
            torch.cuda.synchronize()
            assert bool(torch.isfinite(torch.view_as_real(h_all)).all())
        for idx in groups:
            if whole:
                h_gpu = h_all[torch.from_numpy(idx).cuda()].cpu().numpy()
            else:
                h = ctx.waveform_batch(torch.from_numpy(np.ascontiguousarray(th[idx])).cuda())
                torch.cuda.synchronize()
                assert bool(torch.isfinite(torch.view_as_real(h)).all())
                h_gpu = h.cpu().numpy()
                del h
            h_ref = oracle.waveform(f, dets, cfg.gmst, th[idx], cfg.spin_order)
            worst = max(worst, assert_h_close(h_gpu, h_ref))
            rows += len(idx)
            del h_gpu, h_ref
        del h_all
    print(f"{name} B={batch} rows compared={rows} worst |dh|/max|h| = {worst:.2e}")
