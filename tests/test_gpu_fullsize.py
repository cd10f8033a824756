"""`-m gpu`: the five BASELINE.json workloads at FULL size, in the launch configuration bench.py times.
The oracle cannot finish the full batches in seconds, so each run is checked (i) on sampled proposals the
oracle computes one by one, and (ii) by properties that hold for every proposal at any size:
Cauchy-Schwarz lnL <= 1/2 <d|d>, <h|h> > 0, finite outputs, run-to-run identical bits."""
import numpy as np
import pytest

from paper_1904_02863_b200 import inputs

from gpu_common import assert_h_close, assert_lnl_close, make_ctx, make_problem

pytestmark = pytest.mark.gpu

_cache = {}


def _problem(oracle, name):
    key = name                                  # C4 is the C1 shape with its own seeds
    if key not in _cache:
        _cache.clear()                          # keep at most one (C3 is ~100 MB of tables)
        _cache[key] = make_problem(oracle, inputs.CONFIGS[name])
    return _cache[key]


def _sample(n, k, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    fixed = [0, 1, n - 1] if n >= 3 else list(range(n))
    extra = rng.choice(n, size=min(k, n), replace=False).tolist() if n > 3 else []
    return np.array(sorted(set(fixed + extra)))


CASES = [("C0", 256, 256), ("C1", 4096, 48), ("C2", 1024, 10), ("C3", 256, 5),
         ("C4", 1, 1), ("C4", 16, 16), ("C4", 256, 32), ("C4", 4096, 32), ("C4", 65536, 48)]


@pytest.mark.parametrize("name,batch,n_sample", CASES, ids=[f"{c[0]}-B{c[1]}" for c in CASES])
def test_lnl_full_size(oracle, name, batch, n_sample):
    import torch
    cfg = inputs.CONFIGS[name]
    f, S, dets, d, th_all = _problem(oracle, name)
    th = th_all[:batch]
    with make_ctx(cfg, f, d, S, dets, max_batch=batch) as ctx:
        thd = torch.from_numpy(th).cuda()
        lnl, parts = ctx.lnl_batch(thd, want_parts=True)
        lnl2, parts2 = ctx.lnl_batch(thd, want_parts=True)
        torch.cuda.synchronize()
        assert torch.equal(lnl, lnl2) and torch.equal(parts, parts2)
        lnl, parts = lnl.cpu().numpy(), parts.cpu().numpy()
        plan = ctx.plan(batch)
    assert np.all(np.isfinite(lnl)) and np.all(np.isfinite(parts)) and np.all(parts[..., 2] > 0)
    dd = sum(oracle.inner(cfg.delta_f, d[i], d[i], S[i]).real for i in range(cfg.n_det))
    assert np.all(lnl <= 0.5 * dd)
    idx = _sample(batch, n_sample, 1000 + batch)
    lnl_ref, parts_ref, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th[idx], cfg.spin_order)
    worst = assert_lnl_close(lnl[idx], parts[idx], lnl_ref, parts_ref)
    print(f"{name} B={batch} plan={plan} sampled={len(idx)} worst_rel={worst:.2e}")


WCASES = [("C0", 256, 256), ("C1", 4096, 12), ("C2", 24, 3), ("C3", 8, 2)]


@pytest.mark.parametrize("name,batch,n_sample", WCASES, ids=[f"{c[0]}-B{c[1]}" for c in WCASES])
def test_waveform_full_size(oracle, name, batch, n_sample):
    """gw_waveform_batch on the full band; C1 on its full 4096-proposal batch (1.6 GB of h), the long-signal
    configs on a slab of proposals (their full outputs are 12.8 GB / 12.8 GB)."""
    import torch
    cfg = inputs.CONFIGS[name]
    f, S, dets, d, th_all = _problem(oracle, name)
    th = th_all[:batch]
    with make_ctx(cfg, f, d, S, dets, max_batch=batch) as ctx:
        h = ctx.waveform_batch(torch.from_numpy(th).cuda())
        torch.cuda.synchronize()
        idx = _sample(batch, n_sample, 2000 + batch)
        h_gpu = h[torch.from_numpy(idx).cuda()].cpu().numpy()
        finite = bool(torch.isfinite(torch.view_as_real(h)).all())
        del h
    assert finite
    h_ref = oracle.waveform(f, dets, cfg.gmst, th[idx], cfg.spin_order)
    worst = assert_h_close(h_gpu, h_ref)
    print(f"{name} B={batch} sampled={len(idx)} worst |dh|/max|h| = {worst:.2e}")


@pytest.mark.parametrize("name,batch,n_sample", [("C2", 1024, 6), ("C3", 256, 3)], ids=["C2-tidal", "C3-tidal"])
def test_lnl_full_size_tidal(oracle, name, batch, n_sample):
    """The neutron-star workloads at full size with the tidal option (NEXT-1; 13-column theta, TIDAL kernel variant),
    same data as above (a point-mass injection), sampled proposals against the oracle + run-to-run identical bits."""
    import torch
    from paper_1904_02863_b200 import GwContext
    cfg = inputs.CONFIGS[name]
    f, S, dets, d, th_all = _problem(oracle, name)
    th, lam = th_all[:batch], inputs.tidal_lambdas(cfg, batch)
    th13 = np.ascontiguousarray(np.hstack([th, lam]))
    with GwContext(f, d, S, dets, cfg.gmst, spin_order=cfg.spin_order, max_batch=batch, tidal_order=2) as ctx:
        thd = torch.from_numpy(th13).cuda()
        lnl, parts = ctx.lnl_batch(thd, want_parts=True)
        lnl2, parts2 = ctx.lnl_batch(thd, want_parts=True)
        torch.cuda.synchronize()
        assert torch.equal(lnl, lnl2) and torch.equal(parts, parts2)
        lnl, parts = lnl.cpu().numpy(), parts.cpu().numpy()
    assert np.all(np.isfinite(lnl)) and np.all(parts[..., 2] > 0)
    idx = _sample(batch, n_sample, 3000 + batch)
    lnl_ref, parts_ref, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th[idx], cfg.spin_order,
                                       lambdas=lam[idx], tidal_order=2)
    worst = assert_lnl_close(lnl[idx], parts[idx], lnl_ref, parts_ref)
    print(f"{name} tidal B={batch} sampled={len(idx)} worst_rel={worst:.2e}")
