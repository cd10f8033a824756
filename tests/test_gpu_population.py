"""`-m gpu`: the population likelihood (Eq. 3; include/gwpop.h) through the C-ABI against the oracle, Lambda by
Lambda, on the seeded synthetic catalogues P0 (small), P1 (2e5 samples, the GWTC-1 size of PAPER.md:119) and P2 (4e6
samples) -- every Lambda of the batch, at the sizes and in the launch configuration bench.py times.
Tolerance: |d lnL| <= 1e-10 (|lnL| + N)."""
import numpy as np
import pytest

from paper_1904_02863_b200 import inputs

pytestmark = pytest.mark.gpu

POP_RTOL = 1e-10


def _assert_close(got, ref, n_events):
    finite = np.isfinite(ref)
    assert np.array_equal(np.isnan(got), np.isnan(ref)) and np.array_equal(got == -np.inf, ref == -np.inf)
    err = np.abs(got[finite] - ref[finite]) / (np.abs(ref[finite]) + n_events)
    worst = float(err.max()) if err.size else 0.0
    assert worst <= POP_RTOL, f"max |dlnL| / (|lnL| + N) = {worst:.3e}"
    return worst


@pytest.mark.parametrize("name", ["P0", "P1", "P2"])
def test_population_lnl_every_lambda(oracle, name):
    import torch
    from paper_1904_02863_b200.population import GwPopContext
    cfg = inputs.POP_CONFIGS[name]
    s, p0 = inputs.pop_samples(cfg)
    lam = inputs.pop_lambdas(cfg)
    if name == "P2":
        lam = lam[:16]                                   # the oracle needs ~2 s per Lambda on 4e6 samples
    ref, _, _ = oracle.pop_lnl(s, p0, lam)
    assert np.all(np.isfinite(ref))
    with GwPopContext(s, p0, max_batch=len(lam)) as ctx:
        lam_d = torch.from_numpy(lam).cuda()
        out = ctx.lnl_batch(lam_d)
        again = ctx.lnl_batch(lam_d)
        torch.cuda.synchronize()
        assert torch.equal(out, again)                   # run-to-run identical bits
        got = out.cpu().numpy()
        # one Lambda per call (the sampler's pattern, TL = 1 kernel) and pairs (TL = 2) agree with the batched pass
        one = np.array([ctx.lnl_batch(lam_d[k:k + 1].contiguous()).item() for k in range(min(4, len(lam)))])
        two = ctx.lnl_batch(lam_d[:2].contiguous()).cpu().numpy()
        host = ctx.lnl_batch_host(lam)
        info = ctx.info()
    worst = _assert_close(got, ref, cfg.n_events)
    assert np.array_equal(one, got[:len(one)]) and np.array_equal(two, got[:2]) and np.array_equal(host, got)
    print(f"{name}: {cfg.n_events} x {cfg.n_samples} samples, {len(lam)} Lambdas, chunks/event {info['chunks_per_event']}, "
          f"worst |dlnL|/(|lnL|+N) = {worst:.2e}")


def test_population_edge_cases(oracle):
    """Ragged sizes (n not a multiple of the chunk, a single sample, a single event), the removable singularities
    alpha = 1 and beta_q = -1, beta_q < -1, lam = 0 / 1, xi = 0 / 1, invalid Lambda (NaN) and empty support (-inf)."""
    import torch
    from paper_1904_02863_b200.population import GwPopContext
    base = np.array([2.35, 5.0, 70.0, 0.1, 33.0, 5.0, 1.3, 2.0, 4.0, 0.6, 1.0, 1.5])
    rows = [base]
    for k, v in ((0, 1.0), (0, -1.5), (6, -1.0), (6, -2.5), (3, 0.0), (3, 1.0), (9, 0.0), (9, 1.0), (7, 0.7), (8, 0.6)):
        r = base.copy(); r[k] = v; rows.append(r)
    bad1 = base.copy(); bad1[2] = 4.0                    # m_max < m_min
    bad2 = base.copy(); bad2[10] = 0.0                   # sigma = 0
    bad3 = base.copy(); bad3[4] = np.nan
    empty = base.copy(); empty[1], empty[2] = 96.0, 99.0  # no sample above 95 Msun
    lam = np.stack(rows + [bad1, bad2, bad3, empty])
    for n_events, n_samples in ((1, 1), (3, 1000), (2, 1025), (7, 2049), (130, 37)):
        cfg = inputs.PopConfig("t", 9, n_events, n_samples, len(lam))
        s, p0 = inputs.pop_samples(cfg)
        ref, _, _ = oracle.pop_lnl(s, p0, lam)
        with GwPopContext(s, p0, max_batch=len(lam)) as ctx:
            got = ctx.lnl_batch(torch.from_numpy(lam).cuda()).cpu().numpy()
            dev = GwPopContext(torch.from_numpy(s).cuda(), torch.from_numpy(p0).cuda(), max_batch=len(lam))
            got_dev = dev.lnl_batch(torch.from_numpy(lam).cuda()).cpu().numpy()
            dev.close()
        assert np.all(np.isnan(got[-4:-1])) and got[-1] == -np.inf
        _assert_close(got, ref, n_events)
        assert np.array_equal(got, got_dev, equal_nan=True)       # device-resident inputs: the same bits


def test_population_rejects_bad_inputs():
    import torch
    from paper_1904_02863_b200.binding import GW_ERR_INVALID_ARG, GwError
    from paper_1904_02863_b200.population import GwPopContext
    cfg = inputs.PopConfig("t", 8, 2, 300, 4)
    s, p0 = inputs.pop_samples(cfg)
    for k, v in ((0, -1.0), (1, 1.5), (2, 0.0), (3, 1.0), (4, 1.2), (5, np.nan)):
        bad = s.copy(); bad[1, 17, k] = v
        with pytest.raises(GwError) as ei:
            GwPopContext(bad, p0)
        assert ei.value.code == GW_ERR_INVALID_ARG
    badp = p0.copy(); badp[0, 3] = 0.0
    with pytest.raises(GwError):
        GwPopContext(s, badp)
    with GwPopContext(s, p0, max_batch=4) as ctx:
        lam = torch.from_numpy(inputs.pop_lambdas(inputs.POP_CONFIGS["P0"])[:5]).cuda()
        with pytest.raises(GwError):
            ctx.lnl_batch(lam)                                       # more proposals than reserved
        assert ctx.lnl_batch(lam[:0].contiguous()).numel() == 0     # empty batch: GW_OK, nothing written
        n0 = ctx.launch_count()
        ctx.lnl_batch(lam[:4].contiguous())
        torch.cuda.synchronize()
        assert ctx.launch_count() == n0 + 3                          # setup + main + finish
