"""`-m gpu`, collected last (the file name sorts after every other test file): gw_pop_lnl_static, the population
likelihood entry point that allocates nothing (include/gwpop.h) -- its scratch is a file-scope `static __device__` array
inside the library -- against the existing context path gw_pop_lnl_batch on the same device-resident inputs.  Both run
the same kernels in the same grids, so the outputs are compared within the tolerance of tests/test_gpu_population.py
(|d lnL| <= 1e-10 (|lnL| + N)) and, on top of that, bit for bit.  Each test makes two static calls in a row on one
stream with no synchronisation between them, on problems of different shapes, so that the second call runs on whatever
the first one left in the shared array.  Nothing here depends on state left by other tests: the file passes alone in a
fresh process and after the rest of the suite."""
import numpy as np
import pytest

from paper_1904_02863_b200 import inputs

pytestmark = pytest.mark.gpu

POP_RTOL = 1e-10                                             # tests/test_gpu_population.py, DESIGN.md section 14


def _problem(torch, cfg, extra_rows=()):
    s, p0 = inputs.pop_samples(cfg)
    lam = inputs.pop_lambdas(cfg)
    if len(extra_rows):
        lam = np.ascontiguousarray(np.vstack([lam] + [np.asarray(r)[None] for r in extra_rows]))
    return torch.from_numpy(s).cuda(), torch.from_numpy(p0).cuda(), torch.from_numpy(lam).cuda()


def _context_path(torch, s_d, p_d, lam_d):
    from paper_1904_02863_b200.population import GwPopContext
    with GwPopContext(s_d, p_d, max_batch=lam_d.shape[0]) as ctx:
        out = ctx.lnl_batch(lam_d)
        torch.cuda.synchronize()
        return out.cpu().numpy()


def _assert_same(got, ref, n_events):
    assert np.array_equal(np.isnan(got), np.isnan(ref)) and np.array_equal(got == -np.inf, ref == -np.inf)
    finite = np.isfinite(ref)
    assert finite.any()
    err = np.abs(got[finite] - ref[finite]) / (np.abs(ref[finite]) + n_events)
    assert float(err.max()) <= POP_RTOL, f"max |dlnL| / (|lnL| + N) = {float(err.max()):.3e}"
    assert np.array_equal(got, ref, equal_nan=True)          # same kernels, same grids, same order: the same bits


def test_static_entry_point_matches_context_path_two_calls_in_a_row():
    import torch
    from paper_1904_02863_b200 import population
    base = np.array([2.35, 5.0, 70.0, 0.1, 33.0, 5.0, 1.3, 2.0, 4.0, 0.6, 1.0, 1.5])
    invalid = base.copy(); invalid[2] = 4.0                   # m_max < m_min: NaN for that Lambda only
    empty = base.copy(); empty[1], empty[2] = 96.0, 99.0      # no sample above 95 Msun: -inf
    cfg_a = inputs.POP_CONFIGS["P0"]                          # 10 x 2000 samples, 64 Lambda
    cfg_b = inputs.PopConfig("t", 9, 7, 2049, 21)             # ragged chunk tail; smaller than A in every part
    a = _problem(torch, cfg_a)
    b = _problem(torch, cfg_b, extra_rows=(invalid, empty))
    out_a = torch.full((a[2].shape[0],), 123.0, dtype=torch.float64, device="cuda")
    out_b = torch.full((b[2].shape[0],), 123.0, dtype=torch.float64, device="cuda")
    # two calls in a row, nothing between them: the second runs on the scratch contents the first one left
    population.lnl_static(a[0], a[1], a[2], out=out_a)
    population.lnl_static(b[0], b[1], b[2], out=out_b)
    torch.cuda.synchronize()
    got_a, got_b = out_a.cpu().numpy(), out_b.cpu().numpy()
    # ... and the other order, single Lambda (TL = 1 kernel) and pairs (TL = 2) included
    one_b = population.lnl_static(b[0], b[1], b[2][:1].contiguous())
    again_a = population.lnl_static(a[0], a[1], a[2])
    two_a = population.lnl_static(a[0], a[1], a[2][:2].contiguous())
    torch.cuda.synchronize()
    ref_a, ref_b = _context_path(torch, *a), _context_path(torch, *b)
    _assert_same(got_a, ref_a, cfg_a.n_events)
    _assert_same(got_b, ref_b, cfg_b.n_events)
    assert np.isnan(got_b[-2]) and got_b[-1] == -np.inf and np.all(np.isfinite(got_b[:-2]))
    _assert_same(again_a.cpu().numpy(), ref_a, cfg_a.n_events)
    assert one_b.item() == ref_b[0] and np.array_equal(two_a.cpu().numpy(), ref_a[:2])


def test_static_entry_point_limit_bad_samples_and_bad_pointers():
    import torch
    from paper_1904_02863_b200 import population
    from paper_1904_02863_b200.binding import GW_ERR_INVALID_ARG, GwError
    cfg = inputs.PopConfig("t", 8, 3, 700, 5)
    s_d, p_d, lam_d = _problem(torch, cfg)
    ref = _context_path(torch, s_d, p_d, lam_d)
    # beyond the static array: a clear error, nothing enqueued (the P2 catalogue of 4e6 samples needs 3.2e7 doubles)
    assert population.static_need(100, 40000, 64) > population.STATIC_SCRATCH_DOUBLES
    assert 0 < population.static_need(10, 20000, 64) <= population.STATIC_SCRATCH_DOUBLES      # GWTC-1 size fits
    big_s = torch.empty((100, 40000, 6), dtype=torch.float64, device="cuda")
    big_p = torch.empty((100, 40000), dtype=torch.float64, device="cuda")
    with pytest.raises(GwError) as ei:
        population.lnl_static(big_s, big_p, lam_d)
    assert ei.value.code == population.GW_POP_ERR_TOO_LARGE and "static array holds" in str(ei.value)
    del big_s, big_p
    # host memory is not accepted (the kernels would read it through the wrong address space)
    lib = population._lib()
    host = np.zeros(3 * 700 * 6)
    out = torch.empty(5, dtype=torch.float64, device="cuda")
    assert lib.gw_pop_lnl_static(3, 700, host.ctypes.data, p_d.data_ptr(), 5, lam_d.data_ptr(), out.data_ptr(), None) == GW_ERR_INVALID_ARG
    assert lib.gw_pop_lnl_static(3, 700, s_d.data_ptr(), p_d.data_ptr(), 5, lam_d.data_ptr(), None, None) == GW_ERR_INVALID_ARG
    assert lib.gw_pop_lnl_static(0, 700, s_d.data_ptr(), p_d.data_ptr(), 5, lam_d.data_ptr(), out.data_ptr(), None) == GW_ERR_INVALID_ARG
    assert lib.gw_pop_lnl_static(3, 700, s_d.data_ptr(), p_d.data_ptr(), 0, lam_d.data_ptr(), out.data_ptr(), None) == 0
    # a sample outside the domain: every lnL of THAT call is NaN; the flag is cleared by the next call
    bad_s = s_d.clone(); bad_s[1, 17, 1] = 1.5                # q > 1
    got_bad = population.lnl_static(bad_s, p_d, lam_d)
    got_ok = population.lnl_static(s_d, p_d, lam_d)
    torch.cuda.synchronize()
    assert bool(torch.isnan(got_bad).all())
    _assert_same(got_ok.cpu().numpy(), ref, cfg.n_events)
    # a non-default stream
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(st):
        got_st = population.lnl_static(s_d, p_d, lam_d, stream=st)
    st.synchronize()
    _assert_same(got_st.cpu().numpy(), ref, cfg.n_events)
