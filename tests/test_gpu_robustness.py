"""`-m gpu`: memory safety and API-contract checks of the CUDA path that need no oracle arithmetic beyond a
reference value (compute-sanitizer is closed on this GPU pool, so out-of-bounds writes are hunted with guard
bands around every caller-owned output buffer)."""
import numpy as np
import pytest

from paper_1904_02863_b200 import inputs

from gpu_common import assert_h_close, assert_lnl_close, make_ctx, make_problem

pytestmark = pytest.mark.gpu

GUARD = 4096          # doubles of guard band on each side
CANARY = -7.25e300


def _guarded(torch, n_doubles):
    buf = torch.full((n_doubles + 2 * GUARD,), CANARY, dtype=torch.float64, device="cuda")
    return buf, buf[GUARD:GUARD + n_doubles]


def _intact(torch, buf, n_doubles):
    return bool((buf[:GUARD] == CANARY).all()) and bool((buf[GUARD + n_doubles:] == CANARY).all())


@pytest.mark.parametrize("name,red,batches", [
    ("C1", dict(f_max=181.75, batch=600), [1, 5, 16, 33, 255, 256, 257, 600]),
    ("C0", dict(f_max=100.0, batch=300), [1, 7, 300]),
])
def test_outputs_stay_inside_their_buffers(oracle, name, red, batches):
    import torch
    cfg = inputs.CONFIGS[name].reduced(**red)
    f, S, dets, d, th = make_problem(oracle, cfg)
    with make_ctx(cfg, f, d, S, dets) as ctx:
        for B in batches:
            thd = torch.from_numpy(th[:B]).cuda()
            nl, npart, nh = B, B * cfg.n_det * 3, B * cfg.n_det * cfg.n_bins * 2
            lbuf, lnl = _guarded(torch, nl)
            pbuf, parts = _guarded(torch, npart)
            hbuf, h = _guarded(torch, nh)
            ctx.lnl_batch(thd, out=lnl, parts=parts.view(B, cfg.n_det, 3))
            ctx.waveform_batch(thd, out=torch.view_as_complex(h.view(B, cfg.n_det, cfg.n_bins, 2)))
            torch.cuda.synchronize()
            assert _intact(torch, lbuf, nl) and _intact(torch, pbuf, npart) and _intact(torch, hbuf, nh), B
            assert bool((lnl != CANARY).all()) and bool((parts != CANARY).all()) and bool((h != CANARY).all()), B


def test_non_default_stream_and_two_contexts(oracle):
    """Calls enqueue on the stream they are given; two contexts on two streams do not disturb each other."""
    import torch
    cfg_a = inputs.CONFIGS["C1"].reduced(f_max=150.0, batch=300)
    cfg_b = inputs.CONFIGS["C2"].reduced(f_max=24.0, batch=90)
    pa, pb = make_problem(oracle, cfg_a), make_problem(oracle, cfg_b)
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    with make_ctx(cfg_a, pa[0], pa[3], pa[1], pa[2]) as ca, make_ctx(cfg_b, pb[0], pb[3], pb[1], pb[2]) as cb:
        ta, tb = torch.from_numpy(pa[4]).cuda(), torch.from_numpy(pb[4]).cuda()
        torch.cuda.synchronize()
        outs_a, outs_b = [], []
        for _ in range(5):
            with torch.cuda.stream(sa):
                outs_a.append(ca.lnl_batch(ta, want_parts=True, stream=sa))
            with torch.cuda.stream(sb):
                outs_b.append(cb.lnl_batch(tb, want_parts=True, stream=sb))
        sa.synchronize(); sb.synchronize()
    ref_a = oracle.lnl(pa[0], cfg_a.delta_f, pa[3], pa[1], pa[2], cfg_a.gmst, pa[4], cfg_a.spin_order)
    ref_b = oracle.lnl(pb[0], cfg_b.delta_f, pb[3], pb[1], pb[2], cfg_b.gmst, pb[4], cfg_b.spin_order)
    for lnl, parts in outs_a:
        assert_lnl_close(lnl.cpu().numpy(), parts.cpu().numpy(), ref_a[0], ref_a[1])
        assert torch.equal(lnl, outs_a[0][0])
    for lnl, parts in outs_b:
        assert_lnl_close(lnl.cpu().numpy(), parts.cpu().numpy(), ref_b[0], ref_b[1])
        assert torch.equal(lnl, outs_b[0][0])


def test_reserve_growth_keeps_results(oracle):
    """gw_ctx_reserve reallocates the workspace; results before and after are identical bits for the same plan."""
    import torch
    cfg = inputs.CONFIGS["C1"].reduced(f_max=200.0, batch=1000)
    f, S, dets, d, th = make_problem(oracle, cfg)
    with make_ctx(cfg, f, d, S, dets, max_batch=64) as ctx:
        thd = torch.from_numpy(th).cuda()
        small = ctx.lnl_batch(thd[:64].contiguous()).clone()
        ctx.reserve(1000)
        again = ctx.lnl_batch(thd[:64].contiguous())
        full, parts = ctx.lnl_batch(thd, want_parts=True)
        torch.cuda.synchronize()
        assert torch.equal(small, again)
        ctx.reserve(10)                                   # never shrinks
        assert ctx.info()["max_batch"] == 1000
    ref = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, cfg.spin_order)
    assert_lnl_close(full.cpu().numpy(), parts.cpu().numpy(), ref[0], ref[1])


def test_nan_rows_in_every_lane_layout(oracle):
    """An out-of-domain proposal poisons only its own outputs, whatever the lanes-per-proposal layout."""
    import torch
    cfg = inputs.CONFIGS["C1"].reduced(f_max=301.25, batch=600)
    f, S, dets, d, th = make_problem(oracle, cfg)
    with make_ctx(cfg, f, d, S, dets) as ctx:
        for B in (2, 9, 40, 300, 600):
            bad = th[:B].copy()
            bad[B // 2, inputs.P_MC] = -3.0
            good = ctx.lnl_batch(torch.from_numpy(th[:B]).cuda()).cpu().numpy()
            got = ctx.lnl_batch(torch.from_numpy(bad).cuda()).cpu().numpy()
            assert np.isnan(got[B // 2])
            keep = np.arange(B) != B // 2
            assert np.array_equal(got[keep], good[keep]), B


def test_launch_count_and_plan_are_stable(oracle):
    import torch
    cfg = inputs.CONFIGS["C1"].reduced(f_max=120.0, batch=64)
    f, S, dets, d, th = make_problem(oracle, cfg)
    with make_ctx(cfg, f, d, S, dets) as ctx:
        n0 = ctx.launch_count()                           # precompute + norm
        assert n0 == 2
        thd = torch.from_numpy(th).cuda()
        ctx.lnl_batch(thd)
        ctx.waveform_batch(thd)
        torch.cuda.synchronize()
        assert ctx.launch_count() == n0 + 4               # (setup + fused) + (setup + waveform)
        assert ctx.plan(64) == ctx.plan(64)


def test_batch_call_is_capturable_in_a_cuda_graph(oracle):
    """The batch calls neither allocate nor synchronise nor copy (PAPER.md:45/:49 lesson), so one can be captured
    in a CUDA graph; replays give the same bits, and follow new theta written into the captured buffer."""
    import torch
    cfg = inputs.CONFIGS["C1"].reduced(f_max=150.0, batch=40)
    f, S, dets, d, th = make_problem(oracle, cfg)
    with make_ctx(cfg, f, d, S, dets) as ctx:
        thd = torch.from_numpy(th).cuda()
        out = torch.empty(40, dtype=torch.float64, device="cuda")
        eager = ctx.lnl_batch(thd).clone()
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        g = torch.cuda.CUDAGraph()
        with torch.cuda.stream(side):
            ctx.lnl_batch(thd, out=out, stream=side)
            with torch.cuda.graph(g, stream=side):
                ctx.lnl_batch(thd, out=out, stream=side)
        torch.cuda.current_stream().wait_stream(side)
        out.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(out, eager)
        thd.copy_(torch.from_numpy(th[::-1].copy()).cuda())
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(out, eager.flip(0))


def test_sub_band_contexts_add_up(oracle):
    """Bin sharding (sharding.bin_shard_edges): contexts built on contiguous sub-bands give parts whose sum is the
    full-band result (what a bin-sharded multi-GPU run exchanges)."""
    import torch
    from paper_1904_02863_b200 import GwContext
    from paper_1904_02863_b200.sharding import bin_shard_edges, lnl_from_parts
    cfg = inputs.CONFIGS["C2"].reduced(f_max=30.0, batch=48)              # 1281 bins
    f, S, dets, d, th = make_problem(oracle, cfg)
    thd = torch.from_numpy(th).cuda()
    total = None
    for lo, hi in bin_shard_edges(cfg.n_bins, 3):
        with GwContext(f[lo:hi], d[:, lo:hi], S[:, lo:hi], dets, cfg.gmst, max_batch=48) as ctx:
            _, parts = ctx.lnl_batch(thd, want_parts=True)
            torch.cuda.synchronize()
            total = parts.clone() if total is None else total + parts
    with make_ctx(cfg, f, d, S, dets) as ctx:
        full_lnl, full_parts = ctx.lnl_batch(thd, want_parts=True)
        torch.cuda.synchronize()
    ref = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, cfg.spin_order)
    assert_lnl_close(lnl_from_parts(total).cpu().numpy(), total.cpu().numpy(), ref[0], ref[1])
    assert_lnl_close(full_lnl.cpu().numpy(), full_parts.cpu().numpy(), ref[0], ref[1])


@pytest.mark.gpu
def test_one_cta_per_sm_grids_are_not_doubled_up(oracle):
    """DESIGN.md section 7, exclusive grids: a plan of at most one CTA per SM must take the same time whether
    or not another kernel is still resident when it is launched (setup kernel under programmatic dependent
    launch, the L2 flush before it).  Unprotected, the step took 1.7x the two kernels' own time."""
    import torch
    cfg = inputs.CONFIGS["C1"]
    f, S, dets, d, th = make_problem(oracle, cfg)
    ctx = make_ctx(cfg, f, d, S, dets)
    B = cfg.batch
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    ctx.force_plan(1, max(1, n_sm // ((B + 255) // 256)))      # 16 tiles x 9 chunks = 144 CTAs on 148 SMs
    assert ctx.plan(B)["n_ctas"] <= n_sm
    thd = torch.from_numpy(th[:B]).cuda()
    lnl = torch.empty(B, dtype=torch.float64, device="cuda")
    busy = torch.empty(64 << 20, dtype=torch.uint8, device="cuda")
    for _ in range(5):
        ctx.lnl_batch(thd, out=lnl)
    ctx.kernel_timing(True)
    alone = []
    for _ in range(10):
        ctx.lnl_batch(thd, out=lnl)
        k1, k3 = ctx.last_kernel_ms()
        alone.append(k1 + k3)
    ctx.kernel_timing(False)
    steps = []
    for _ in range(30):
        busy.fill_(1)                                          # still draining when the step's kernels launch
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); ctx.lnl_batch(thd, out=lnl); e1.record()
        torch.cuda.synchronize()
        steps.append(e0.elapsed_time(e1))
    assert np.median(steps) < 1.35 * np.median(alone), (np.median(steps), np.median(alone))


@pytest.mark.parametrize("seed", range(3))
def test_call_sequences_leave_no_state_behind(oracle, seed):
    """Tickets, group tickets and partial sums are reused from call to call (self-resetting counters): a random
    sequence of batch sizes and pinned launch shapes on ONE context must give, call by call, the bits a fresh
    context gives for the same call."""
    import torch
    from paper_1904_02863_b200 import GwError
    cfg = inputs.CONFIGS["C1"].reduced(f_max=332.5, batch=700)        # 1251 bins
    f, S, dets, d, th = make_problem(oracle, cfg)
    rng = np.random.Generator(np.random.PCG64(9000 + seed))
    calls = []
    for _ in range(40):
        B = int(rng.choice([1, 3, 8, 31, 64, 200, 256, 257, 512, 700]))
        lpp = int(rng.choice([0, 1, 2, 4, 8, 16, 32]))
        nc = 0 if lpp == 0 else int(rng.choice([1, 2, 5, 16, 33, 40, 70]))
        calls.append((B, lpp, nc))
    thd = torch.from_numpy(th).cuda()

    def run(ctx, B, lpp, nc):
        ctx.force_plan(lpp, nc)
        try:
            out, parts = ctx.lnl_batch(thd[:B].contiguous(), want_parts=True)
        except GwError:
            return None
        torch.cuda.synchronize()
        return out.cpu().numpy(), parts.cpu().numpy()

    with make_ctx(cfg, f, d, S, dets, max_batch=700) as shared:
        got = [run(shared, *c) for c in calls]
    n_checked = 0
    for c, g in zip(calls, got):
        with make_ctx(cfg, f, d, S, dets, max_batch=700) as fresh:
            want = run(fresh, *c)
        assert (g is None) == (want is None), c
        if g is not None:
            assert np.array_equal(g[0], want[0]) and np.array_equal(g[1], want[1]), c
            n_checked += 1
    assert n_checked >= 20


def test_tidal_outputs_stay_inside_their_buffers_and_theta_is_read_with_its_stride(oracle):
    """Guard bands around the outputs of the TIDAL kernel variants, and theta [B][13] placed at the very end of its
    allocation's used range with a NaN canary after it: a read with the wrong stride or past the last row would
    poison a result.  After a reserve() growth the 13-column host staging still holds the whole batch."""
    import torch
    from paper_1904_02863_b200 import GwContext
    cfg = inputs.CONFIGS["C2"].reduced(f_max=60.0, duration_s=4.0, batch=600)
    f, S, dets, d, th = make_problem(oracle, cfg)
    lam = inputs.tidal_lambdas(cfg)
    th13 = np.ascontiguousarray(np.hstack([th, lam]))
    with GwContext(f, d, S, dets, cfg.gmst, spin_order=cfg.spin_order, max_batch=64, tidal_order=2) as ctx:
        ctx.reserve(600)
        ref_host = ctx.lnl_batch_host(th13)
        for B in (1, 5, 33, 256, 257, 600):
            tbuf = torch.full((B * 13 + GUARD,), float("nan"), dtype=torch.float64, device="cuda")
            tbuf[:B * 13] = torch.from_numpy(th13[:B].ravel()).cuda()
            thd = tbuf[:B * 13].view(B, 13)
            nl, npart, nh = B, B * cfg.n_det * 3, B * cfg.n_det * cfg.n_bins * 2
            lbuf, lnl = _guarded(torch, nl)
            pbuf, parts = _guarded(torch, npart)
            hbuf, h = _guarded(torch, nh)
            ctx.lnl_batch(thd, out=lnl, parts=parts.view(B, cfg.n_det, 3))
            ctx.waveform_batch(thd, out=torch.view_as_complex(h.view(B, cfg.n_det, cfg.n_bins, 2)))
            torch.cuda.synchronize()
            assert _intact(torch, lbuf, nl) and _intact(torch, pbuf, npart) and _intact(torch, hbuf, nh), B
            assert bool(torch.isfinite(lnl).all()) and bool(torch.isfinite(parts).all()) and bool(torch.isfinite(h).all()), B
        assert np.array_equal(ref_host, lnl.cpu().numpy())          # B = 600: host variant == device variant


def test_first_call_on_a_non_blocking_stream_right_after_create_and_reserve(oracle):
    """The workspace counters (cross-chunk tickets) are zeroed by create / reserve; a batch call issued at once on a
    NON-BLOCKING stream (not ordered against the legacy default stream) must find them zeroed: multi-chunk plans,
    one-level and two-level finish, straight after gw_ctx_create and straight after gw_ctx_reserve."""
    import torch
    from paper_1904_02863_b200 import binding
    cfg = inputs.CONFIGS["C1"].reduced(f_max=600.0, batch=700)
    f, S, dets, d, th = make_problem(oracle, cfg)
    ref = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, cfg.spin_order)
    stream = torch.cuda.Stream()                 # torch's pool streams are created with cudaStreamNonBlocking
    thd = torch.from_numpy(th).cuda()
    torch.cuda.synchronize()
    for n_chunks in (7, 40):
        for first in (300, 700):
            ctx = binding.GwContext(f, d, S, dets, cfg.gmst, spin_order=cfg.spin_order, max_batch=first)
            ctx.force_plan(1, n_chunks)
            lnl, parts = ctx.lnl_batch(thd[:first].contiguous(), want_parts=True, stream=stream)
            stream.synchronize()
            assert_lnl_close(lnl.cpu().numpy(), parts.cpu().numpy(), ref[0][:first], ref[1][:first])
            ctx.reserve(2 * first)                                              # new workspace, new counters
            lnl, parts = ctx.lnl_batch(thd[:first].contiguous(), want_parts=True, stream=stream)
            stream.synchronize()
            assert_lnl_close(lnl.cpu().numpy(), parts.cpu().numpy(), ref[0][:first], ref[1][:first])
            ctx.close()


def test_large_fixed_delay_is_poisoned_not_garbled(oracle):
    """A FIXED detector with a huge dt_s pushes f (t_c + dt) beyond the domain of the integer range reduction: the
    outputs are NaN (boundary contract), while a moderate delay still matches the oracle."""
    import torch
    from paper_1904_02863_b200 import GwContext
    f = 20.0 + np.arange(640) / 4.0
    S = inputs.analytic_psd(f)[None].repeat(2, axis=0)
    th = np.tile(np.array(inputs.CONFIGS["C0"].theta_inj), (4, 1))
    th[:, inputs.P_TC] = [0.0, 0.05, -0.03, 0.01]
    rng = np.random.Generator(np.random.PCG64(11))
    d = (rng.standard_normal((2, f.size)) + 1j * rng.standard_normal((2, f.size))) * np.sqrt(S / (4 * 0.25))
    for dt0, dt1, finite in ((0.3, -0.2, True), (4.0e6, 0.0, False), (0.0, 4.0e6, False)):
        dets = np.stack([inputs.fixed_detector(1.0, 0.0, dt0), inputs.fixed_detector(0.3, -0.6, dt1)])
        with GwContext(f, d, S, dets, 0.0, spin_order=0, max_batch=4) as ctx:
            thd = torch.from_numpy(th).cuda()
            lnl, parts = ctx.lnl_batch(thd, want_parts=True)
            h = ctx.waveform_batch(thd)
            torch.cuda.synchronize()
            lnl, parts, h = lnl.cpu().numpy(), parts.cpu().numpy(), h.cpu().numpy()
        if finite:
            ref = oracle.lnl(f, 0.25, d, S, dets, 0.0, th, 0)
            assert_lnl_close(lnl, parts, ref[0], ref[1])
            assert_h_close(h, oracle.waveform(f, dets, 0.0, th, 0))
        else:
            assert np.all(np.isnan(lnl)) and np.all(np.isnan(h))
