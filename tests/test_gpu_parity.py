"""`-m gpu`: the CUDA path (through the C-ABI of include/gwlnl.h) against the CPU oracle, element by element,
on the same seeded inputs (SURVEY.md section 9 gates 2-4; tolerances from BASELINE.json north_star)."""
import os

import numpy as np
import pytest

from paper_1904_02863_b200 import inputs

from gpu_common import assert_h_close, assert_lnl_close, make_ctx, make_problem

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    return torch


def _dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


# reduced shapes: several stages (128 bins) and chunks, ragged tails in bins and in proposals
SMALL = [
    ("C0", dict(f_max=512.0, batch=256)),          # config 0 at full size: 3937 bins, 256 proposals, 1 fixed det
    ("C1", dict(f_max=181.75, batch=300)),         # 648 bins (5 stages + 8), 300 proposals (2 tiles, ragged)
    ("C2", dict(f_max=24.5, batch=70)),            # BNS: 577 bins at df = 1/128, phases ~1e4 rad
    ("C3", dict(f_max=11.25, batch=40)),           # 10 Hz start, df = 1/512: 641 bins, phases ~4.5e4 rad
    ("C4", dict(f_max=2048.0, batch=48)),          # config-1 shape at full band (8113 bins)
]


@pytest.mark.parametrize("name,red", SMALL, ids=[s[0] for s in SMALL])
def test_waveform_elementwise(oracle, torch_cuda, name, red):
    torch = torch_cuda
    cfg = inputs.CONFIGS[name].reduced(**red)
    f, S, dets, d, th = make_problem(oracle, cfg)
    nb = min(cfg.batch, 64)
    with make_ctx(cfg, f, d, S, dets) as ctx:
        h = ctx.waveform_batch(_dev(torch, th[:nb]))
        torch.cuda.synchronize()
        h_gpu = h.cpu().numpy()
    h_ref = oracle.waveform(f, dets, cfg.gmst, th[:nb], cfg.spin_order)
    assert h_gpu.shape == h_ref.shape
    assert_h_close(h_gpu, h_ref)


@pytest.mark.parametrize("name,red", SMALL, ids=[s[0] for s in SMALL])
def test_lnl_every_proposal(oracle, torch_cuda, name, red):
    torch = torch_cuda
    cfg = inputs.CONFIGS[name].reduced(**red)
    f, S, dets, d, th = make_problem(oracle, cfg)
    with make_ctx(cfg, f, d, S, dets) as ctx:
        lnl, parts = ctx.lnl_batch(_dev(torch, th), want_parts=True)
        torch.cuda.synchronize()
        lnl, parts = lnl.cpu().numpy(), parts.cpu().numpy()
    lnl_ref, parts_ref, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, cfg.spin_order)
    assert_lnl_close(lnl, parts, lnl_ref, parts_ref)
    # row 0 is the injection: coherent, Re<d|h> = <h|h> + N(0, <h|h>)
    hh0 = parts[0, :, 2].sum()
    assert abs(parts[0, :, 0].sum() - hh0) < 5.0 * np.sqrt(hh0)


@pytest.mark.parametrize("batch", [1, 2, 3, 7, 8, 9, 16, 31, 33, 64, 100, 255, 257, 600])
def test_lnl_all_lane_layouts(oracle, torch_cuda, batch):
    """Every lanes-per-proposal layout of the fused kernel (1..32 lanes, ragged tiles) gives the oracle's lnL."""
    torch = torch_cuda
    cfg = inputs.CONFIGS["C1"].reduced(f_max=301.25, batch=600)        # 1126 bins
    f, S, dets, d, th = make_problem(oracle, cfg)
    with make_ctx(cfg, f, d, S, dets) as ctx:
        plan = ctx.plan(batch)
        lnl, parts = ctx.lnl_batch(_dev(torch, th[:batch]), want_parts=True)
        torch.cuda.synchronize()
        lnl, parts = lnl.cpu().numpy(), parts.cpu().numpy()
    lnl_ref, parts_ref, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th[:batch], cfg.spin_order)
    assert_lnl_close(lnl, parts, lnl_ref, parts_ref)
    assert plan["lanes_per_prop"] * plan["props_per_cta"] == 256


@pytest.mark.parametrize("lpp", [1, 2, 4, 8, 16, 32])
@pytest.mark.parametrize("n_chunks", [1, 3, 40])
def test_every_lane_width_and_chunking_forced(oracle, torch_cuda, lpp, n_chunks):
    """gw_ctx_force_plan pins the launch shape, so every lanes-per-proposal layout is exercised with one chunk (direct
    finish), a few chunks (single-level finish) and 40 chunks (two-level finish), whatever the planner would choose."""
    torch = torch_cuda
    cfg = inputs.CONFIGS["C1"].reduced(f_max=301.25, batch=100)        # 1126 bins
    f, S, dets, d, th = make_problem(oracle, cfg)
    with make_ctx(cfg, f, d, S, dets) as ctx:
        ctx.force_plan(lpp, n_chunks)
        plan = ctx.plan(100)
        assert plan["lanes_per_prop"] == lpp and plan["n_chunks"] == n_chunks
        lnl, parts = ctx.lnl_batch(_dev(torch, th), want_parts=True)
        again = ctx.lnl_batch(_dev(torch, th))
        torch.cuda.synchronize()
        assert torch.equal(lnl, again)
        lnl, parts = lnl.cpu().numpy(), parts.cpu().numpy()
        ctx.force_plan(0, 0)
        assert ctx.plan(100)["lanes_per_prop"] * ctx.plan(100)["props_per_cta"] == 256
    lnl_ref, parts_ref, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, cfg.spin_order)
    assert_lnl_close(lnl, parts, lnl_ref, parts_ref)


@pytest.mark.parametrize("n_det", [1, 2, 4, 5, 6, 7, 8])
def test_detector_counts(oracle, torch_cuda, n_det):
    """1 ... GW_MAX_DET = 8 detectors (mixed GEOMETRIC / FIXED with non-zero fixed delays of both signs): lnL, parts
    and the waveform against the oracle; counts above 4 run the one-CTA-per-SM kernel variants."""
    torch = torch_cuda
    base = inputs.CONFIGS["C1"].reduced(f_max=150.0, batch=40)
    rows = [inputs.geometric_detector("H1"), inputs.fixed_detector(0.6, -0.3, 0.0123),
            inputs.geometric_detector("V1"), inputs.geometric_detector("L1"),
            inputs.fixed_detector(-0.2, 0.7, -0.0071), inputs.geometric_detector("H1"),
            inputs.fixed_detector(0.35, 0.35, 0.0), inputs.geometric_detector("V1")][:n_det]
    dets = np.stack(rows)
    f = inputs.frequency_grid(base)
    S = np.tile(inputs.analytic_psd(f), (n_det, 1))
    th = inputs.proposals(base)
    rng = np.random.Generator(np.random.PCG64(777 + n_det))
    z = rng.standard_normal((n_det, f.size, 2))
    sig = oracle.waveform(f, dets, base.gmst, th[:1])[0]
    d = sig + (z[..., 0] + 1j * z[..., 1]) * np.sqrt(S / (4 * base.delta_f))
    from paper_1904_02863_b200 import GwContext
    with GwContext(f, d, S, dets, base.gmst, max_batch=64) as ctx:
        thd = _dev(torch, th)
        lnl, parts = ctx.lnl_batch(thd, want_parts=True)
        h = ctx.waveform_batch(thd)
        torch.cuda.synchronize()
        lnl, parts, h = lnl.cpu().numpy(), parts.cpu().numpy(), h.cpu().numpy()
    lnl_ref, parts_ref, _ = oracle.lnl(f, base.delta_f, d, S, dets, base.gmst, th)
    assert_lnl_close(lnl, parts, lnl_ref, parts_ref)
    assert_h_close(h, oracle.waveform(f, dets, base.gmst, th))


def test_precompute_norms(oracle, torch_cuda):
    """Kernel K0: I7_I = sum (4 df/S) f^(-7/3) against the oracle's compensated sum; <h|h> = |C|^2 A0^2 I7 (pin P2)."""
    for name, red in SMALL:
        cfg = inputs.CONFIGS[name].reduced(**red)
        f, S, dets = inputs.frequency_grid(cfg), inputs.psd(cfg), inputs.detectors(cfg)
        with make_ctx(cfg, f, np.zeros_like(S, dtype=complex), S, dets) as ctx:
            i7 = ctx.norms()
        ref = oracle.norm_i7(f, cfg.delta_f, S[0])
        np.testing.assert_allclose(i7, ref, rtol=1e-13)


def test_no_spin_option(oracle, torch_cuda):
    """spin_order = 0 ignores chi1, chi2 (config C0 is non-spinning)."""
    torch = torch_cuda
    cfg = inputs.CONFIGS["C1"].reduced(f_max=120.0, batch=33)
    f, S, dets, d, th = make_problem(oracle, cfg)
    from paper_1904_02863_b200 import GwContext
    with GwContext(f, d, S, dets, cfg.gmst, spin_order=0, max_batch=64) as ctx:
        lnl, parts = ctx.lnl_batch(_dev(torch, th), want_parts=True)
        torch.cuda.synchronize()
    lnl_ref, parts_ref, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, spin_order=0)
    assert_lnl_close(lnl.cpu().numpy(), parts.cpu().numpy(), lnl_ref, parts_ref)


def test_bitwise_determinism_and_prefix_stability(oracle, torch_cuda):
    """Gate 4: >= 10 repeats give identical bits; a proposal's lnL does not depend on what else shares the
    batch as long as the launch shape (plan) is unchanged."""
    torch = torch_cuda
    cfg = inputs.CONFIGS["C1"].reduced(f_max=420.0, batch=700)
    f, S, dets, d, th = make_problem(oracle, cfg)
    with make_ctx(cfg, f, d, S, dets) as ctx:
        thd = _dev(torch, th)
        first, first_parts = ctx.lnl_batch(thd, want_parts=True)
        first, first_parts = first.clone(), first_parts.clone()
        for _ in range(10):
            again, again_parts = ctx.lnl_batch(thd, want_parts=True)
            torch.cuda.synchronize()
            assert torch.equal(again, first) and torch.equal(again_parts, first_parts)
        # same plan (tile count and chunking) for 700 and 690 proposals => identical bits for the shared prefix
        if ctx.plan(700) == ctx.plan(690):
            sub = ctx.lnl_batch(thd[:690].contiguous())
            torch.cuda.synchronize()
            assert torch.equal(sub, first[:690])
        # waveform: pure function of (theta_b, bin)
        h1 = ctx.waveform_batch(thd[:50].contiguous()).clone()
        h2 = ctx.waveform_batch(thd[10:60].contiguous())
        torch.cuda.synchronize()
        assert torch.equal(h1[10:], h2[:40])


def test_host_variants_match_device_variants(oracle, torch_cuda):
    torch = torch_cuda
    cfg = inputs.CONFIGS["C1"].reduced(f_max=200.0, batch=130)
    f, S, dets, d, th = make_problem(oracle, cfg)
    with make_ctx(cfg, f, d, S, dets) as ctx:
        lnl_d, parts_d = ctx.lnl_batch(_dev(torch, th), want_parts=True)
        h_d = ctx.waveform_batch(_dev(torch, th))
        torch.cuda.synchronize()
        lnl_h, parts_h = ctx.lnl_batch_host(th, want_parts=True)
        h_h = ctx.waveform_batch_host(th)
        lnl_only = ctx.lnl_batch_host(th)
    assert np.array_equal(lnl_h, lnl_d.cpu().numpy()) and np.array_equal(parts_h, parts_d.cpu().numpy())
    assert np.array_equal(h_h, h_d.cpu().numpy()) and np.array_equal(lnl_only, lnl_h)


@pytest.mark.parametrize("batch", [1, 130, 1500, 2600])
def test_host_variant_with_pinned_output(oracle, torch_cuda, batch):
    """A pinned lnL buffer is written by the kernel itself (include/gwlnl.h, host variants): same bits as the staged
    copy into a pageable buffer, nothing outside the n_prop entries is touched, and a sub-array offset works.
    From 2048 proposals a pinned theta buffer is read in place by the setup kernel (batch 2600: a ragged last CTA)."""
    torch = torch_cuda
    cfg = inputs.CONFIGS["C1"].reduced(f_max=200.0, batch=2600)
    f, S, dets, d, th = make_problem(oracle, cfg)
    th = th[:batch]
    with make_ctx(cfg, f, d, S, dets) as ctx:
        staged = ctx.lnl_batch_host(th)                                   # pageable numpy output
        pinned = torch.full((batch + 16,), -7.0, dtype=torch.float64).pin_memory()
        view = pinned.numpy()[8:8 + batch]
        th_pin = torch.from_numpy(th.copy()).pin_memory()
        got, parts = ctx.lnl_batch_host(th_pin.numpy(), out=view, want_parts=True)
        again = ctx.lnl_batch_host(th_pin.numpy(), out=view)
    assert np.array_equal(view, staged) and np.array_equal(again, staged)
    assert np.all(pinned.numpy()[:8] == -7.0) and np.all(pinned.numpy()[8 + batch:] == -7.0)
    assert np.isfinite(parts).all()


def test_device_resident_context_inputs(oracle, torch_cuda):
    """gw_ctx_create accepts device pointers for freqs / data / psd."""
    torch = torch_cuda
    cfg = inputs.CONFIGS["C1"].reduced(f_max=100.0, batch=20)
    f, S, dets, d, th = make_problem(oracle, cfg)
    from paper_1904_02863_b200 import GwContext
    with GwContext(f, d, S, dets, cfg.gmst, max_batch=32) as a, \
            GwContext(_dev(torch, f), _dev(torch, d), _dev(torch, S), dets, cfg.gmst, max_batch=32) as b:
        la = a.lnl_batch(_dev(torch, th))
        lb = b.lnl_batch(_dev(torch, th))
        torch.cuda.synchronize()
        assert torch.equal(la, lb)


def test_identities_on_gpu(oracle, torch_cuda):
    """Pin P3 through the CUDA path: d = 0 => lnL = -1/2 <h|h>; noiseless data at the truth => +1/2 <h|h>, Im<d|h> = 0."""
    torch = torch_cuda
    cfg = inputs.CONFIGS["C1"].reduced(f_max=256.0, batch=64)
    f, S, dets = inputs.frequency_grid(cfg), inputs.psd(cfg), inputs.detectors(cfg)
    th = inputs.proposals(cfg)
    with make_ctx(cfg, f, np.zeros_like(S, dtype=complex), S, dets) as ctx:
        lnl, parts = ctx.lnl_batch(_dev(torch, th), want_parts=True)
        torch.cuda.synchronize()
        lnl, parts = lnl.cpu().numpy(), parts.cpu().numpy()
        assert np.all(parts[..., :2] == 0)
        np.testing.assert_allclose(lnl, -0.5 * parts[..., 2].sum(axis=1), rtol=1e-14)
        sig = ctx.waveform_batch(_dev(torch, th[:1]))[0].cpu().numpy()      # the library's own h as data
    with make_ctx(cfg, f, sig, S, dets) as ctx:
        lnl, parts = ctx.lnl_batch(_dev(torch, th), want_parts=True)
        torch.cuda.synchronize()
        lnl, parts = lnl.cpu().numpy(), parts.cpu().numpy()
    hh = parts[0, :, 2].sum()
    assert lnl[0] == pytest.approx(0.5 * hh, rel=1e-10)
    assert np.abs(parts[0, :, 1]).max() < 1e-9 * hh
    assert np.all(lnl[1:] < 0.5 * hh)                                       # Cauchy-Schwarz


def test_edge_cases_and_errors(oracle, torch_cuda):
    torch = torch_cuda
    from paper_1904_02863_b200 import GwContext, GwError
    from paper_1904_02863_b200 import binding
    cfg = inputs.CONFIGS["C1"].reduced(f_max=60.0, batch=16)
    f, S, dets, d, th = make_problem(oracle, cfg)
    with GwContext(f, d, S, dets, cfg.gmst, max_batch=16) as ctx:
        # n_prop == 0: OK, writes nothing
        empty = torch.empty((0, 11), dtype=torch.float64, device="cuda")
        out = ctx.lnl_batch(empty)
        assert out.numel() == 0
        assert ctx.waveform_batch(empty).shape == (0, 3, f.size)
        # more than reserved: INVALID_ARG, then reserve and retry
        big = _dev(torch, np.tile(th, (2, 1)))
        with pytest.raises(GwError) as ei:
            ctx.lnl_batch(big)
        assert ei.value.code == binding.GW_ERR_INVALID_ARG
        ctx.reserve(32)
        assert ctx.info()["max_batch"] == 32
        both = ctx.lnl_batch(big)
        torch.cuda.synchronize()
        assert torch.equal(both[:16], both[16:])
        # out-of-domain rows give NaN there and nowhere else
        bad = th.copy()
        bad[3, inputs.P_MC] = -1.0
        bad[5, inputs.P_Q] = 1.5
        bad[7, inputs.P_DL] = 0.0
        bad[9, inputs.P_COSI] = 1.2
        bad[11, inputs.P_TC] = np.nan
        lnl, parts = ctx.lnl_batch(_dev(torch, bad), want_parts=True)
        h = ctx.waveform_batch(_dev(torch, bad))
        good = ctx.lnl_batch(_dev(torch, th))
        torch.cuda.synchronize()
        lnl, h, good = lnl.cpu().numpy(), h.cpu().numpy(), good.cpu().numpy()
        rows = [3, 5, 7, 9, 11]
        assert np.all(np.isnan(lnl[rows])) and np.all(np.isnan(h[rows]))
        keep = np.setdiff1d(np.arange(16), rows)
        assert np.array_equal(lnl[keep], good[keep]) and np.all(np.isfinite(h[keep]))
    # smallest grid: 2 bins
    f2, S2 = f[:2], S[:, :2]
    with GwContext(f2, d[:, :2], S2, dets, cfg.gmst, max_batch=16) as ctx:
        lnl = ctx.lnl_batch_host(th)
    ref, _, _ = oracle.lnl(f2, cfg.delta_f, d[:, :2], S2, dets, cfg.gmst, th)
    np.testing.assert_allclose(lnl, ref, rtol=1e-9, atol=1e-12)
    # create-time validation
    fbad = f.copy(); fbad[5] += 1e-3
    for args in [(fbad, d, S), (f, d, -S), (f[::-1].copy(), d, S)]:
        with pytest.raises(GwError) as ei:
            GwContext(args[0], args[1], args[2], dets, cfg.gmst)
        assert ei.value.code == binding.GW_ERR_INVALID_ARG
    skew = dets.copy(); skew[0, 4:7] *= 1.01
    with pytest.raises(GwError):
        GwContext(f, d, S, skew, cfg.gmst)
    with pytest.raises(GwError):
        GwContext(f, d[:2], S[:2], np.tile(dets[:1], (9, 1)), cfg.gmst)      # 9 detectors > GW_MAX_DET


def test_time_shift_interchange(oracle, torch_cuda):
    """Pin P4 on the GPU: a FIXED detector with dt = tau is the same as t_c + tau (PAPER.md:69 factor)."""
    torch = torch_cuda
    cfg = inputs.CONFIGS["C0"].reduced(f_max=128.0, batch=32)
    f, S = inputs.frequency_grid(cfg), inputs.psd(cfg)
    th = inputs.proposals(cfg)
    tau = 0.0123
    from paper_1904_02863_b200 import GwContext
    zero = np.zeros_like(S, dtype=complex)
    with GwContext(f, zero, S, inputs.fixed_detector(1.0, 0.0, tau)[None], 0.0, spin_order=0, max_batch=32) as a, \
            GwContext(f, zero, S, inputs.fixed_detector(1.0, 0.0, 0.0)[None], 0.0, spin_order=0, max_batch=32) as b:
        th2 = th.copy(); th2[:, inputs.P_TC] += tau
        ha = a.waveform_batch_host(th)
        hb = b.waveform_batch_host(th2)
    scale = np.abs(hb).max(axis=-1, keepdims=True)
    assert (np.abs(ha - hb) / scale).max() < 1e-11
    np.testing.assert_allclose(np.abs(ha), np.abs(hb), rtol=1e-12)


def _random_shape_case(oracle, torch_cuda, seed, det_lo, det_hi):
    torch = torch_cuda
    from paper_1904_02863_b200 import GwContext, GwError
    rng = np.random.Generator(np.random.PCG64(4242 + seed))
    n_det = int(rng.integers(det_lo, det_hi + 1))
    M = int(rng.choice([2, 3, 5, 31, 33, 127, 129, 257, 640, 1000, 2500]))
    B = int(rng.choice([1, 2, 5, 8, 17, 32, 100, 255, 256, 300, 700]))
    df = float(rng.choice([1 / 128, 1 / 16, 0.125, 0.25, 1.0]))
    f0 = float(rng.choice([10.0, 20.0, 35.5]))
    f = f0 + np.arange(M) * df
    bns = bool(rng.integers(0, 2))
    isco, marg, spin = int(rng.integers(0, 2)), int(rng.integers(0, 2)), int(rng.integers(0, 2))
    rng3 = np.random.Generator(np.random.PCG64(999 + seed))          # one case in three each: tidal order 0, 1, 2
    tidal = int(rng3.integers(0, 3))
    if spin and rng3.random() < 0.5:                                 # half of the spinning cases: spin_order 2
        spin = 2
    names = ["H1", "L1", "V1"]
    rows = []
    for i in range(n_det):
        if rng.random() < 0.3:
            rows.append(inputs.fixed_detector(float(rng.uniform(-1, 1)), float(rng.uniform(-1, 1)), float(rng.uniform(-0.03, 0.03))))
        else:
            rows.append(inputs.geometric_detector(names[int(rng.integers(0, 3))]))
    dets = np.stack(rows)
    S = np.stack([inputs.analytic_psd(f) * float(rng.uniform(0.5, 2.0)) for _ in range(n_det)])
    th = np.empty((B, 11))
    th[:, inputs.P_MC] = rng.uniform(1.0, 2.0, B) if bns else rng.uniform(5.0, 60.0, B)
    th[:, inputs.P_Q] = rng.uniform(0.2, 1.0, B)
    th[:, inputs.P_CHI1] = rng.uniform(-0.9, 0.9, B)
    th[:, inputs.P_CHI2] = rng.uniform(-0.9, 0.9, B)
    th[:, inputs.P_DL] = rng.uniform(50, 3000, B)
    th[:, inputs.P_TC] = rng.uniform(-0.5, 0.5, B)
    th[:, inputs.P_PHIC] = rng.uniform(-7, 7, B)
    th[:, inputs.P_COSI] = rng.uniform(-1, 1, B)
    th[:, inputs.P_RA] = rng.uniform(0, 2 * np.pi, B)
    th[:, inputs.P_DEC] = np.arcsin(rng.uniform(-1, 1, B))
    th[:, inputs.P_PSI] = rng.uniform(0, np.pi, B)
    gmst = float(rng.uniform(0, 2 * np.pi))
    z = rng.standard_normal((n_det, M, 2))
    d = oracle.waveform(f, dets, gmst, th[:1], spin)[0] + (z[..., 0] + 1j * z[..., 1]) * np.sqrt(S / (4 * df))
    rng2 = np.random.Generator(np.random.PCG64(777 + seed))          # every other case: a pinned launch shape
    lam = rng3.uniform(0, 5000, (B, 2))
    tkw = dict(lambdas=lam, tidal_order=tidal) if tidal else {}
    with GwContext(f, d, S, dets, gmst, spin_order=spin, max_batch=B, isco_cut=isco, phase_marginal=marg,
                   tidal_order=tidal) as ctx:
        thd = _dev(torch, np.hstack([th, lam]) if tidal else th)
        if rng2.random() < 0.5:
            lpp = int(rng2.choice([1, 2, 4, 8, 16, 32]))
            ctx.force_plan(lpp, int(rng2.integers(1, max(2, min(80, M // lpp + 1)))))
            try:
                lnl, parts = ctx.lnl_batch(thd, want_parts=True)
            except GwError:                                          # shape does not fit the reserved workspace
                ctx.force_plan(0, 0)
                lnl, parts = ctx.lnl_batch(thd, want_parts=True)
        else:
            lnl, parts = ctx.lnl_batch(thd, want_parts=True)
        h = ctx.waveform_batch(thd[: min(B, 16)].contiguous())
        torch.cuda.synchronize()
        lnl, parts, h = lnl.cpu().numpy(), parts.cpu().numpy(), h.cpu().numpy()
    lnl_ref, parts_ref, _ = oracle.lnl(f, df, d, S, dets, gmst, th, spin, isco_cut=isco, **tkw)
    if marg:
        lnl_ref = oracle.lnl_phase_marginal(parts_ref)
    hh = parts_ref[..., 2].sum(axis=1)
    keep = hh > 0                                     # isco_cut below the band: h = 0, lnL = 0 exactly
    assert np.all(lnl[~keep] == 0) and np.all(parts[~keep] == 0)
    if keep.any():
        # Gate A16 plus the conditioning term of DESIGN.md section 8: the fp64 phase of either side is defined to
        # ~1e-11 rad (a few ulp of its largest term), and a phase offset dphi moves Re<d|h> by |<d|h>| dphi, which
        # the A16 scale does not cover when the signal is buried (<h|h> << |Im<d|h>|; soak seed 444: 3 bins,
        # <h|h> = 4e-7, |<d|h>| = 6e-4).  dphi = 1e-10 rad.
        scale = np.abs(parts_ref[keep][..., 0].sum(axis=1)) + hh[keep]
        modulus = np.hypot(parts_ref[keep][..., 0].sum(axis=1), parts_ref[keep][..., 1].sum(axis=1))
        assert np.all(np.abs(lnl[keep] - lnl_ref[keep]) <= 1e-8 * scale + 1e-10 * modulus)
        pscale = (np.hypot(parts_ref[keep][..., 0], parts_ref[keep][..., 1]) + parts_ref[keep][..., 2])[..., None]
        ok = pscale[..., 0] > 0
        assert (np.abs(parts[keep] - parts_ref[keep])[ok] / pscale[ok]).max() <= 1e-8
    if tidal:
        tkw["lambdas"] = lam[: min(B, 16)]
    h_ref = oracle.waveform(f, dets, gmst, th[: min(B, 16)], spin, isco_cut=isco, **tkw)
    hs = np.abs(h_ref).max(axis=-1, keepdims=True)
    nz = hs[..., 0] > 0
    assert np.all(h[~nz] == 0)
    if nz.any():
        assert (np.abs(h - h_ref)[nz] / hs[nz]).max() <= 1e-9


@pytest.mark.parametrize("seed", range(int(os.environ.get("GW_RANDOM_SHAPES", "24"))))   # soak: GW_RANDOM_SHAPES=500
def test_random_shapes(oracle, torch_cuda, seed):
    """Seeded random shapes: bins 2..2500, proposals 1..700, 1..4 detectors (geometric and fixed mixed), random band,
    resolution, mass range and options (incl. the tidal orders) -- ragged tails everywhere the launch planner can put one."""
    _random_shape_case(oracle, torch_cuda, seed, 1, 4)


@pytest.mark.parametrize("seed", range(100, 100 + int(os.environ.get("GW_RANDOM_SHAPES_MANY_DET", "8"))))
def test_random_shapes_five_to_eight_detectors(oracle, torch_cuda, seed):
    """The same seeded random shapes with 5..8 detectors (the one-CTA-per-SM kernel variants)."""
    _random_shape_case(oracle, torch_cuda, seed, 5, 8)



def test_cuda_phase_against_40_digit_arithmetic(torch_cuda):
    """Pin P7 applied to the CUDA path itself (no oracle involved): arg h of a FIXED (F+ = 1, Fx = 0, dt = 0) detector
    against the 40-digit TaylorF2 phase of tests/test_oracle_phase.py, to the same ulp-relative bound as the oracle."""
    torch = torch_cuda
    import mpmath as mp
    from test_oracle_phase import _mp_phase
    from paper_1904_02863_b200 import GwContext
    mp.mp.dps = 40
    rng = np.random.default_rng(11)
    f = np.array([10.0, 10.0 + 1 / 512, 13.7, 20.0, 33.25, 64.0, 150.5, 512.0, 1024.0, 2047.5])
    f = 10.0 + np.round((f - 10.0) * 512) / 512                       # on a uniform 1/512 Hz grid
    grid = 10.0 + np.arange(int(round((f.max() - 10.0) * 512)) + 1) / 512
    idx = np.round((f - 10.0) * 512).astype(int)
    th = np.zeros((24, 11))
    for b in range(24):
        bns = b % 2 == 0
        th[b] = [rng.uniform(1.1, 1.3) if bns else rng.uniform(20, 40), rng.uniform(0.5, 1), rng.uniform(-0.8, 0.8),
                 rng.uniform(-0.8, 0.8), 100.0, rng.uniform(-0.1, 0.1), rng.uniform(0, 2 * np.pi), 1.0, 0, 0, 0]
    S = np.ones((1, grid.size))
    d = np.zeros((1, grid.size), complex)
    with GwContext(grid, d, S, inputs.fixed_detector(1.0, 0.0, 0.0)[None], 0.0, max_batch=24) as ctx:
        h = ctx.waveform_batch(_dev(torch, th))[:, 0, :][:, _dev(torch, idx)].cpu().numpy()
    worst = 0.0
    for b in range(24):
        for k, fk in enumerate(grid[idx]):
            want = _mp_phase(fk, th[b], 1, None)
            got = np.angle(h[b, k])                                    # arg h = -Psi (mod 2 pi)
            err = float(abs(mp.mpf(got) + want - 2 * mp.pi * mp.nint((mp.mpf(got) + want) / (2 * mp.pi))))
            bound = 16 * np.spacing(float(abs(want))) + 1e-13
            worst = max(worst, err / bound)
            assert err < bound, (b, fk, err, bound)
    assert worst > 0


def test_phase_domain_guard(oracle, torch_cuda):
    """A proposal whose phase would leave the domain of the integer range reduction (|phase| >= 2^31 quarter turns)
    gives NaN, not garbage; one well inside the domain (Mc = 0.05 Msun, 3.6e6 turns at 10 Hz) still matches the oracle."""
    torch = torch_cuda
    from paper_1904_02863_b200 import GwContext
    f = 10.0 + np.arange(400) / 16.0
    S = inputs.analytic_psd(f)[None]
    dets = inputs.fixed_detector(1.0, 0.0, 0.0)[None]
    th = np.tile(np.array(inputs.CONFIGS["C0"].theta_inj), (3, 1))
    th[0, inputs.P_MC] = 0.05
    th[1, inputs.P_MC] = 1.0e-4          # ~1e11 turns at 10 Hz: out of domain
    rng = np.random.Generator(np.random.PCG64(5))
    d = (rng.standard_normal((1, f.size)) + 1j * rng.standard_normal((1, f.size))) * np.sqrt(S / (4 / 16.0))
    with GwContext(f, d, S, dets, 0.0, spin_order=0, max_batch=3) as ctx:
        lnl, parts = ctx.lnl_batch(_dev(torch, th), want_parts=True)
        h = ctx.waveform_batch(_dev(torch, th))
        torch.cuda.synchronize()
        lnl, parts, h = lnl.cpu().numpy(), parts.cpu().numpy(), h.cpu().numpy()
    assert np.isnan(lnl[1]) and np.all(np.isnan(h[1])) and np.all(np.isfinite(lnl[[0, 2]]))
    ref = oracle.lnl(f, 1 / 16.0, d, S, dets, 0.0, th[[0, 2]], 0)
    assert_lnl_close(lnl[[0, 2]], parts[[0, 2]], ref[0], ref[1])


@pytest.mark.parametrize("n_det", [1, 3, 4, 6, 8])
@pytest.mark.parametrize("lpp,n_chunks,batch", [(32, 16, 1), (32, 9, 20), (32, 2, 300), (16, 16, 40), (8, 5, 70), (4, 7, 130),
                                               (2, 3, 200), (32, 17, 5)])
def test_cluster_finish_matches_ticket_finish_bit_for_bit(oracle, torch_cuda, n_det, lpp, n_chunks, batch):
    """Small multi-lane grids reduce the chunk sums of a tile through a thread-block cluster and distributed shared
    memory (gw_ctx_cluster_finish, default on); the ticket path through global partial sums adds the same numbers in
    the same order.  Both against the oracle, and against each other bit for bit; 17 chunks exceed the cluster size
    and fall back to the ticket path by themselves."""
    torch = torch_cuda
    from paper_1904_02863_b200 import GwContext
    cfg = inputs.CONFIGS["C1"].reduced(f_max=420.0, batch=300)
    f, S, dets_all, d_all, th = make_problem(oracle, cfg)
    if n_det >= 4:
        extra = n_det - 3
        dets = np.concatenate([dets_all] + [inputs.fixed_detector(0.4 - 0.1 * k, -0.3 + 0.1 * k, 0.002 * (k + 1))[None]
                                            for k in range(extra)])
        d = np.concatenate([d_all] + [d_all[k % 3:k % 3 + 1] * (0.7 + 0.05 * k) for k in range(extra)])
        S4 = np.concatenate([S] + [S[k % 3:k % 3 + 1] for k in range(extra)])
    else:
        dets, d, S4 = dets_all[:n_det], d_all[:n_det], S[:n_det]
    thd = _dev(torch, th[:batch])
    with GwContext(f, d, S4, dets, cfg.gmst, spin_order=cfg.spin_order, max_batch=batch) as ctx:
        ctx.force_plan(lpp, n_chunks)
        a_lnl, a_parts = ctx.lnl_batch(thd, want_parts=True)
        a2, _ = ctx.lnl_batch(thd, want_parts=True)
        ctx.cluster_finish(False)
        b_lnl, b_parts = ctx.lnl_batch(thd, want_parts=True)
        torch.cuda.synchronize()
    assert torch.equal(a_lnl, b_lnl) and torch.equal(a_parts, b_parts) and torch.equal(a_lnl, a2)
    ref = oracle.lnl(f, cfg.delta_f, d, S4, dets, cfg.gmst, th[:batch], cfg.spin_order)
    assert_lnl_close(a_lnl.cpu().numpy(), a_parts.cpu().numpy(), ref[0], ref[1])


@pytest.mark.parametrize("batch", [1, 16, 300, 512, 513])
def test_host_variant_graph_path_matches_launch_by_launch(oracle, torch_cuda, batch):
    """gw_lnl_batch_host sends batches of up to 512 proposals through a library-owned CUDA graph (pinned staging in and
    out, one launch per call): same bits as the launch-by-launch path and as the device variant, fresh theta on every
    replay, with and without parts, pageable and pinned caller buffers; 513 proposals take the other path by themselves."""
    torch = torch_cuda
    cfg = inputs.CONFIGS["C1"].reduced(f_max=260.0, batch=513)
    f, S, dets, d, th = make_problem(oracle, cfg)
    th = th[:batch]
    with make_ctx(cfg, f, d, S, dets, max_batch=batch) as ctx:
        dev_lnl, dev_parts = ctx.lnl_batch(_dev(torch, th), want_parts=True)
        torch.cuda.synchronize()
        n0 = ctx.launch_count()
        g_lnl, g_parts = ctx.lnl_batch_host(th, want_parts=True)
        g_only = ctx.lnl_batch_host(th)
        assert ctx.launch_count() == n0 + 4
        th2 = th[::-1].copy()                                   # a replay of the cached graph must read the new theta
        g_rev = ctx.lnl_batch_host(th2)
        pin_in = torch.from_numpy(th).pin_memory().numpy()
        pin_out = torch.empty(batch, dtype=torch.float64).pin_memory().numpy()
        ctx.lnl_batch_host(pin_in, out=pin_out)
        ctx.host_graph(False)
        p_lnl, p_parts = ctx.lnl_batch_host(th, want_parts=True)
        p_rev = ctx.lnl_batch_host(th2)
    assert np.array_equal(g_lnl, dev_lnl.cpu().numpy()) and np.array_equal(g_parts, dev_parts.cpu().numpy())
    assert np.array_equal(g_lnl, p_lnl) and np.array_equal(g_parts, p_parts) and np.array_equal(g_only, g_lnl)
    assert np.array_equal(g_rev, g_lnl[::-1]) and np.array_equal(p_rev, g_rev) and np.array_equal(pin_out, g_lnl)


@pytest.mark.parametrize("lpp,n_ctas,vbins", [(1, 7, 0), (1, 7, 30), (1, 12, 30), (1, 10, 40), (4, 12, 10), (4, 6, 30),
                                              (32, 4, 30), (32, 5, 20), (32, 61, 3), (2, 4, 30), (2, 148, 30)])
@pytest.mark.parametrize("option", ["plain", "isco_cut", "tidal"])
def test_balanced_grids_with_boundary_bins(oracle, torch_cuda, lpp, n_ctas, vbins, option):
    """Pinned balanced grids (gw_ctx_force_grid: n_ctas CTAs share the flattened (tile, bin) space) with boundary bins
    between the tiles (gw_ctx_boundary_bins), for one-lane and multi-lane layouts and the kernel variants: against the
    oracle, run-to-run identical bits, and -- where the range arithmetic says so -- with CTAs whose range only touches a
    tile's boundary positions (segments of no bins, which must contribute exact zeros)."""
    torch = torch_cuda
    from paper_1904_02863_b200 import GwContext, binding
    cfg = inputs.CONFIGS["C1"].reduced(f_max=100.0, batch=2000 if lpp == 1 else 700)           # 321 bins
    f, S, dets, d, th = make_problem(oracle, cfg)
    kw, okw = {}, {}
    if option == "isco_cut":
        kw, okw = dict(isco_cut=1), dict(isco_cut=1)
    if option == "tidal":
        lam = inputs.tidal_lambdas(cfg, len(th))
        th = np.ascontiguousarray(np.hstack([th, lam]))
        kw, okw = dict(tidal_order=2), dict(lambdas=lam, tidal_order=2)
    with GwContext(f, d, S, dets, cfg.gmst, spin_order=cfg.spin_order, max_batch=len(th), **kw) as ctx:
        ctx.boundary_bins(vbins)
        ctx.force_grid(lpp, n_ctas)
        plan = ctx.plan(len(th))
        used = ctx.plan_boundary_bins(len(th))
        assert plan["lanes_per_prop"] == lpp and plan["n_ctas"] == n_ctas
        thd = _dev(torch, th)
        lnl, parts = ctx.lnl_batch(thd, want_parts=True)
        lnl2, parts2 = ctx.lnl_batch(thd, want_parts=True)
        torch.cuda.synchronize()
        assert torch.equal(lnl, lnl2) and torch.equal(parts, parts2)
    n_tiles = (len(th) + 256 // lpp - 1) // (256 // lpp)
    rows = [binding.plan_cta_segments(n_tiles, f.size, n_ctas, k, boundary_bins=used) for k in range(n_ctas)]
    n_empty = sum(int((r[:, 2] == r[:, 1]).sum()) for r in rows)
    if (lpp, n_ctas, vbins) in ((1, 12, 30), (1, 10, 40), (4, 12, 10), (4, 6, 30), (32, 4, 30), (32, 5, 20), (2, 4, 30)):
        assert used == vbins * lpp and n_empty > 0                        # these shapes do have zero-bin segments
    ref = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th[:, :11], cfg.spin_order, **okw)
    assert_lnl_close(lnl.cpu().numpy(), parts.cpu().numpy(), ref[0], ref[1])
