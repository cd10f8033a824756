#!/usr/bin/env python3
"""bench.py -- likelihood evaluations/s of the fused waveform+lnL hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C1] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch of synthetic proposals: gw_lnl_batch = setup kernel
(K1) + fused kernel (K3) on the workload's full batch.  The default workload is BASELINE.json configs[1]
(C1: 3 detectors, 8113 bins, 4096 proposals); --workload C0|C2|C3|C4:<B> runs the others (parity-test cases).
Inputs are seeded and synthetic (paper_1904_02863_b200/inputs.py); the injection is computed with the library's
own gw_waveform_batch, so the product arm never touches oracle/.

Timing: per-step CUDA events on the launching stream, L2 flushed (a 256 MiB write, then a 256 MiB read of a
second buffer so that no dirty lines are left for the timed kernel to write back) before every timed step,
>= 3 warm-up steps after a clock ramp, clocks sampled through NVML during the timed region.  N > 1: one process
per GPU under torchrun, proposals sharded with no collective on the data path (weak scaling); NCCL carries only
the barrier and the max-over-ranks reduction of the measured time.

--impl reference times the CPU oracle (oracle/, plain C, fp64) on the host cores on a bounded sample of the
same workload; it is the one place besides `cpu_baseline` where bench.py executes oracle/.
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "likelihood evals/sec (fp64, waveform+lnL)"
UNIT = "lnL/s"
FP64_LANES_PER_SM = 64          # B200 fp64 FMA lanes per SM (37.2 TFLOP/s at 1965 MHz x 148 SMs)
L2_FLUSH_BYTES = 256 << 20
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel are NOT measured by this script:
# they are carried over from the committed `ncu --set full` captures listed in profiles/dram_traffic.json (the JSON
# line names the capture in roofline.traffic_source); null where no capture exists for the workload and options.
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "dram_traffic.json")


def ncu_traffic(key):
    """(bytes per launch, source) from profiles/dram_traffic.json, or (None, None)."""
    try:
        ent = json.load(open(TRAFFIC_FILE)).get(key)
    except Exception:
        ent = None
    return (float(ent["bytes_per_launch"]), ent["source"]) if ent else (None, None)


def parse_workload(spec):
    from paper_1904_02863_b200 import inputs
    name, _, b = spec.partition(":")
    cfg = inputs.CONFIGS[name]
    batch = int(b) if b else (4096 if name == "C4" else cfg.batch)
    return name, cfg, batch


def executed_per_bin(n_det, tidal_order=0):
    """fp64 instructions the fused kernel EXECUTES per (proposal, bin): 9 phase + 12 sincos +
    4 for the reference detector + 8 per further detector (+4 with the tidal option) -- 41 at N_det = 3.  The closed
    form <h|h> and the trimmed sincos are algorithmic savings, so this is below W_alg."""
    return 9 + 12 + 4 + 8 * (n_det - 1) + (4 if tidal_order else 0)


def walg_per_bin(n_det, tidal_order=0):
    """Algorithmic fp64 FMA-equivalents per (proposal, bin): SURVEY.md 8(d) W_alg = 31 + 8 N_det; the tidal
    option adds x^5 (t10 + t12 x^2) from the tabulated x, x^2: 4 more."""
    return 31 + 8 * n_det + (4 if tidal_order else 0)


class ClockSampler:
    """NVML clock / throttle-reason samples during the timed region (a thread; ~2 ms cadence)."""

    def __init__(self, index):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as e:          # no NVML: report that, do not invent numbers
            self.nv, self.err = None, repr(e)

    def _run(self):
        nv = self.nv
        names = {"hw_slowdown": nv.nvmlClocksEventReasonHwSlowdown,
                 "hw_thermal_slowdown": nv.nvmlClocksEventReasonHwThermalSlowdown,
                 "sw_thermal_slowdown": nv.nvmlClocksEventReasonSwThermalSlowdown,
                 "sw_power_cap": nv.nvmlClocksEventReasonSwPowerCap}
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.002)

    def __enter__(self):
        if self.nv is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thread is not None:
            self._thread.join()

    def summary(self):
        if self.nv is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml unavailable: " + self.err]}
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def build_problem(cfg, batch_total, tidal_order=0):
    """freqs, data, psd, det rows, theta[batch_total] -- the injection comes from the library's own waveform.
    With the tidal option theta has 13 columns (seeded Lambda_1, Lambda_2 appended; the injection stays point-mass)."""
    from dataclasses import replace
    from paper_1904_02863_b200 import binding, inputs
    f = inputs.frequency_grid(cfg)
    S = inputs.psd(cfg)
    dets = inputs.detectors(cfg)
    d = inputs.make_data(cfg, binding.waveform_for_inputs)
    draw = max(cfg.batch, batch_total)
    th = inputs.proposals(replace(cfg, batch=draw))[:batch_total]
    if tidal_order:
        th = np.ascontiguousarray(np.hstack([th, inputs.tidal_lambdas(replace(cfg, batch=draw))[:batch_total]]))
    return f, S, dets, d, th


def oracle_rate(cfg, f, S, dets, d, th, target_s, n_threads=0, tidal_order=0):
    """Time the oracle, as it stands, for about target_s seconds of wall time on a bounded sample of the
    workload: a prefix of the proposals, passed over repeatedly if the whole batch is quicker than target_s."""
    import oracle
    oracle.build()

    def run(rows):
        kw = dict(lambdas=rows[:, 11:13], tidal_order=tidal_order) if tidal_order else {}
        return oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, rows[:, :11], cfg.spin_order, n_threads, **kw)

    pilot = th[: min(len(th), max(2, 2 * (os.cpu_count() or 1)))]
    run(pilot)                                                                              # thread start-up
    t0 = time.perf_counter()
    run(pilot)
    dt = max(time.perf_counter() - t0, 1e-6)
    n = int(min(len(th), max(len(pilot), len(pilot) * target_s / dt)))
    passes = max(1, int(round(target_s / max(dt * n / len(pilot), 1e-6))))
    t0 = time.perf_counter()
    for _ in range(passes):
        _, _, used = run(th[:n])
    dt = time.perf_counter() - t0
    return n * passes / dt, used, n, dt, passes


def run_reference(args):
    """--impl reference: the oracle on the host cores; each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    name, cfg, batch = parse_workload(args.workload)
    import oracle
    oracle.build()
    from paper_1904_02863_b200 import inputs
    f, S, dets = inputs.frequency_grid(cfg), inputs.psd(cfg), inputs.detectors(cfg)
    d = inputs.make_data(cfg, oracle.waveform)
    th = inputs.proposals(cfg)[:batch] if batch <= cfg.batch else inputs.proposals(cfg)
    # size one step to ~ (90 s budget) / (steps + warmup)
    per_step_s = min(10.0, 90.0 / max(1, args.steps + args.warmup))
    cores = os.cpu_count() or 1          # torchrun exports OMP_NUM_THREADS=1; the oracle is timed on all host cores
    rate, used, n, _, _ = oracle_rate(cfg, f, S, dets, d, th, min(per_step_s, 3.0), n_threads=cores)
    n = max(1, min(len(th), int(rate * per_step_s)))
    for _ in range(args.warmup):
        oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th[:n], cfg.spin_order, cores)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _, _, used = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th[:n], cfg.spin_order, cores)
    dt = time.perf_counter() - t0
    value = n * args.steps / dt
    sample = f"first {n} of {batch} proposals of {name} per step, all {cfg.n_bins} bins x {cfg.n_det} detectors"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{name}: {cfg.n_det} det x {cfg.n_bins} bins x {batch} proposals per GPU",
                       "global_batch": batch, "bins": cfg.n_bins, "detectors": cfg.n_det},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": used, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def run_population(args):
    """--workload P0|P1|P2[:B]: the population likelihood, Eq. 3.  A step is one
    gw_pop_lnl_batch call: B hyper-parameter proposals over the N x n resident samples.  HBM-bound map-reduce: the
    roofline is read against bytes (7 input arrays of the paper's data flow, = 56 B per sample and pass;
    the kernel streams 8 transformed planes = 64 B)."""
    import torch
    from paper_1904_02863_b200.csrc import build as csrc_build
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        raise SystemExit("bench.py: the population workload is timed on one GPU")
    torch.cuda.set_device(0)
    if os.path.exists(csrc_build.NVCC):
        csrc_build.build()
        csrc_build.build_probe()
    from paper_1904_02863_b200 import inputs, probes
    from paper_1904_02863_b200.population import GwPopContext
    name, _, b = args.workload.partition(":")
    cfg = inputs.POP_CONFIGS[name]
    B = int(b) if b else 1
    s, p0 = inputs.pop_samples(cfg)
    lam_all = inputs.pop_lambdas(inputs.PopConfig(cfg.name, cfg.index, cfg.n_events, cfg.n_samples, max(B, cfg.batch)))
    lam = np.ascontiguousarray(lam_all[:B])
    ctx = GwPopContext(s, p0, max_batch=B)
    lam_d = torch.from_numpy(lam).cuda()
    out = torch.empty(B, dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream()
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device="cuda")
    n_samp = cfg.n_events * cfg.n_samples
    in_l2 = n_samp * 64 <= (100 << 20)

    def step():
        ctx.lnl_batch(lam_d, out=out)

    probes.fp64_fma_rate(1 << 14)
    for _ in range(max(3, args.warmup)):
        step()
    torch.cuda.synchronize()
    ev0 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    ev1 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    launches0 = ctx.launch_count()
    with ClockSampler(0) as clk:
        for i in range(args.steps):
            flush.fill_(i & 0xff)
            ev0[i].record(stream); step(); ev1[i].record(stream)
        clock_after_mhz = probes.sm_clock_mhz()
        torch.cuda.synchronize()
    launches = ctx.launch_count() - launches0
    step_ms = np.array([a.elapsed_time(b_) for a, b_ in zip(ev0, ev1)])
    value = B * args.steps / (step_ms.sum() * 1e-3)
    # kernel-level pass: every sample is the last of a burst of flushed steps without a host synchronisation in between,
    # so that the SM clock is the loaded one (see run_ours and profiles/r2_timeline.md)
    step_est_ms = float(step_ms.mean()) + 0.05
    burst = int(min(64, max(4, np.ceil(3.0 / step_est_ms))))
    n_samples = int(max(10, min(args.steps, 2000.0 / (burst * step_est_ms))))
    ctx.kernel_timing(True)
    k_ms = []
    for i in range(n_samples):
        for j in range(burst):
            flush.fill_((i + j) & 0xff)
            step()
        k_ms.append(ctx.last_kernel_ms())
    ctx.kernel_timing(False)
    k_ms = np.array(k_ms)
    main_ms = float(k_ms[:, 1].mean())
    passes = 1 if B <= 2 else (B + 3) // 4
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    load_gbs, _ = probes.load_bandwidth(2 << 30, 10)
    alg_bytes = 56.0 * n_samp * passes
    achieved = alg_bytes / (main_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": "pop_main_kernel<%d>" % (B if B <= 2 else 4), "achieved": achieved, "peak": hbm,
                "unit": "GB/s", "frac": achieved / hbm, "traffic": ncu_traffic("%s:%d" % (name, B))[0],
                "traffic_source": ncu_traffic("%s:%d" % (name, B))[1],
                "peak_source": "MEASURED_PEAKS.json hbm_gbs (copy)" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)",
                "pure_load_ceiling_GBps": load_gbs, "frac_of_pure_load": achieved / load_gbs,
                "algorithmic_bytes_per_launch": alg_bytes, "bytes_streamed_per_launch": 64.0 * n_samp * passes,
                "passes_over_the_samples": passes, "proposals_per_pass": min(B, 4),
                "sample_lambda_pairs_per_s": n_samp * B / (main_ms * 1e-3),
                "kernel_ms": main_ms, "kernel_ms_median": float(np.median(k_ms[:, 1])), "kernel_ms_best": float(k_ms[:, 1].min()),
                "kernel_ms_samples": n_samples, "kernel_ms_burst": burst,
                "setup_kernel_ms": float(k_ms[:, 0].mean()), "finish_kernel_ms": float(k_ms[:, 2].mean()),
                "note": "one proposal per pass is HBM-bound; with 4 proposals per pass every plane value read is used four "
                        "times and the exponentials (4 per sample and proposal) bound the kernel instead"}
    # end to end: host Lambda in, host lnL out, synchronised
    lam_pin = torch.from_numpy(lam).pin_memory().numpy()
    out_pin = torch.empty(B, dtype=torch.float64).pin_memory().numpy()
    e2e_warm, t_w = 0, time.perf_counter()                  # as in run_ours: >= max(3, --warmup) calls and >= 0.5 s
    while e2e_warm < max(3, args.warmup) or (time.perf_counter() - t_w < 0.5 and e2e_warm < 20000):
        ctx.lnl_batch_host(lam_pin, out=out_pin)
        e2e_warm += 1
    t0 = time.perf_counter()
    for _ in range(args.steps):
        ctx.lnl_batch_host(lam_pin, out=out_pin)
    e2e_s = time.perf_counter() - t0
    e2e = {"value": B * args.steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(lam.nbytes), "d2h_bytes_per_step": 8 * B,
           "ms_per_step": 1e3 * e2e_s / args.steps, "warmup_calls": e2e_warm, "api": "gw_pop_lnl_batch_host (host Lambda in, host lnL out, stream synchronised)"}
    cpu = None
    if not args.no_cpu_baseline:
        import oracle
        oracle.build()
        nl = 1
        t0 = time.perf_counter()
        _, _, used = oracle.pop_lnl(s, p0, lam_all[:nl], n_threads=os.cpu_count() or 1)
        dt = time.perf_counter() - t0
        nl = int(max(1, min(cfg.batch, args.cpu_seconds / max(dt, 1e-3))))
        t0 = time.perf_counter()
        _, _, used = oracle.pop_lnl(s, p0, lam_all[:nl], n_threads=os.cpu_count() or 1)
        dt = time.perf_counter() - t0
        cpu = {"value": nl / dt, "unit": UNIT, "cores": used, "kind": "oracle",
               "sample": f"{nl} hyper-parameter proposals over all {cfg.n_events} x {cfg.n_samples} samples, {dt:.1f} s wall"}
    clocks = clk.summary()
    clocks["sm_mhz_measured_after_timed_region"] = clock_after_mhz
    ctx.close()
    line = {"metric": "population likelihood evals/sec (fp64, PAPER.md Eq. 3)", "value": value, "unit": UNIT, "n_gpus": 1,
            "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": float(step_ms.mean()),
            "ms_per_step_median": float(np.median(step_ms)), "ms_per_step_best": float(step_ms.min()),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{name}: {cfg.n_events} events x {cfg.n_samples} samples, {B} hyper-parameter proposals per call",
                       "samples": n_samp, "global_batch": B,
                       "l2": "flushed before every timed step (256 MiB write)" + ("; the sample planes (%d MB) would otherwise stay in L2" % (n_samp * 64 >> 20) if in_l2 else "; the sample planes exceed L2")},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu}
    print(json.dumps(line))


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1904_02863_b200.csrc import build as csrc_build

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if local == 0 and os.path.exists(csrc_build.NVCC):
        csrc_build.build()             # no-op when csrc/libgwlnl.so is newer than its sources
        csrc_build.build_probe()
    if world > 1:
        dist.barrier()                 # nobody loads the library while local rank 0 may be rebuilding it
    from paper_1904_02863_b200 import GwContext, binding, probes
    n_gpus = world

    name, cfg, batch = parse_workload(args.workload)
    f, S, dets, d, th_all = build_problem(cfg, batch * world, args.tidal_order)
    from paper_1904_02863_b200.sharding import shard_range
    lo, hi = shard_range(batch * world, rank, world)
    th = np.ascontiguousarray(th_all[lo:hi])
    B, M, n_det = len(th), cfg.n_bins, cfg.n_det
    stream = torch.cuda.current_stream()

    ctx = GwContext(f, d, S, dets, cfg.gmst, spin_order=cfg.spin_order, max_batch=B,
                    isco_cut=int(args.isco_cut), phase_marginal=int(args.phase_marginal),
                    tidal_order=int(args.tidal_order))
    if args.force_grid or args.force_lpp:                 # tuning aid (include/gwlnl_tuning.h): pin the launch shape
        ctx.force_grid(args.force_lpp, args.force_grid)
    if args.no_cluster:
        ctx.cluster_finish(False)
    if args.no_host_graph:
        ctx.host_graph(False)
    thd = torch.from_numpy(th).cuda()
    lnl = torch.empty(B, dtype=torch.float64, device="cuda")
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device="cuda")
    flush_rd = torch.zeros(L2_FLUSH_BYTES // 8, dtype=torch.int64, device="cuda")
    flush_sink = torch.zeros((), dtype=torch.int64, device="cuda")

    def flush_l2(i):
        """Write a buffer larger than L2, then read a second one: the L2 ends up holding clean, unrelated lines
        (a write-only flush would leave ~126 MB of dirty lines whose write-back the timed kernel would pay for)."""
        flush.fill_(i & 0xff)
        torch.sum(flush_rd, dim=(0,), out=flush_sink)
    plan = ctx.plan(B)

    # ---- clock ramp + measured fp64 FMA rate (the measured roofline denominator) ----
    fma_rate, _ = probes.fp64_fma_rate(1 << 14)
    fma_rate, _ = probes.fp64_fma_rate(1 << 15)

    def step():
        ctx.lnl_batch(thd, out=lnl)

    for _ in range(max(3, args.warmup)):
        step()
    torch.cuda.synchronize()

    # ---- timed region: K steps, per-step events, L2 flush before each ----
    ev0 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    ev1 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    launches0 = ctx.launch_count()
    with ClockSampler(local) as clk:
        for i in range(args.steps):
            flush_l2(i)
            ev0[i].record(stream)
            step()
            ev1[i].record(stream)
        clock_after_mhz = probes.sm_clock_mhz()      # the clock the timed kernels actually ran at (enqueued right behind them)
        torch.cuda.synchronize()
    launches = ctx.launch_count() - launches0
    if world > 1:
        dist.barrier()
    step_ms = np.array([a.elapsed_time(b) for a, b in zip(ev0, ev1)])
    total_ms = float(step_ms.sum())
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    value = B * world * args.steps / (total_ms * 1e-3)

    # ---- kernel-level pass (same stream, events inside the library around K3), flushed likewise ----
    # The library keeps one set of events per context, so a sample is read with a host synchronisation -- and an idle gap
    # of a few tens of microseconds is enough for the SM clock to fall by ~9 % (1.79 GHz against 1.95 GHz inside the fused
    # kernel), while it needs ~2 ms of load to come back (profiles/r2_timeline.md).  Every sample is therefore the LAST
    # call of a burst of flushed steps enqueued without a synchronisation, long enough (>= 3 ms) for the clock to be where
    # it is in the timed region above; kernel_ms_after_idle keeps the figure of a kernel that starts on an idle GPU.
    step_est_ms = total_ms / args.steps + 0.1                 # + the two flush kernels
    burst = int(min(64, max(4, np.ceil(3.0 / step_est_ms))))
    n_samples = int(max(10, min(args.steps, 2000.0 / (burst * step_est_ms))))
    ctx.kernel_timing(True)
    k_ms, s_ms, k_idle_ms = [], [], []
    for i in range(n_samples):
        for j in range(burst):
            flush_l2(i + j)
            step()
        a, b = ctx.last_kernel_ms()
        s_ms.append(a)
        k_ms.append(b)
    for i in range(min(n_samples, 20)):                       # one flushed step after a host synchronisation
        flush_l2(i)
        step()
        k_idle_ms.append(ctx.last_kernel_ms()[1])
    ctx.kernel_timing(False)
    fused_ms = float(np.mean(k_ms))
    # what the kernel-alone measurement includes besides the kernel: an empty kernel of the same launch shape, timed the same way
    floor_ms = probes.launch_floor_ms(plan["n_ctas"], 256, 63000, 50)
    # the sustained rate of a sampler loop: calls back to back between ONE pair of events, no L2 flush, no events inside
    n_b2b = 50
    b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    step(); b0.record(stream)
    for _ in range(n_b2b):
        step()
    b1.record(stream); torch.cuda.synchronize()
    b2b_ms = b0.elapsed_time(b1) / n_b2b
    walg = walg_per_bin(n_det, args.tidal_order)
    wexe = executed_per_bin(n_det, args.tidal_order)
    pairs = float(B) * M                                   # (proposal, bin) pairs with algorithmic work
    if args.isco_cut:                                      # only bins up to each proposal's f_ISCO carry work
        from paper_1904_02863_b200.inputs import P_MC, P_Q
        m_tot = th[:, P_MC] * (1.0 + th[:, P_Q]) ** 1.2 / th[:, P_Q] ** 0.6
        f_isco = 1.0 / (6.0 ** 1.5 * np.pi * m_tot * 4.925490947641267e-06)
        pairs = float(np.searchsorted(f, f_isco, side="right").sum())
    flops_per_launch = 2.0 * walg * pairs
    achieved = flops_per_launch / (fused_ms * 1e-3) / 1e12
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    n_sm = torch.cuda.get_device_properties(local).multi_processor_count
    peak = n_sm * FP64_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    plain = not (args.isco_cut or args.phase_marginal or args.tidal_order)
    traffic, traffic_source = ncu_traffic(name) if (B == cfg.batch and plain and world == 1) else (None, None)
    roofline = {"bound": "alu", "kernel": "fused_kernel<%d>" % n_det, "achieved": achieved, "peak": peak,
                "unit": "TFLOP/s", "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_source,
                "frac_note": "frac credits the declared algorithmic work W_alg (SURVEY.md 8(d)); frac_executed counts the "
                             "fp64 instructions the kernel issues and is the fraction of raw fp64-pipe issue slots",
                "executed_fp64_per_prop_bin": wexe, "frac_executed": achieved / peak * wexe / walg,
                "kernel_ms_median": float(np.median(k_ms)), "kernel_ms_best": float(np.min(k_ms)),
                "kernel_ms_samples": n_samples, "kernel_ms_burst": burst,
                "kernel_ms_note": "each sample: the last of `kernel_ms_burst` flushed steps enqueued without a host synchronisation "
                                  "(SM clock as in the timed region); kernel_ms_after_idle: one flushed step right after a host "
                                  "synchronisation (the SM clock has fallen; profiles/r2_timeline.md)",
                "kernel_ms_after_idle": float(np.mean(k_idle_ms)),
                "launch_floor_ms": floor_ms, "frac_net_of_launch_floor": flops_per_launch / ((fused_ms - floor_ms) * 1e-3) / 1e12 / peak,
                "launch_floor_note": "kernel_ms is one launch between two CUDA events; an EMPTY kernel of the same launch shape timed "
                                     "the same way reads launch_floor_ms (gw_probe_launch_floor).  frac uses kernel_ms as measured.",
                "back_to_back_ms_per_call": b2b_ms, "back_to_back_note": "%d gw_lnl_batch calls (setup + fused kernel, overlapped by "
                "programmatic dependent launch) between one pair of events, no L2 flush: the sustained rate of a sampler loop" % n_b2b,
                "frac_back_to_back_step": flops_per_launch / (b2b_ms * 1e-3) / 1e12 / peak,
                "peak_source": "derived: %d SMs x %d fp64 FMA lanes x 2 flop x %.0f MHz (%s)"
                               % (n_sm, FP64_LANES_PER_SM, sm_max,
                                  "MEASURED_PEAKS.json sm_max_mhz" if "sm_max_mhz" in peaks else "fallback clock, B200_PROFILING.md"),
                "peak_measured_fma_probe": 2 * fma_rate / 1e12, "frac_of_measured": achieved / (2 * fma_rate / 1e12),
                "flop_per_launch": flops_per_launch, "walg_fma_per_prop_bin": walg, "proposal_bin_pairs": pairs,
                "kernel_ms": fused_ms, "setup_kernel_ms": float(np.mean(s_ms))}

    # ---- end to end: host buffers through gw_lnl_batch_host (H2D + kernels + D2H + sync inside the call) ----
    th_pin = torch.from_numpy(th).pin_memory()
    out_pin = torch.empty(B, dtype=torch.float64).pin_memory()
    th_host, out_host = th_pin.numpy(), out_pin.numpy()
    # Warm-up: at least max(3, --warmup) calls and at least 0.5 s of calls.  A loop of synchronous calls needs 0.1-0.25 s
    # to reach its steady rate (measured on C1, blocks of 500 calls: 153.9 us per call in the first block after 300 warm-up
    # calls, then 141.9 / 142.0 / 141.9; the kernels' own times are constant, so it is the host side of the loop --
    # link and CPU power states -- that settles).  A sampler makes millions of such calls; the steady rate is the figure.
    e2e_warm, t_w = 0, time.perf_counter()
    while e2e_warm < max(3, args.warmup) or (time.perf_counter() - t_w < 0.5 and e2e_warm < 20000):
        ctx.lnl_batch_host(th_host, out=out_host)
        e2e_warm += 1
    if world > 1:
        dist.barrier()
    e2e_calls = np.empty(args.steps)
    t0 = time.perf_counter()
    for i in range(args.steps):
        t1 = time.perf_counter()
        ctx.lnl_batch_host(th_host, out=out_host)
        e2e_calls[i] = time.perf_counter() - t1
    e2e_s = time.perf_counter() - t0
    if world > 1:
        t = torch.tensor([e2e_s], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    e2e = {"value": B * world * args.steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(th.nbytes) * world,
           "d2h_bytes_per_step": int(out_host.nbytes) * world, "ms_per_step": 1e3 * e2e_s / args.steps,
           "ms_per_step_median": 1e3 * float(np.median(e2e_calls)), "ms_per_step_best": 1e3 * float(e2e_calls.min()),
           "warmup_calls": e2e_warm,
           "api": "gw_lnl_batch_host (pinned host theta in, host lnL out, stream synchronised)"}

    extra = {}
    # ---- small batches: latency of one call replayed from a CUDA graph (SURVEY.md 8(d) timing protocol) ----
    if rank == 0 and B <= 256:
        g = torch.cuda.CUDAGraph()
        side = torch.cuda.Stream()
        side.wait_stream(stream)
        with torch.cuda.stream(side):
            ctx.lnl_batch(thd, out=lnl, stream=side)
            with torch.cuda.graph(g, stream=side):
                ctx.lnl_batch(thd, out=lnl, stream=side)
        stream.wait_stream(side)
        torch.cuda.synchronize()
        for _ in range(10):
            g.replay()
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n_rep = 200
        g0.record(stream)
        for _ in range(n_rep):
            g.replay()
        g1.record(stream)
        torch.cuda.synchronize()
        extra["cuda_graph_replay"] = {"ms_per_call": g0.elapsed_time(g1) / n_rep, "calls": n_rep,
                                      "note": "back-to-back replays of one captured gw_lnl_batch, no L2 flush"}

    # ---- the waveform-only kernel (north_star item (3)): achieved HBM GB/s ----
    if rank == 0 and not args.no_waveform:
        wb = min(B, max(1, int((2 << 30) // (n_det * M * 16))))
        h = torch.empty((wb, n_det, M), dtype=torch.complex128, device="cuda")
        thw = thd[:wb].contiguous()
        for _ in range(3):
            ctx.waveform_batch(thw, out=h)
        ctx.kernel_timing(True)
        w_ms = []
        for i in range(max(3, min(args.steps, 10))):
            flush_l2(i)
            ctx.waveform_batch(thw, out=h)
            w_ms.append(ctx.last_kernel_ms()[1])
        ctx.kernel_timing(False)
        gbs = wb * n_det * M * 16 / (np.mean(w_ms) * 1e-3) / 1e9
        hbm = float(peaks.get("hbm_gbs", 6650.0))
        del h
        store_gbs, _ = probes.store_bandwidth(2 << 30, 10)          # the pure-store ceiling, same run
        extra["waveform_kernel"] = {"proposals": wb, "bytes_stored": wb * n_det * M * 16, "kernel_ms": float(np.mean(w_ms)),
                                    "kernel_ms_median": float(np.median(w_ms)), "kernel_ms_best": float(np.min(w_ms)),
                                    "achieved_GBps": gbs, "hbm_peak_GBps": hbm,
                                    "peak_source": "MEASURED_PEAKS.json hbm_gbs (copy: read + write)" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)",
                                    "frac": gbs / hbm,
                                    "pure_store_ceiling_GBps": store_gbs, "frac_of_pure_store": gbs / store_gbs,
                                    "pure_store_source": "gw_probe_store_bandwidth: 2 GiB of 16-byte streaming stores, best of 10, this run"}

    # ---- CPU baseline: the oracle as it stands on this box's host cores (rank 0, N = 1 only) ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        rate, used, n, dt, passes = oracle_rate(cfg, f, S, dets, d, th, args.cpu_seconds, n_threads=os.cpu_count() or 1,
                                                    tidal_order=args.tidal_order)
        cpu = {"value": rate, "unit": UNIT, "cores": used, "kind": "oracle",
               "sample": f"first {n} of {B} proposals x {passes} passes, all {M} bins x {n_det} detectors, {dt:.1f} s wall"}
        r1, u1, n1, dt1, p1 = oracle_rate(cfg, f, S, dets, d, th, min(3.0, args.cpu_seconds), n_threads=1,
                                              tidal_order=args.tidal_order)
        cpu["single_thread"] = {"value": r1, "cores": u1, "sample": f"first {n1} proposals x {p1} passes, {dt1:.1f} s wall"}

    clocks = clk.summary()
    clocks["sm_mhz_measured_after_timed_region"] = clock_after_mhz
    clocks["note"] = ("sm_mhz: NVML samples during the timed region (the requested clock); sm_mhz_measured_after_timed_region: "
                      "clock64 against globaltimer in a probe kernel enqueued right behind the last timed step")
    ctx.close()
    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": n_gpus, "steps": args.steps,
                "warmup": max(3, args.warmup), "ms_per_step": total_ms / args.steps,
                "ms_per_step_median": float(np.median(step_ms)), "ms_per_step_best": float(np.min(step_ms)),
                "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": f"{name}: {n_det} det x {M} bins x {B} proposals per GPU",
                           "global_batch": B * world, "bins": M, "detectors": n_det, "parallelism": f"proposals sharded x{world}",
                           "l2": "flushed before every timed step: 256 MiB write, then a 256 MiB read of a second buffer (no dirty lines left)", "plan": plan,
                           "pinned": {"grid": args.force_grid, "lanes_per_prop": args.force_lpp, "no_cluster": bool(args.no_cluster)},
                           "options": {"isco_cut": int(args.isco_cut), "phase_marginal": int(args.phase_marginal),
                                       "tidal_order": int(args.tidal_order)}},
                "bin_det_proposals_per_s": value * M * n_det,
                "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
                "roofline": roofline, "cpu_baseline": cpu}
        line.update(extra)
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C1")
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-waveform", action="store_true")
    ap.add_argument("--force-grid", type=int, default=0, help="tuning aid: pin the fused kernel's grid to this many CTAs")
    ap.add_argument("--force-lpp", type=int, default=0, help="tuning aid: pin the lanes per proposal (1, 2, ..., 32)")
    ap.add_argument("--no-host-graph", action="store_true", help="tuning aid: small host calls launch by launch, not through the library's graph")
    ap.add_argument("--no-cluster", action="store_true", help="tuning aid: small grids through the ticket finish, not clusters")
    ap.add_argument("--isco-cut", action="store_true", help="NEXT-1 option: h = 0 above f_ISCO (not the headline config)")
    ap.add_argument("--phase-marginal", action="store_true", help="NEXT-1 option: lnL marginalised over phi_c")
    ap.add_argument("--tidal-order", type=int, default=0, choices=[0, 1, 2],
                    help="NEXT-1 option: 5PN (1) or 5PN + 6PN (2) tidal phase terms; theta rows of 13 columns")
    args = ap.parse_args()
    if args.workload.startswith("P"):
        if args.impl == "reference":
            raise SystemExit("bench.py: --impl reference covers the single-event workloads C0..C4")
        run_population(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
