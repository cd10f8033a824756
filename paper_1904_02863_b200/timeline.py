"""Diagnostic aid (NOT the product path): per-CTA timeline of the fused kernel and the SM clock it runs at.

    python -m paper_1904_02863_b200.timeline [--workload C1[:B]] [--boundary-bins V] [--force-grid N]

Builds ``csrc/libgwlnl_timeline.so`` (the product sources with -DGW_TIMELINE: thread 0 of every CTA of the fused kernel
stores the nanosecond globaltimer and clock64 at kernel entry, sweep start, every stage start, sweep end, ticket and exit;
csrc/gw_kernels.cu, GW_STAMP), loads THAT library instead of csrc/libgwlnl.so for this process, and prints

  * the timeline of the last of 40 back-to-back gw_lnl_batch calls (the loaded state): when the CTAs start, sweep, take
    their ticket and exit; the CTAs that cross a tile boundary; the in-kernel SM clock (clock64 against globaltimer
    between sweep start and sweep end);
  * the in-kernel clock and the kernel's span for a call that follows an idle gap of 0 ... 100 ms, and for the first 30
    calls after 0.5 s of idling (the clock ramp);
  * the cycles per (warp, bin) of the sweep, to hold against the SASS model of profiles/r2_fused_hot_loop_sass.md.

Nothing here is used by bench.py, the tests of the product path or the library itself.
"""
from __future__ import annotations

import argparse
import ctypes
import json
import time
from dataclasses import replace

import numpy as np

WORDS = 32          # 64-bit words per CTA (gw_kernels.cu, GW_STAMP)


def _problem(cfg, batch):
    from . import binding, inputs
    f, S, dets = inputs.frequency_grid(cfg), inputs.psd(cfg), inputs.detectors(cfg)
    d = inputs.make_data(cfg, binding.waveform_for_inputs)
    th = inputs.proposals(replace(cfg, batch=max(cfg.batch, batch)))[:batch]
    return f, S, dets, d, np.ascontiguousarray(th)


def _stats(x):
    x = np.asarray(x, dtype=np.float64)
    x = x[~np.isnan(x)]
    return None if x.size == 0 else [round(float(x.min()), 2), round(float(np.median(x)), 2), round(float(x.max()), 2)]


class Timeline:
    def __init__(self, workload: str = "C1", boundary_bins: int = -1, force_grid: int = 0):
        import torch
        from .csrc import build as csrc_build
        from . import binding, inputs
        self.torch = torch
        lib = binding.load_library(csrc_build.build_timeline())          # first use of the library in this process
        lib.gw_timeline_set_buffer.argtypes = [ctypes.c_void_p]
        lib.gw_timeline_set_buffer.restype = ctypes.c_int
        self.lib = lib
        name, _, b = workload.partition(":")
        self.cfg = inputs.CONFIGS[name]
        self.B = int(b) if b else self.cfg.batch
        f, S, dets, d, th = _problem(self.cfg, self.B)
        self.ctx = binding.GwContext(f, d, S, dets, self.cfg.gmst, spin_order=self.cfg.spin_order, max_batch=self.B)
        if boundary_bins >= 0:
            self.ctx.boundary_bins(boundary_bins)
        if force_grid:
            self.ctx.force_grid(1, force_grid)
        self.plan = self.ctx.plan(self.B)
        self.vbins = self.ctx.plan_boundary_bins(self.B)
        self.n_cta = self.plan["n_ctas"]
        self.th = torch.from_numpy(th).cuda()
        self.out = torch.empty(self.B, dtype=torch.float64, device="cuda")
        self.bufs = torch.zeros(32, self.n_cta * WORDS, dtype=torch.int64, device="cuda")
        n_tiles = (self.B + self.plan["props_per_cta"] - 1) // self.plan["props_per_cta"]
        rows = [binding.plan_cta_segments(n_tiles, self.cfg.n_bins, self.n_cta, c, boundary_bins=self.vbins)
                for c in range(self.n_cta)]
        self.bins = np.array([int((r[:, 2] - r[:, 1]).sum()) for r in rows])
        self.n_seg = np.array([int((r[:, 2] > r[:, 1]).sum()) for r in rows])

    def call(self):
        self.ctx.lnl_batch(self.th, out=self.out)

    def stamp_into(self, i):
        assert self.lib.gw_timeline_set_buffer(self.bufs[i].data_ptr()) == 0

    def read(self, i):
        """(times in us relative to the first CTA's entry [n_cta][24], clock64 values [n_cta][8]); 0 stamps -> NaN."""
        t = self.bufs[i].cpu().numpy().reshape(self.n_cta, WORDS).astype(np.float64)
        ns, clk = t[:, :24].copy(), t[:, 24:].copy()
        base = ns[:, 0].min()
        ns[ns == 0] = np.nan
        clk[clk == 0] = np.nan
        # a stamp the CTA did not reach in this call (e.g. the ticket of a two-level finish) may be left from an earlier one
        stale = ns < ns[:, :1]
        ns[stale] = np.nan
        clk[stale[:, :8]] = np.nan
        return (ns - base) * 1e-3, clk

    def clock_and_span(self, i):
        """In-kernel SM clock [MHz] (median over the single-segment CTAs: clock64 / globaltimer between sweep start and
        sweep end) and the kernel's span first entry -> last exit [us]."""
        us, clk = self.read(i)
        one = np.isnan(us[:, 5]) & ~np.isnan(us[:, 2])
        mhz = (clk[one, 2] - clk[one, 1]) / (us[one, 2] - us[one, 1])
        return round(float(np.median(mhz)), 1), round(float(np.nanmax(us[:, 4])), 2)

    # ---- the three reports -------------------------------------------------------------------------------------------
    def loaded(self, n_calls: int = 40):
        torch = self.torch
        for _ in range(n_calls):
            self.call()
        torch.cuda.synchronize()
        self.bufs[0].zero_()
        self.stamp_into(0)
        for _ in range(n_calls):
            self.call()
        torch.cuda.synchronize()
        us, clk = self.read(0)
        mhz, span = self.clock_and_span(0)
        one = np.isnan(us[:, 5])
        two = ~one
        sweep = us[one, 2] - us[one, 1]
        warps_per_sched = 2.0 * min(2, max(1, int(np.ceil(self.n_cta / 148.0))))
        bins_one = self.bins[one]
        # cycles per (warp, bin): a CTA's 8 warps sit on 4 schedulers; with two co-resident CTAs the older one runs first
        cyc = sweep * mhz / (bins_one * 2.0)
        rep = {"plan": self.plan, "boundary_bins": self.vbins, "in_kernel_sm_mhz": mhz, "span_us": span,
               "ctas": {"single_segment": int(one.sum()), "crossing_a_tile_boundary": int(two.sum())},
               "single_segment_ctas_us(min,median,max)": {
                   "sweep_start": _stats(us[one, 1]), "sweep_end": _stats(us[one, 2]), "ticket": _stats(us[one, 3]),
                   "exit": _stats(us[one, 4]), "sweep_length": _stats(sweep), "bins": _stats(bins_one),
                   "cycles_per_warp_bin_if_alone_on_the_SM": _stats(cyc) if warps_per_sched == 2.0 else None},
               "crossing_ctas_us(min,median,max)": None if not two.any() else {
                   "first_sweep_end": _stats(us[two, 2]), "second_sweep_start": _stats(us[two, 5]),
                   "between_the_segments": _stats(us[two, 5] - us[two, 2]), "second_sweep_end": _stats(us[two, 6]),
                   "exit": _stats(us[two, 4]), "bins": _stats(self.bins[two])},
               "stage_starts_us_median_single_segment": [round(float(np.nanmedian(us[one, k])), 2) for k in range(8, 24)
                                                         if not np.isnan(us[one, k]).all()],
               "last_exits_us": [round(float(v), 2) for v in np.sort(us[:, 4])[-6:]],
               "exit_minus_ticket_us_of_the_6_last": [round(float(v), 2) for v in
                                                      (us[:, 4] - np.where(np.isnan(us[:, 7]), us[:, 3], us[:, 7]))[np.argsort(us[:, 4])[-6:]]]}
        return rep

    def after_idle(self, gaps_us=(0, 20, 100, 1000, 10000, 100000), reps: int = 3):
        torch = self.torch
        out = {}
        for gap in gaps_us:
            vals = []
            for _ in range(reps):
                self.stamp_into(1)
                for _ in range(60):
                    self.call()                                   # ~7 ms of load on C1
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                while (time.perf_counter() - t0) * 1e6 < gap:
                    pass
                self.bufs[1].zero_()
                self.call()
                torch.cuda.synchronize()
                vals.append(self.clock_and_span(1))
            out[f"{gap} us"] = vals
        return out

    def ramp(self, n_calls: int = 30, idle_s: float = 0.5):
        torch = self.torch
        torch.cuda.synchronize()
        time.sleep(idle_s)
        self.bufs.zero_()
        torch.cuda.synchronize()
        time.sleep(idle_s)
        for i in range(n_calls):
            self.stamp_into(i)
            self.call()
        torch.cuda.synchronize()
        return [self.clock_and_span(i) for i in range(n_calls)]

    def synchronous_loop(self, n_calls: int = 200):
        torch = self.torch
        for i in range(n_calls):
            self.stamp_into(i % 32)
            self.bufs[i % 32].zero_()
            self.call()
            torch.cuda.synchronize()
        return [self.clock_and_span(i % 32) for i in range(n_calls - 5, n_calls)]


def main():
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("--workload", default="C1")
    ap.add_argument("--boundary-bins", type=int, default=-1, help="gw_ctx_boundary_bins (default: the library's)")
    ap.add_argument("--force-grid", type=int, default=0, help="pin the grid to this many one-lane CTAs")
    ap.add_argument("--no-clock", action="store_true", help="skip the idle-gap and ramp measurements")
    args = ap.parse_args()
    tl = Timeline(args.workload, args.boundary_bins, args.force_grid)
    print(json.dumps({"workload": args.workload, "loaded_last_of_40_back_to_back_calls": tl.loaded()}))
    if not args.no_clock:
        print(json.dumps({"workload": args.workload,
                          "[in-kernel MHz, span us] after an idle gap (60 calls of load, host waits, one call)": tl.after_idle()}))
        print(json.dumps({"workload": args.workload, "[in-kernel MHz, span us] of 30 consecutive calls after 0.5 s idle": tl.ramp()}))
        print(json.dumps({"workload": args.workload, "[in-kernel MHz, span us] last 5 of 200 synchronised calls": tl.synchronous_loop()}))


if __name__ == "__main__":
    main()
