"""`-m gpu`: the diagnostic timeline build (paper_1904_02863_b200/timeline.py, csrc/libgwlnl_timeline.so = the product
sources with -DGW_TIMELINE) run in a process of its own (a process loads ONE library), on the headline workload: the
stamps are consistent, and the sweep of a one-CTA-per-SM grid costs what the SASS model of the hot loop says --
113.8 cycles per (warp, bin) (profiles/r2_fused_hot_loop_sass.md, tests/test_hot_loop_model.py) -- by the clock the
kernel actually ran at.  This is the measured half of DESIGN.md section 9's account of where C1's time goes."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_timeline_of_the_headline_workload_matches_the_hot_loop_model():
    out = subprocess.run([sys.executable, "-m", "paper_1904_02863_b200.timeline", "--workload", "C1", "--no-clock"],
                         cwd=ROOT, capture_output=True, text=True, timeout=900)
    assert out.returncode == 0, out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][0]
    rep = json.loads(line)["loaded_last_of_40_back_to_back_calls"]
    assert rep["plan"]["lanes_per_prop"] == 1 and rep["plan"]["n_ctas"] <= 148          # one CTA per SM
    one = rep["single_segment_ctas_us(min,median,max)"]
    assert 0.0 <= one["sweep_start"][0] <= one["sweep_start"][2] < one["sweep_end"][0] <= one["exit"][2] <= rep["span_us"] + 1e-9
    assert 1500.0 < rep["in_kernel_sm_mhz"] < 2100.0
    cyc = one["cycles_per_warp_bin_if_alone_on_the_SM"]
    assert abs(cyc[1] - 113.8) <= 0.03 * 113.8, cyc                                       # median over the CTAs
    assert rep["span_us"] < 135.0
    crossing = rep["crossing_ctas_us(min,median,max)"]
    if crossing is not None:                                                             # boundary bins: they end with the rest
        assert crossing["second_sweep_end"][2] <= one["sweep_end"][2] + 2.0
