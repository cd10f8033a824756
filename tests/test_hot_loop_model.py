"""`-m "not gpu"`: the hot loop of the fused kernel as ptxas built it, read from the SASS of csrc/libgwlnl.so
(csrc/hot_loop_model.py).  The loop sits at the 128-register limit of two CTAs per SM, and edits OUTSIDE it have made
ptxas spill around it and reorder it (a branch in the kernel's outer loop: 569 -> 596 model cycles per trip and 23 % on
the GPU).  These checks hold the product build to the loop that profiles/
r2_fused_hot_loop_sass.md documents: 41 fp64 instructions per (proposal, bin) for three detectors, no spill inside the
loop, and the issue-cycle model of 113.8 cycles per (warp, bin) within 1 %."""
import os

import pytest

CUOBJDUMP = "/usr/local/cuda/bin/cuobjdump"
pytestmark = pytest.mark.skipif(not os.path.exists(CUOBJDUMP), reason="cuobjdump not installed")


@pytest.fixture(scope="module")
def hlm():
    from paper_1904_02863_b200.csrc import build as csrc_build, hot_loop_model
    return hot_loop_model, csrc_build.build()


def test_headline_hot_loop_is_the_documented_one(hlm):
    mod, lib = hlm
    m = mod.model(lib, 3)
    assert m["spill_in_loop"] == 0
    assert m["fp64"] == 5 * 41 and m["lds"] == 5 * 8                  # five bins per trip
    assert m["model_cycles_per_trip"] <= 569.0 * 1.01, m              # 113.8 cycles per (warp, bin)


@pytest.mark.parametrize("ndet,fp64_per_bin", [(1, 25), (2, 33), (4, 49)])
def test_other_detector_counts_have_no_spill_in_the_loop(hlm, ndet, fp64_per_bin):
    mod, lib = hlm
    m = mod.model(lib, ndet)
    assert m["spill_in_loop"] == 0 and m["fp64"] == 5 * fp64_per_bin, m
