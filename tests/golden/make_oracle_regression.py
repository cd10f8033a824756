#!/usr/bin/env python3
"""Write tests/golden/oracle_regression.txt from the oracle alone (never from the CUDA path).

    python tests/golden/make_oracle_regression.py
Case: config C1 reduced to f_max = 64 Hz (177 bins), 12 proposals, 3 detectors, seeded as inputs.py states."""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle  # noqa: E402
from paper_1904_02863_b200 import inputs  # noqa: E402


def case():
    cfg = inputs.CONFIGS["C1"].reduced(f_max=64.0, batch=12)
    f, S, dets = inputs.frequency_grid(cfg), inputs.psd(cfg), inputs.detectors(cfg)
    d = inputs.make_data(cfg, oracle.waveform)
    th = inputs.proposals(cfg)
    lnl, parts, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, cfg.spin_order, n_threads=1)
    return lnl, parts


if __name__ == "__main__":
    lnl, parts = case()
    with open(os.path.join(HERE, "oracle_regression.txt"), "w") as fh:
        fh.write("# lnL, then parts[det][Re<d|h>, Im<d|h>, <h|h>] per proposal; hex floats; see README.md\n")
        for b in range(len(lnl)):
            row = [lnl[b]] + list(parts[b].ravel())
            fh.write(" ".join(float(v).hex() for v in row) + "\n")
    print("wrote", len(lnl), "rows")
