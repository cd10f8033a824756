"""The oracle still reproduces its stored regression values (tests/golden/README.md): not a pin, a tripwire."""
import os
import sys

import numpy as np

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def test_oracle_regression_values(oracle):
    sys.path.insert(0, GOLD)
    import make_oracle_regression as mk
    lnl, parts = mk.case()
    rows = [l.split() for l in open(os.path.join(GOLD, "oracle_regression.txt")) if not l.startswith("#")]
    want = np.array([[float.fromhex(v) for v in r] for r in rows])
    got = np.concatenate([lnl[:, None], parts.reshape(len(lnl), -1)], axis=1)
    assert got.shape == want.shape
    # libm differences between machines are allowed at the few-ulp level of the terms being summed
    scale = np.abs(want[:, 1:]).max(axis=1, keepdims=True)
    assert np.all(np.abs(got - want) <= 1e-11 * scale)
