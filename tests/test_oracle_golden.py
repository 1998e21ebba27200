"""The oracle still reproduces the values stored by tests/golden/make_golden.py (oracle-only)."""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden"))


def test_config1_golden_values():
    import make_golden
    got = make_golden.compute()
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "config1_oracle.txt")
    stored = {}
    for line in open(path):
        if line.startswith("#"):
            continue
        k, *v = line.split()
        stored[k] = np.array([float(x) for x in v])
    assert set(stored) == set(got)
    for k in stored:
        assert np.allclose(got[k], stored[k], rtol=1e-12, atol=0), k
    # the prescribed omega = 1.0 makes the history grow by ~3.1-3.6x per sweep
    h = stored["richardson_hist"]
    assert np.all(h[1:] / h[:-1] > 2.5)
