"""Drift guard: the oracle's config-1 result must equal the stored samples (tests/golden/make_golden.py)."""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.join(os.path.dirname(__file__), "golden"))
import make_golden  # noqa: E402


def test_cfg1_oracle_matches_stored_samples():
    psi = make_golden.run_cfg1()
    path = os.path.join(os.path.dirname(__file__), "golden", "cfg1_oracle_samples.txt")
    rows = [l.split() for l in open(path) if not l.startswith("#")]
    for r in rows:
        if r[0] == "norm":
            assert abs(np.sum(np.abs(psi) ** 2) / float.fromhex(r[1]) - 1) < 1e-13
        else:
            j, i = int(r[0]), int(r[1])
            ref = complex(float.fromhex(r[2]), float.fromhex(r[3]))
            assert abs(psi[j, i] - ref) <= 1e-13 * max(abs(ref), 1e-3)
    # physics sanity of the stored state: the norm decayed roughly like exp(-gamma t), gamma t = 0.1
    import paper_2411_18341_b200.workloads as wl
    n0 = np.sum(np.abs(wl.cfg1().fields["psi_p"]) ** 2)
    assert abs(np.sum(np.abs(psi) ** 2) / n0 - np.exp(-0.1)) < 1e-3
