"""Writes tests/golden/cfg1_oracle_samples.txt: sampled values of the ORACLE's config-1 result.

Calls only oracle/ and the seeded input generator (no CUDA path).  This is a drift guard for the
oracle, not an independent pin (those are tests/test_oracle_pins.py): a change of the oracle's
arithmetic must come with a regenerated file and a commit message naming the passage of the paper
or the DESIGN.md reading that justifies it.
    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle as orc  # noqa: E402
from paper_2411_18341_b200 import workloads  # noqa: E402


def run_cfg1():
    w = workloads.cfg1()
    o = orc.Oracle(w.nx, w.ny, w.dx, w.dy, orc.make_params(**w.params), model=w.model, V=w.V)
    o.set_field("psi_p", w.fields["psi_p"])
    o.step_rk4(w.n_steps)
    return o.psi_p[0]


SAMPLES = [(0, 0), (32, 32), (31, 40), (5, 60), (63, 63), (17, 3)]

if __name__ == "__main__":
    psi = run_cfg1()
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg1_oracle_samples.txt")
    with open(path, "w") as f:
        f.write("# BASELINE.json config 1 after 1000 RK4 steps, from oracle/ (written by make_golden.py)\n")
        f.write("# j i re im   (C99 hex floats);  last line: sum |psi|^2\n")
        for j, i in SAMPLES:
            f.write(f"{j} {i} {float(psi[j, i].real).hex()} {float(psi[j, i].imag).hex()}\n")
        f.write(f"norm {float(np.sum(np.abs(psi) ** 2)).hex()}\n")
    print(path)
