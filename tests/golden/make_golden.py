"""Writes tests/golden/oracle_c1_first16_1000steps.txt from the ORACLE ONLY (never from the CUDA path).

    python tests/golden/make_golden.py

The file freezes what the oracle, as pinned by tests/test_oracle_pins.py, returns for the first 16
particles of BASELINE.json configs[0] after 1 000 steps of 180 d (the parity horizon of
BASELINE.json's north_star).  It is a regression guard on the oracle's arithmetic: a later change
to oracle/glisse_oracle.cpp that moves these numbers must name, in its commit message, the passage
of PAPER.md or the DESIGN.md reading that justifies it.  The paper prints no worked numerical
example, so there is no paper-printed fixture.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2011_03484_b200 import inputs  # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_c1_first16_1000steps.txt")


def compute():
    w = inputs.config(1).subset(16)
    S = oracle.OracleSim.from_workload(w)
    S.advance(1000)
    pos, vel, flag, rstep = S.read()
    q, qd = S.read_planets()
    return pos, vel, flag, rstep, q, qd


if __name__ == "__main__":
    pos, vel, flag, rstep, q, qd = compute()
    with open(OUT, "w") as f:
        f.write("# oracle, BASELINE.json configs[0] first 16 particles, 1000 steps of 180 d; written by make_golden.py\n")
        f.write("# particle rows: x y z vx vy vz flag removal_step ; then planet rows: x y z vx vy vz\n")
        for i in range(pos.shape[1]):
            f.write(" ".join(float(t).hex() for t in (*pos[:, i], *vel[:, i])) + f" {flag[i]} {rstep[i]}\n")
        for j in range(q.shape[0]):
            f.write(" ".join(float(t).hex() for t in (*q[j], *qd[j])) + "\n")
    print("wrote", OUT)
