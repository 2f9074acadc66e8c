"""Writes tests/golden/oracle_residuals.txt from the CPU oracle ONLY (never the CUDA path).

The paper prints no worked numerical example (no value of u, dt, eta or ||H||), so these are not
paper values: they are regression anchors for the oracle itself ("parity unpinned" outputs, see
oracle/hr_oracle.h), regenerated with `python tests/golden/make_golden.py`.
Columns: case steps residual_mode0 residual_mode1 max|u|
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import hr_workloads as W  # noqa: E402
from oracle.hr_oracle import Oracle  # noqa: E402

CASES = [("config0", lambda: W.config(0), (0, 50, 200)),
         ("config1_quarter", lambda: dict(W.config(1, scale=0.25), eta=30.0), (0, 100, 400))]


def rows():
    for name, make, marks in CASES:
        o = Oracle(make())
        u, v = np.zeros(o.ntot), np.zeros(o.ntot)
        done = 0
        for m in marks:
            u, v = o.step(u, v, m - done)
            done = m
            yield name, m, o.residual(u, 0), o.residual(u, 1), float(np.abs(u).max())


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_residuals.txt")
    with open(out, "w") as f:
        f.write("# written by tests/golden/make_golden.py from oracle/ only; see its docstring\n")
        for r in rows():
            f.write("%s %d %.17e %.17e %.17e\n" % r)
    print(open(out).read())
