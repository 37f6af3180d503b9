"""Writes tests/golden/oracle_regression.txt: outputs of the ORACLE (oracle/, nothing else) on a few tiny seeded inputs.

    python tests/golden/make_golden.py

The paper prints no worked numerical example, so there is no value of the paper's to store; what is
stored here is a regression fixture of the oracle itself -- the right-hand side L(q) (Eq. 6-10), the CFL time
step and the state after one 3-stage Runge-Kutta step on inputs of the seeded generator
paper_2305_09163_b200.workloads.random_state (which holds no step of the method) -- so that a later change to the oracle's
arithmetic cannot pass unnoticed (it must come with a regenerated file and a commit message that names the passage or the
DESIGN.md reading behind it).  This script calls only oracle/ and the input generator; no value ever comes from the CUDA path.
Numbers are written as C99 hexadecimal floats (exact).
"""
from __future__ import annotations

import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2305_09163_b200 import workloads as wl  # noqa: E402

CASES = [  # (name, ndim, n, n_fluids, seed, periodic, stretched)
    ("d1_f2_extrap", 1, (12,), 2, 7, False, False),
    ("d2_f2_periodic", 2, (5, 4), 2, 8, True, False),
    ("d3_f2_extrap", 3, (4, 3, 3), 2, 9, False, False),
    ("d3_f3_periodic", 3, (3, 3, 3), 3, 10, True, False),
    ("d3_f2_stretched", 3, (4, 4, 3), 2, 11, False, True),
]
OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_regression.txt")


def compute(case):
    name, ndim, n, nf, seed, periodic, stretched = case
    prob, q = wl.random_state(ndim, n, nf, seed=seed, periodic=periodic, rough=False)
    if stretched:
        prob = wl.with_stretched_grid(prob)
    orc = oracle.Oracle(prob)
    it = prob.interior()
    q0 = q.copy()
    L = orc.rhs(q0)[it]
    dt = orc.cfl_dt(q.copy(), prob.cfl)
    q1 = q.copy()
    orc.rk3_step(q1, dt)
    return prob, L, dt, q1[it]


def main():
    with open(OUT, "w") as f:
        f.write("# written by tests/golden/make_golden.py (oracle only); see its docstring.  Format: a line `case <name> <neq> <cells>`,\n")
        f.write("# a line `dt <hex>`, then neq lines `L <eq> <hex> ...` and neq lines `q1 <eq> <hex> ...` (interior cells, C order z, y, x)\n")
        for case in CASES:
            prob, L, dt, q1 = compute(case)
            f.write(f"case {case[0]} {prob.neq} {L[0].size}\n")
            f.write(f"dt {float(dt).hex()}\n")
            for k in range(prob.neq):
                f.write(f"L {k} " + " ".join(float(v).hex() for v in L[k].ravel()) + "\n")
            for k in range(prob.neq):
                f.write(f"q1 {k} " + " ".join(float(v).hex() for v in q1[k].ravel()) + "\n")
    print(OUT)


if __name__ == "__main__":
    main()
