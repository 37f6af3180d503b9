"""The oracle against its stored regression fixture (tests/golden/oracle_regression.txt, written by
tests/golden/make_golden.py from the oracle alone), and the CUDA path against the same stored values.

The paper prints no worked example, so the fixture pins the oracle to ITSELF IN TIME, not to the paper: a change to the
oracle's arithmetic shows up here and has to be justified (commit message naming the passage or DESIGN.md reading) together
with a regenerated file.  What pins the oracle to the paper and the mathematics is tests/test_oracle_pins.py.
"""
from __future__ import annotations

import importlib.util
import os

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
mg = importlib.util.module_from_spec(spec)
spec.loader.exec_module(mg)


def read_golden():
    out, cur = {}, None
    with open(mg.OUT) as f:
        for line in f:
            if line.startswith("#"):
                continue
            t = line.split()
            if t[0] == "case":
                cur = {"neq": int(t[2]), "cells": int(t[3]), "L": {}, "q1": {}}
                out[t[1]] = cur
            elif t[0] == "dt":
                cur["dt"] = float.fromhex(t[1])
            else:
                cur[t[0]][int(t[1])] = np.array([float.fromhex(v) for v in t[2:]])
    return out


GOLD = read_golden()


@pytest.mark.parametrize("case", mg.CASES, ids=[c[0] for c in mg.CASES])
def test_oracle_reproduces_its_fixture(case):
    prob, L, dt, q1 = mg.compute(case)
    g = GOLD[case[0]]
    assert g["neq"] == prob.neq and g["cells"] == L[0].size
    assert abs(dt - g["dt"]) <= 1e-15 * g["dt"]
    for k in range(prob.neq):
        for got, ref in ((L[k].ravel(), g["L"][k]), (q1[k].ravel(), g["q1"][k])):
            # the same source under -ffp-contract=off: equal to the last bits (a few ulp of the row's scale are allowed
            # for another compiler version's sqrt / division sequences)
            assert np.max(np.abs(got - ref)) <= 1e-14 * max(np.max(np.abs(ref)), 1e-300)


@pytest.mark.gpu
@pytest.mark.parametrize("case", mg.CASES, ids=[c[0] for c in mg.CASES])
def test_cuda_path_against_the_stored_fixture(case):
    """mfc_rhs, mfc_cfl_dt and mfc_rk3_step through the C ABI against the STORED oracle values (no oracle call here)."""
    from gpu_util import Gpu
    from paper_2305_09163_b200 import workloads as wl

    name, ndim, n, nf, seed, periodic, stretched = case
    prob, q = wl.random_state(ndim, n, nf, seed=seed, periodic=periodic, rough=False)
    if stretched:
        prob = wl.with_stretched_grid(prob)
    g = GOLD[name]
    it = prob.interior()
    with Gpu(prob) as gpu:
        L = gpu.rhs(q)[it]
        dt = gpu.cfl_dt(q)
        q1 = gpu.rk3(q, [g["dt"]])[it]
    assert abs(dt - g["dt"]) <= 1e-13 * g["dt"]
    nfl, D = prob.nf, prob.ndim
    for label, got, ref, tol in (("L", L, g["L"], 1e-10), ("q1", q1, g["q1"], 1e-12)):
        S = np.array([np.max(np.abs(ref[k])) for k in range(prob.neq)])
        S[nfl:nfl + D] = S[nfl:nfl + D].max()                      # the momentum rows share one scale
        if label == "L":
            S = np.maximum(S, 1e-6 * S.max())                      # rows that cancel to round-off (tiny smooth inputs)
        for k in range(prob.neq):
            assert np.max(np.abs(got[k].ravel() - ref[k])) <= tol * S[k], (label, k)
