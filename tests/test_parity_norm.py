"""Evidence for the parity norm of DESIGN.md section 4 (CPU only; `-m "not gpu"`).

north_star asks for "max relative error per conserved variable <= 1e-10 after one RHS".  SURVEY.md 8(c)-D scales row
k by S_k = max |oracle_k|; tests/gpu_util.py additionally floors S_k at K ulp of the flux terms that cancel in that
row (rhs_floors, K = ROUNDOFF_K).  This file shows, with the oracle alone, that the floor is needed and how large it
has to be: the SAME source (oracle/mfc_oracle.c) is built twice -- as the oracle proper (-ffp-contract=off) and with
FMA contraction allowed (what nvcc does to the CUDA path by default; oracle.variant_flags()) -- and the two results,
both correct fp64 evaluations of the same formulas, are compared in both norms.
"""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from gpu_util import RHS_TOL, ROUNDOFF_K, rhs_floors, row_scales
from paper_2305_09163_b200 import workloads as wl


def two_builds(prob, q):
    path, tag = oracle.build_variant()
    strict, other = oracle.Oracle(prob), oracle.Oracle(prob, path)
    qa = q.copy()
    La = strict.rhs(qa)[prob.interior()]
    Lb = other.rhs(q.copy())[prob.interior()]
    floors = rhs_floors(prob, strict, qa)
    d = np.array([np.max(np.abs(La[k] - Lb[k])) for k in range(prob.neq)])
    return d, row_scales(prob, La), row_scales(prob, La, floors), floors, tag


CASES = {
    "cfg1@64": lambda: wl.cfg1(n=64),
    "cfg2@48": lambda: wl.cfg2(n=48),
    "cfg3@64": lambda: wl.cfg3(n=64),
    "random_3d": lambda: wl.random_state(3, (40, 29, 33), 2, seed=7, periodic=False),
    "random_2d_3f": lambda: wl.random_state(2, (130, 45), 3, seed=8),
}


@pytest.mark.parametrize("case", list(CASES))
def test_two_correct_evaluations_agree_in_the_floored_norm(case):
    prob, q = CASES[case]()
    d, S0, S, floors, tag = two_builds(prob, q)
    assert np.any(d > 0.0), "the second build is bit-identical: it demonstrates nothing"
    err = d / S
    print(f"{case} [{tag}]: floored {err}, unfloored {d / S0}, ulp of flux scale {d / (floors * RHS_TOL / ROUNDOFF_K)}")
    assert np.all(err <= RHS_TOL)


@pytest.mark.parametrize("case", ["cfg2@48", "cfg3@64"])
def test_unfloored_norm_rejects_a_correct_evaluation(case):
    """Quiescent bubbles: the volume-fraction RHS is pure cancellation noise away from the shock, so two correct
    evaluations differ by far more than 1e-10 of max |L_alpha| -- the literal norm cannot be met by ANY independent
    fp64 implementation, which is why S_k has a round-off floor."""
    prob, q = CASES[case]()
    d, S0, S, floors, tag = two_builds(prob, q)
    k = prob.neq - 1
    assert d[k] / S0[k] > 10.0 * RHS_TOL
    assert d[k] / S[k] <= RHS_TOL


def test_floor_is_within_an_order_of_magnitude_of_the_demonstrated_round_off():
    """Where the floor binds hardest (cfg1: momentum rows of a uniform-pressure, uniform-velocity advection are pure
    cancellation) the allowed error, K ulp of the flux scale over dx, is at most 10 x what FMA contraction alone produces.
    (The GPU suite, whose kernels also regroup the algebra, reaches 3.8 ulp: tests/test_gpu_parity.py prints it.)"""
    prob, q = CASES["cfg1@64"]()
    d, S0, S, floors, tag = two_builds(prob, q)
    allowed = RHS_TOL * S
    ulps = d / (floors * RHS_TOL / ROUNDOFF_K)          # floors = K eps / tol * flux scale / dx
    assert ulps.max() >= ROUNDOFF_K / 10.0, ulps
    assert np.min(allowed / np.maximum(d, 1e-300)) <= 10.0
