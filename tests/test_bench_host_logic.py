"""Host-side arithmetic of bench.py: the algorithmic work per cell that the roofline fractions are quoted on
 and the DRAM traffic read from the committed ncu capture.  CPU only."""
from __future__ import annotations

import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402
from paper_2305_09163_b200 import workloads as wl  # noqa: E402


def test_algorithmic_work_per_cell_matches_the_survey_counts():
    prob3, _ = wl.cfg3(n=8)
    flops, nbytes = bench.rhs_algorithmic(prob3)
    # D = 3, NEQ = 7: 3 x (7 x 80 WENO + 102 HLLC + 3 x 7 difference) + 25 cons->prim + 4 x 7 RK combine
    assert flops == 3 * (7 * 80 + 102 + 21) + 25 + 28 == 2102
    # q_s read + result written + q_n read in two of the three stages, 7 doubles each
    assert nbytes == pytest.approx(7 * 8 * (2 + 2 / 3))
    prob4, _ = wl.cfg4(n=8)
    flops4, nbytes4 = bench.rhs_algorithmic(prob4)
    assert flops4 == 3 * (9 * 80 + 116 + 27) + 25 + 36 and nbytes4 == pytest.approx(9 * 8 * (2 + 2 / 3))


def test_committed_dram_traffic_is_at_least_the_compulsory_bytes():
    prob, _ = wl.cfg3(n=8)
    _, nbytes = bench.rhs_algorithmic(prob)
    t, src = bench.ncu_traffic("cfg3", "rhs_fused")
    assert t is not None and "recorded" in src and "commit" in src     # provenance: which commit the capture belongs to
    cells = 256 ** 3
    assert 1.0 <= t / (nbytes * cells) < 1.3          # re-reads stay small: each cell is read once (plus halos)
    assert bench.ncu_traffic("cfg3", "no_such_kernel") == (None, None) and bench.ncu_traffic("", "rhs_fused") == (None, None)


def test_metric_and_unit_are_the_baseline_ones():
    import json
    with open(os.path.join(ROOT, "BASELINE.json")) as f:
        base = json.load(f)
    assert "grind time" in base["metric"] and "ns/(cell" in base["metric"]
    assert bench.METRIC == "grind_time_ns_per_cell_eqn_rhs" and bench.UNIT == "ns/(cell*eqn*RHS)" and bench.RHS_PER_STEP == 3
