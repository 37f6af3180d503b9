"""GPU-vs-oracle parity through the C ABI (needs a B200: `-m gpu`).

Bars (BASELINE.json north_star): max relative error per conserved variable <= 1e-10 after one RHS evaluation
and <= 1e-8 after 10 RK3 steps, fp64, in the norm of DESIGN.md "Parity norm".  The cons->prim stage is held to
bit equality.  Inputs are the seeded generators of workloads.py.
"""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from gpu_util import RHS_TOL, Gpu, parity_errors, parity_report, rhs_floors, row_scales
from paper_2305_09163_b200 import binding as B
from paper_2305_09163_b200 import workloads as wl

pytestmark = pytest.mark.gpu

RK_TOL = 1.0e-8
ULP_BACKSTOP = 8.0
TEMPLATE_SET = [(1, 1), (1, 2), (1, 3), (2, 1), (2, 2), (2, 3), (3, 1), (3, 2), (3, 3)]
# several tiles of the fused kernel plus ragged tails: tiles of 32 x 16 (32 x 12 with three fluids, 32 x 8 in 2D)
# cells, z segments of 8 planes
SIZES = {1: (1201,), 2: (301, 45), 3: (67, 29, 41)}


def check_rhs(prob, q, tol=RHS_TOL, **kw):
    orc = oracle.Oracle(prob)
    qo = q.copy()
    ref = orc.rhs(qo)
    with Gpu(prob, **kw) as g:
        got = g.rhs(q)
    err, unfloored, ulps = parity_report(prob, got, ref, rhs_floors(prob, orc, qo))
    # the unfloored error (S_k = max |oracle_k|, no round-off floor) and the error in ulp of the flux terms that cancel
    # are reported beside the asserted one (`pytest -s`, the failure message, and gpurun_out/parity_report.txt)
    fmt = lambda a: np.array2string(a, precision=2, separator=", ")
    msg = f"{prob.name}: RHS error floored {fmt(err)} | unfloored {fmt(unfloored)} | in ulp of flux scale/dx {fmt(ulps)}"
    print(msg)
    _log_report(msg)
    assert np.all(err <= tol), msg
    # backstop under the floored norm: the error in ulp of the flux terms that cancel (the suite's worst case is 3.7, two
    # CPU builds of the oracle differ by 2.2; the floor alone would let 12 pass)
    assert np.all(ulps <= ULP_BACKSTOP), msg
    return err


def _log_report(msg):
    import os
    d = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")
    if os.path.isdir(d):
        with open(os.path.join(d, "parity_report.txt"), "a") as f:
            f.write(msg + "\n")


# ---------------------------------------------------------------------------------------------
# a0 + a1: ghost fill and cons->prim, bit for bit
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ndim,nf", TEMPLATE_SET)
@pytest.mark.parametrize("periodic", [True, False])
def test_prim_array_is_bit_identical(ndim, nf, periodic):
    n = {1: (37,), 2: (19, 11), 3: (9, 7, 5)}[ndim]
    prob, q = wl.random_state(ndim, n, nf, seed=3, periodic=periodic)
    orc = oracle.Oracle(prob)
    qo = q.copy()
    orc.fill_ghosts(qo)
    ref = orc.cons_to_prim(qo)
    with Gpu(prob) as g:
        got = g.prim(q)
    assert np.array_equal(got, ref)


def test_prim_mixed_boundary_kinds():
    prob, q = wl.random_state(3, (8, 6, 5), 2, seed=6, periodic=True)
    prob.bc_lo = (wl.BC_EXTRAP, wl.BC_PERIODIC, wl.BC_EXTRAP)
    prob.bc_hi = (wl.BC_EXTRAP, wl.BC_PERIODIC, wl.BC_EXTRAP)
    orc = oracle.Oracle(prob)
    qo = q.copy()
    orc.fill_ghosts(qo)
    ref = orc.cons_to_prim(qo)
    with Gpu(prob) as g:
        got = g.prim(q)
    assert np.array_equal(got, ref)


@pytest.mark.parametrize("ndim,n,lo,hi", [
    (1, (37,), (wl.BC_EXTRAP,), (wl.BC_EXTRAP,)), (2, (12, 9), (wl.BC_PERIODIC, wl.BC_EXTRAP), (wl.BC_PERIODIC, wl.BC_EXTRAP)),
    (3, (10, 7, 5), (wl.BC_PERIODIC,) * 3, (wl.BC_PERIODIC,) * 3),
    (3, (9, 8, 6), (wl.BC_EXTRAP, wl.BC_PERIODIC, wl.BC_EXTRAP), (wl.BC_EXTRAP, wl.BC_PERIODIC, wl.BC_EXTRAP))])
def test_ghost_cells_of_q_hold_the_boundary_fill_after_rhs(ndim, n, lo, hi):
    """a0 in memory ("ghost cells of q are overwritten by every mfc_rhs"): whatever the ghost
    cells held, after mfc_rhs the whole padded array equals the oracle's ghost fill, corners included, bit for bit."""
    import dataclasses
    prob, q = wl.random_state(ndim, n, 2, seed=8, periodic=True)
    prob = dataclasses.replace(prob, bc_lo=tuple(lo) + (wl.BC_EXTRAP,) * (3 - ndim), bc_hi=tuple(hi) + (wl.BC_EXTRAP,) * (3 - ndim))
    core = q[prob.interior()].copy()
    q[...] = np.random.default_rng(0).normal(size=q.shape)  # garbage in the ghosts
    q[prob.interior()] = core
    ref = q.copy()
    oracle.Oracle(prob).fill_ghosts(ref)
    with Gpu(prob) as g:
        qd = g.to_dev(q)
        out = g.torch.zeros_like(qd)
        B.mfc_rhs(g.ctx, qd.data_ptr(), out.data_ptr(), g.stream)
        g.torch.cuda.synchronize()
        after = qd.cpu().numpy()
    assert np.array_equal(after, ref)


# ---------------------------------------------------------------------------------------------
# a2 + a3: WENO5 face states and HLLC fluxes on one line
# ---------------------------------------------------------------------------------------------
def random_prim_line(prob, n, rng, smooth):
    nf, D = prob.nf, prob.ndim
    x = np.linspace(0, 1, n + 2 * wl.NG)
    rough = (lambda a: a * rng.uniform(-1, 1, size=x.size) + 0.5 * (rng.uniform(size=x.size) < 0.05)) if not smooth else (lambda a: 0.0)
    z = [np.sin(2 * np.pi * (i + 1) * x + rng.uniform(0, 6)) + rough(0.3) for i in range(nf)]
    e = [np.exp(1.5 * zi) for zi in z]
    alpha = [np.clip(ei / sum(e), 1e-6, 1.0) for ei in e]
    if nf > 1:
        alpha[-1] = 1.0 - sum(alpha[:-1])
    else:
        alpha = [np.ones_like(x)]
    rho0 = [1000.0, 1.2, 0.6][:nf]
    w = np.zeros((prob.neq, x.size))
    for i in range(nf):
        w[i] = alpha[i] * rho0[i] * (1 + 0.1 * np.sin(5 * x + i) + rough(0.05))
        if i < nf - 1:
            w[nf + D + 1 + i] = alpha[i]
    for d in range(D):
        w[nf + d] = 400.0 * (np.sin(3 * x + d) + rough(0.5))      # sub- and supersonic in air-rich cells
    w[nf + D] = 1.0e5 * np.exp(np.sin(4 * x) + rough(0.5))
    return w


@pytest.mark.parametrize("ndim,nf", TEMPLATE_SET)
@pytest.mark.parametrize("smooth", [True, False])
def test_line_face_states_and_fluxes(ndim, nf, smooth):
    n = 777
    prob, _ = wl.random_state(ndim, {1: (8,), 2: (8, 8), 3: (8, 8, 8)}[ndim], nf, seed=1)
    orc = oracle.Oracle(prob)
    rng = np.random.default_rng(100 * ndim + nf)
    with Gpu(prob) as g:
        for direction in range(ndim):
            w = random_prim_line(prob, n, rng, smooth)
            rL, rR, rF, ru = orc.line(direction, w)
            gL, gR, gF, gu = g.line(direction, w)
            for e in range(prob.neq):
                s = np.max(np.abs(w[e])) + 1e-300
                # reconstructed values: a few ulp of the local data
                assert np.max(np.abs(gL[e] - rL[e])) <= 1e-13 * s, (direction, e)
                assert np.max(np.abs(gR[e] - rR[e])) <= 1e-13 * s, (direction, e)
            # fluxes: HLLC applied to each side's own face states (rounding differences of the states are
            # amplified by the wave-speed switches only up to continuity)
            for e in range(prob.neq):
                s = np.max(np.abs(rF[e])) + 1e-300
                assert np.max(np.abs(gF[e] - rF[e])) <= 1e-11 * s, (direction, e)
            assert np.max(np.abs(gu - ru)) <= 1e-11 * np.max(np.abs(ru))


@pytest.mark.parametrize("ndim,nf", [(1, 2), (3, 2), (3, 3)])
def test_hllc_kernel_on_identical_inputs(ndim, nf):
    """HLLC alone: feed the GPU Riemann solver the oracle's own face states by making them exact:
    a piecewise-constant line has vL = vR = cell value wherever the stencil is constant."""
    prob, _ = wl.random_state(ndim, {1: (8,), 3: (8, 8, 8)}[ndim], nf, seed=1)
    orc = oracle.Oracle(prob)
    rng = np.random.default_rng(7)
    n = 600
    base = random_prim_line(prob, n // 6 + 1, rng, smooth=False)[:, : n // 6 + 1]
    w = np.repeat(base, 6, axis=1)[:, : n + 2 * wl.NG]          # plateaus of 6 cells
    with Gpu(prob) as g:
        for direction in range(ndim):
            rL, rR, rF, ru = orc.line(direction, w)
            gL, gR, gF, gu = g.line(direction, w)
            for e in range(prob.neq):
                s = np.max(np.abs(rF[e])) + 1e-300
                assert np.max(np.abs(gF[e] - rF[e])) <= 1e-12 * s, (direction, e)


# ---------------------------------------------------------------------------------------------
# a0..a4: one RHS evaluation, every template instantiation, ragged sizes, small marching segments
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ndim,nf", TEMPLATE_SET)
@pytest.mark.parametrize("periodic", [True, False])
def test_rhs_parity_random_states(ndim, nf, periodic):
    prob, q = wl.random_state(ndim, SIZES[ndim], nf, seed=10 * ndim + nf, periodic=periodic)
    check_rhs(prob, q, march_segment=8)


MIXED_BCS = [
    (2, (wl.BC_PERIODIC, wl.BC_EXTRAP), (wl.BC_PERIODIC, wl.BC_EXTRAP)),
    (2, (wl.BC_EXTRAP, wl.BC_PERIODIC), (wl.BC_EXTRAP, wl.BC_PERIODIC)),
    (3, (wl.BC_EXTRAP, wl.BC_PERIODIC, wl.BC_EXTRAP), (wl.BC_EXTRAP, wl.BC_PERIODIC, wl.BC_EXTRAP)),
    (3, (wl.BC_PERIODIC, wl.BC_EXTRAP, wl.BC_PERIODIC), (wl.BC_PERIODIC, wl.BC_EXTRAP, wl.BC_PERIODIC)),
    (3, (wl.BC_PERIODIC, wl.BC_PERIODIC, wl.BC_EXTRAP), (wl.BC_PERIODIC, wl.BC_PERIODIC, wl.BC_EXTRAP)),
]


@pytest.mark.parametrize("ndim,lo,hi", MIXED_BCS)
@pytest.mark.parametrize("even", [False, True])
def test_rhs_and_rk3_parity_mixed_boundary_kinds_on_the_fused_path(ndim, lo, hi, even):
    """Periodic in some dimensions, extrapolation in others, through mfc_rhs / mfc_rk3_step (the fused kernels' own
    ghost handling), at sizes with odd and even padded extents (the two staging paths of the 3D kernel)."""
    import dataclasses
    n = {2: (301, 45), 3: (67, 29, 41)}[ndim] if not even else {2: (300, 46), 3: (66, 30, 40)}[ndim]
    prob, q = wl.random_state(ndim, n, 2, seed=70 + ndim, periodic=True)
    prob = dataclasses.replace(prob, bc_lo=tuple(lo) + (wl.BC_EXTRAP,) * (3 - ndim), bc_hi=tuple(hi) + (wl.BC_EXTRAP,) * (3 - ndim))
    check_rhs(prob, q, march_segment=8)
    prob_s, q_s = wl.random_state(ndim, {2: (130, 45), 3: (40, 29, 33)}[ndim] if not even else {2: (130, 44), 3: (40, 30, 32)}[ndim],
                                  2, seed=80 + ndim, periodic=True, rough=False)
    prob_s = dataclasses.replace(prob_s, bc_lo=prob.bc_lo, bc_hi=prob.bc_hi)
    check_rk(prob_s, q_s, march_segment=8)


# ---------------------------------------------------------------------------------------------
# the two staging paths of the 3D kernel (TMA boxes / per-thread cp.async): every 3D instantiation, forced
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("nf", [1, 2, 3])
@pytest.mark.parametrize("periodic", [True, False])
@pytest.mark.parametrize("order", [5, 3, 1])
def test_rhs_parity_tma_staging_and_bitwise_agreement_with_cp_async(nf, periodic, order):
    """At an even padded extent both staging paths apply: each is held to the oracle, and they give the same bits
    (same arithmetic on the same staged values).  Ragged tiles in x and y, several z segments."""
    import dataclasses
    prob, q = wl.random_state(3, (70, 29, 41), nf, seed=300 + nf, periodic=periodic)
    prob = dataclasses.replace(prob, weno_order=order)
    check_rhs(prob, q, march_segment=8, staging=B.MFC_STAGING_TMA)
    with Gpu(prob, march_segment=8, staging=B.MFC_STAGING_TMA) as g1, Gpu(prob, march_segment=8, staging=B.MFC_STAGING_CPASYNC) as g2:
        it = prob.interior()
        assert np.array_equal(g1.rhs(q)[it], g2.rhs(q)[it])
        orc = oracle.Oracle(prob)
        dts = [0.5 * orc.cfl_dt(q.copy(), prob.cfl)] * 3
        assert np.array_equal(g1.rk3(q, dts)[it], g2.rk3(q, dts)[it])


def test_tma_staging_refuses_an_odd_padded_extent_and_auto_falls_back():
    prob, q = wl.random_state(3, (33, 17, 9), 2, seed=5, periodic=True, rough=False)
    with Gpu(prob, staging=B.MFC_STAGING_TMA) as g:
        with pytest.raises(B.MfcError):
            g.rhs(q)
    check_rhs(prob, q, staging=B.MFC_STAGING_AUTO)


# ---------------------------------------------------------------------------------------------
# the 3D kernel with specialised Z warps (staging = 3; what AUTO runs for two fluids on a uniform grid
# with an even padded extent): forced, against the oracle and against the one-loop kernel
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("periodic", [True, False])
@pytest.mark.parametrize("order", [5, 3, 1])
@pytest.mark.parametrize("n,seg", [((70, 29, 41), 8), ((32, 12, 9), 0), ((96, 50, 7), 3), ((34, 13, 64), 0)])
def test_rhs_parity_split_kernel(periodic, order, n, seg):
    """Ragged tiles in x and y (rows past the domain in the last tile row), one to many z segments, segments of a single
    plane; every reconstruction order.  The split kernel sums the three directions in another order than the one-loop
    kernel, so the two are compared at round-off, not bitwise."""
    import dataclasses
    prob, q = wl.random_state(3, n, 2, seed=400 + order, periodic=periodic)
    prob = dataclasses.replace(prob, weno_order=order)
    check_rhs(prob, q, march_segment=seg, staging=B.MFC_STAGING_ROLES)
    with Gpu(prob, march_segment=seg, staging=B.MFC_STAGING_ROLES) as g1, Gpu(prob, march_segment=seg, staging=B.MFC_STAGING_TMA) as g2:
        it = prob.interior()
        a, b = g1.rhs(q)[it], g2.rhs(q)[it]
        scale = np.max(np.abs(b), axis=(1, 2, 3), keepdims=True) + 1e-300
        assert np.max(np.abs(a - b) / scale) <= 1e-12


@pytest.mark.parametrize("n", [(4, 3, 3), (4, 4, 4), (6, 3, 5), (34, 3, 3), (4, 13, 3), (4, 3, 14), (32, 12, 3)])
@pytest.mark.parametrize("periodic", [True, False])
def test_rhs_parity_split_kernel_smallest_grids(n, periodic):
    """Degenerate sizes: fewer cells than ghost layers + 1 per dimension, one tile with most of its rows and lanes past the
    domain, segments shorter than the three planes the z direction runs ahead."""
    prob, q = wl.random_state(3, n, 2, seed=440, periodic=periodic, rough=False)
    check_rhs(prob, q, staging=B.MFC_STAGING_ROLES)
    check_rhs(prob, q, march_segment=1, staging=B.MFC_STAGING_ROLES)


@pytest.mark.parametrize("nf", [1, 3])
@pytest.mark.parametrize("periodic", [True, False])
def test_rhs_and_rk3_parity_split_kernel_one_and_three_fluids(nf, periodic):
    prob, q = wl.random_state(3, (70, 29, 41), nf, seed=420 + nf, periodic=periodic)
    check_rhs(prob, q, march_segment=8, staging=B.MFC_STAGING_ROLES)
    prob, q = wl.random_state(3, (40, 30, 33), nf, seed=430 + nf, periodic=periodic, rough=False)
    check_rk(prob, q, march_segment=8, staging=B.MFC_STAGING_ROLES)


@pytest.mark.parametrize("rough", [False, True])
@pytest.mark.parametrize("kapila", [False, True])
def test_rk3_parity_split_kernel(rough, kapila):
    import dataclasses
    prob, q = wl.random_state(3, (40, 30, 33), 2, seed=410, periodic=not rough, rough=rough)
    prob = dataclasses.replace(prob, kapila=kapila)
    check_rk(prob, q, march_segment=8, staging=B.MFC_STAGING_ROLES)


def test_split_kernel_is_reproducible_and_refuses_what_it_does_not_cover():
    """Run-to-run bitwise reproducibility (a race between the warp kinds would show here), and a forced choice fails for an
    odd padded extent while AUTO falls back to a kernel that applies."""
    prob, q = wl.random_state(3, (64, 24, 40), 2, seed=411, periodic=False)
    with Gpu(prob, staging=B.MFC_STAGING_ROLES) as g:
        ref = g.rhs(q)
        for _ in range(5):
            assert np.array_equal(g.rhs(q), ref, equal_nan=True)
    p3, q3 = wl.random_state(3, (33, 17, 9), 2, seed=5, periodic=True, rough=False)
    with Gpu(p3, staging=B.MFC_STAGING_ROLES) as g:
        with pytest.raises(B.MfcError):
            g.rhs(q3)
    check_rhs(p3, q3, staging=B.MFC_STAGING_AUTO)


@pytest.mark.parametrize("seg", [1, 5, 32, 1000])
@pytest.mark.parametrize("n0", [40, 41])
def test_rhs_is_independent_of_the_marching_segment(seg, n0):
    prob, q = wl.random_state(3, (n0, 33, 37), 2, seed=77, periodic=False)
    with Gpu(prob, march_segment=7) as g:
        ref = g.rhs(q)
    with Gpu(prob, march_segment=seg) as g:
        got = g.rhs(q)
    it = prob.interior()
    assert np.array_equal(got[it], ref[it])


@pytest.mark.parametrize("ndim,n", [(1, (3,)), (2, (3, 3)), (3, (3, 3, 3)), (3, (3, 300, 4)), (2, (255, 3)), (1, (32,)), (1, (33,)), (1, (64,)),
                                    (2, (64, 16)), (2, (65, 17)), (3, (32, 16, 8)), (3, (33, 17, 9)), (3, (31, 15, 3))])
def test_rhs_parity_smallest_and_tile_edge_sizes(ndim, n):
    prob, q = wl.random_state(ndim, n, 2, seed=5, periodic=True, rough=False)
    check_rhs(prob, q)


@pytest.mark.parametrize("ndim,nf,periodic", [(1, 2, False), (2, 2, True), (3, 2, False), (3, 3, True)])
def test_uniform_state_has_exactly_zero_rhs_on_gpu(ndim, nf, periodic):
    prob, q = wl.random_state(ndim, SIZES[ndim], nf, seed=2, periodic=periodic)
    it = prob.interior()
    q[it] = q[it][:, :1, :1, :1]                 # one admissible cell everywhere
    with Gpu(prob, march_segment=8) as g:
        got = g.rhs(q)
    assert np.all(got[it] == 0.0)


# Lower-order reconstructions: same parity bars with opts.weno_order = 3, 1
@pytest.mark.parametrize("order", [1, 3])
@pytest.mark.parametrize("ndim,nf,periodic", [(1, 2, False), (2, 2, True), (2, 1, False), (3, 2, False), (3, 3, True), (3, 1, True)])
def test_rhs_parity_lower_order_reconstruction(order, ndim, nf, periodic):
    import dataclasses
    prob, q = wl.random_state(ndim, SIZES[ndim], nf, seed=50 + 3 * ndim + nf, periodic=periodic)
    prob = dataclasses.replace(prob, weno_order=order)
    check_rhs(prob, q, march_segment=8)
    with Gpu(prob) as g1, Gpu(dataclasses.replace(prob, weno_order=5)) as g5:       # the option is really on
        it = prob.interior()
        assert not np.allclose(g1.rhs(q)[it], g5.rhs(q)[it], rtol=1e-6)


@pytest.mark.parametrize("order", [1, 3])
@pytest.mark.parametrize("rough", [False, True])
def test_rk3_parity_lower_order_reconstruction(order, rough):
    import dataclasses
    prob, q = wl.random_state(3, (40, 29, 33), 2, seed=92, periodic=True, rough=rough)
    check_rk(dataclasses.replace(prob, weno_order=order), q, march_segment=8)


@pytest.mark.parametrize("order", [1, 3])
def test_line_states_lower_order_reconstruction(order):
    import dataclasses
    prob, _ = wl.random_state(2, (8, 8), 2, seed=1)
    prob = dataclasses.replace(prob, weno_order=order)
    orc = oracle.Oracle(prob)
    rng = np.random.default_rng(order)
    w = random_prim_line(prob, 333, rng, False)
    rL, rR, rF, ru = orc.line(1, w)
    with Gpu(prob) as g:
        gL, gR, gF, gu = g.line(1, w)
    for e in range(prob.neq):
        s = np.max(np.abs(w[e])) + 1e-300
        assert np.max(np.abs(gL[e] - rL[e])) <= 1e-13 * s and np.max(np.abs(gR[e] - rR[e])) <= 1e-13 * s
        assert np.max(np.abs(gF[e] - rF[e])) <= 1e-11 * (np.max(np.abs(rF[e])) + 1e-300)
    if order == 1:                                                  # piecewise constant: the states are the cell values
        assert np.array_equal(gL, w[:, 2:-2]) and np.array_equal(gR, w[:, 2:-2])


# Kapila source: same parity bar with opts.kapila on
@pytest.mark.parametrize("ndim", [1, 2, 3])
@pytest.mark.parametrize("periodic", [True, False])
def test_rhs_parity_kapila_source(ndim, periodic):
    import dataclasses
    prob, q = wl.random_state(ndim, SIZES[ndim], 2, seed=40 + ndim, periodic=periodic)
    prob = dataclasses.replace(prob, kapila=True)
    check_rhs(prob, q, march_segment=8)
    # the source is really on: the alpha row differs from the Allaire one
    with Gpu(prob) as g1, Gpu(dataclasses.replace(prob, kapila=False)) as g0:
        it = prob.interior()
        a1, a0 = g1.rhs(q)[it], g0.rhs(q)[it]
    assert np.array_equal(a1[:-1], a0[:-1]) and not np.allclose(a1[-1], a0[-1], rtol=1e-6)


def test_rhs_parity_cfg0():
    prob, q = wl.cfg0()
    check_rhs(prob, q)


def test_rhs_parity_cfg1():
    prob, q = wl.cfg1()
    check_rhs(prob, q)


def test_rhs_parity_cfg2():
    prob, q = wl.cfg2()
    check_rhs(prob, q)


def test_rhs_parity_cfg4_reduced():
    prob, q = wl.cfg4(n=96)
    check_rhs(prob, q)


# ---------------------------------------------------------------------------------------------
# Non-uniform Cartesian spacing (Listing 1, Eq. 15): same bars on stretched grids
# ---------------------------------------------------------------------------------------------
NU_CASES = [(1, 1, (1201,)), (1, 2, (600,)), (2, 2, (300, 45)), (2, 3, (131, 46)), (3, 1, (66, 29, 41)), (3, 2, (67, 29, 41)),
            (3, 2, (70, 30, 40)), (3, 3, (40, 29, 33))]


@pytest.mark.parametrize("ndim,nf,n", NU_CASES)
@pytest.mark.parametrize("periodic", [True, False])
def test_rhs_parity_stretched_grid(ndim, nf, n, periodic):
    prob, q = wl.random_state(ndim, n, nf, seed=400 + 10 * ndim + nf, periodic=periodic)
    prob = wl.with_stretched_grid(prob)
    check_rhs(prob, q, march_segment=8)
    with Gpu(prob) as g1, Gpu(__import__("dataclasses").replace(prob, edges=None)) as g0:     # the grid is really in use
        it = prob.interior()
        assert not np.allclose(g1.rhs(q)[it], g0.rhs(q)[it], rtol=1e-3)


@pytest.mark.parametrize("staging", [B.MFC_STAGING_TMA, B.MFC_STAGING_CPASYNC, B.MFC_STAGING_ROLES])
def test_rhs_parity_stretched_grid_both_staging_paths(staging):
    prob, q = wl.random_state(3, (70, 29, 41), 2, seed=433, periodic=False)
    check_rhs(wl.with_stretched_grid(prob), q, march_segment=8, staging=staging)


@pytest.mark.parametrize("dims", [(0,), (1,), (2,), (0, 2)])
def test_rhs_parity_grid_stretched_in_some_dimensions_only(dims):
    prob, q = wl.random_state(3, (40, 29, 33), 2, seed=440 + len(dims) + dims[0], periodic=True)
    check_rhs(wl.with_stretched_grid(prob, dims=dims), q, march_segment=8)


def test_uniform_edges_reproduce_the_uniform_kernel_to_round_off():
    import dataclasses
    prob, q = wl.random_state(3, (40, 29, 33), 2, seed=450, periodic=False)
    pe = dataclasses.replace(prob, edges=tuple(np.linspace(prob.lo[d], prob.hi[d], prob.n[d] + 1) for d in range(3)))
    it = prob.interior()
    with Gpu(prob) as g0, Gpu(pe) as g1:
        a, b = g0.rhs(q)[it], g1.rhs(q)[it]
    for k in range(prob.neq):
        assert np.max(np.abs(a[k] - b[k])) <= 1e-11 * np.max(np.abs(a[k]))


@pytest.mark.parametrize("ndim,nf,n", [(1, 2, (600,)), (2, 2, (130, 45)), (3, 2, (40, 29, 33)), (3, 3, (40, 30, 33))])
@pytest.mark.parametrize("rough", [False, True])
def test_rk3_parity_stretched_grid(ndim, nf, n, rough):
    prob, q = wl.random_state(ndim, n, nf, seed=460 + ndim + nf, periodic=(nf != 2), rough=rough)
    check_rk(wl.with_stretched_grid(prob), q, march_segment=8)


def test_rhs_and_rk3_parity_cfg2_stretched():
    """The shock-bubble workload on the Eq. 15 grid (same per-cell data on stretched cells), default launch configuration."""
    prob, q = wl.cfg2(n=64)
    prob = wl.with_stretched_grid(prob)
    check_rhs(prob, q)
    check_rk(prob, q)


def test_cfl_dt_parity_stretched_grid():
    for ndim, n in [(1, (301,)), (2, (65, 33)), (3, (40, 29, 33))]:
        prob, q = wl.random_state(ndim, n, 2, seed=470 + ndim, periodic=True)
        prob = wl.with_stretched_grid(prob)
        ref = oracle.Oracle(prob).cfl_dt(q, prob.cfl)
        with Gpu(prob) as g:
            got = g.cfl_dt(q)
        assert abs(got - ref) <= 1e-13 * ref


def test_line_states_and_fluxes_stretched_grid():
    n = 777
    prob, _ = wl.random_state(2, (8, n), 2, seed=1)
    prob = wl.with_stretched_grid(prob)
    orc = oracle.Oracle(prob)
    w = random_prim_line(prob, n, np.random.default_rng(480), False)
    rL, rR, rF, ru = orc.line(1, w)
    with Gpu(prob) as g:
        gL, gR, gF, gu = g.line(1, w)
        with pytest.raises(B.MfcError):          # a line of another length has no coefficient table
            g.line(0, w)
    for e in range(prob.neq):
        s = np.max(np.abs(w[e])) + 1e-300
        assert np.max(np.abs(gL[e] - rL[e])) <= 1e-13 * s and np.max(np.abs(gR[e] - rR[e])) <= 1e-13 * s
        assert np.max(np.abs(gF[e] - rF[e])) <= 1e-11 * (np.max(np.abs(rF[e])) + 1e-300)


def test_nonuniform_grid_needs_weno5_and_increasing_edges():
    import dataclasses
    prob, q = wl.random_state(2, (20, 12), 2, seed=1)
    ps = wl.with_stretched_grid(prob)
    with pytest.raises(B.MfcError) as ei:
        Gpu(dataclasses.replace(ps, weno_order=3))
    assert ei.value.code == B.MFC_EUNSUPPORTED
    bad = list(ps.edges)
    bad[0] = np.array(bad[0])
    bad[0][5] = bad[0][3]
    with pytest.raises(B.MfcError) as ei:
        Gpu(dataclasses.replace(ps, edges=tuple(bad)))
    assert ei.value.code == B.MFC_EINVAL


# ---------------------------------------------------------------------------------------------
# full sizes in the launch configuration bench.py times: sampled sub-boxes the oracle can compute
# (L at a cell depends on the 6 axis neighbours up to distance 3 only) plus size-independent properties
# ---------------------------------------------------------------------------------------------
def subbox_reference(prob, q_full, lo, b):
    """oracle L on the b^3 cells starting at interior index lo, from a (b+6)^3 cut-out of q_full."""
    D = prob.ndim
    idx = [np.arange(lo[d] - wl.NG, lo[d] + b + wl.NG) % prob.n[d] + wl.NG for d in range(D)]   # wrap: periodic cut-outs
    cut = q_full[np.ix_(np.arange(prob.neq), idx[2], idx[1], idx[0])]
    edges = None
    if prob.edges is not None:
        # stretched grid: the cut-out keeps its own cell edges (boxes must then stay clear of the boundaries: no wrap)
        assert all(lo[d] >= wl.NG and lo[d] + b + wl.NG <= prob.n[d] for d in range(D))
        edges = tuple(np.asarray(prob.edges[d])[lo[d] - wl.NG:lo[d] + b + wl.NG + 1].copy() for d in range(D))
    sub = wl.Problem("sub", D, (b + 6,) * 3, (0.0,) * 3, tuple((b + 6) * prob.dx[d] for d in range(3)), prob.fluids,
                     (wl.BC_EXTRAP,) * 3, (wl.BC_EXTRAP,) * 3, weno_eps=prob.weno_eps, edges=edges)
    qs = np.zeros(sub.shape())
    qs[sub.interior()] = cut
    L = oracle.Oracle(sub).rhs(qs)
    return L[sub.interior()][:, wl.NG:-wl.NG, wl.NG:-wl.NG, wl.NG:-wl.NG]


def check_full_size_sampled(prob, q, boxes, b=10):
    it = prob.interior()
    with Gpu(prob) as g:
        got = g.rhs(q)[it]
        # property: conservative rows of a periodic domain sum to round-off of their magnitude
        if all(k == wl.BC_PERIODIC for k in prob.bc_lo[:prob.ndim]):
            for k in range(prob.nf + prob.ndim + 1):
                assert abs(got[k].sum()) <= 1e-9 * np.abs(got[k]).sum() + 1e-300
    assert np.all(np.isfinite(got))
    # scales from the GPU field (the oracle cannot produce the full-size one in seconds), floored like row_scales
    S = row_scales(prob, got, rhs_floors(prob, oracle.Oracle(prob), np.ascontiguousarray(q)))
    # with interior ghosts wrapped the cut-out is only valid where the real array is periodic or away from walls
    for lo in boxes:
        ref = subbox_reference(prob, q, lo, b)
        ix = [np.arange(lo[d], lo[d] + b) % prob.n[d] for d in range(3)]          # wraps like the cut-out
        blk = got[np.ix_(np.arange(prob.neq), ix[2], ix[1], ix[0])]
        for k in range(prob.neq):
            if S[k] == 0.0:
                assert np.all(blk[k] == 0.0)
                continue
            err = np.max(np.abs(blk[k] - ref[k])) / S[k]
            assert err <= RHS_TOL, (lo, k, err)


def test_rhs_full_size_cfg3_sampled():
    prob, q = wl.cfg3()
    rng = np.random.default_rng(0)
    boxes = [tuple(int(v) for v in rng.integers(3, 256 - 13, size=3)) for _ in range(12)]
    boxes += [(3, 100, 200), (8, 30, 60), (120, 243, 3), (243, 243, 243)]     # pressure-pulse slab, far corners
    check_full_size_sampled(prob, q, boxes)


def test_rhs_full_size_cfg4_sampled():
    prob, q = wl.cfg4()
    rng = np.random.default_rng(1)
    boxes = [tuple(int(v) for v in rng.integers(0, 384, size=3)) for _ in range(10)]
    boxes += [(0, 0, 0), (379, 379, 379), (380, 5, 190)]                      # wrap around the periodic faces
    check_full_size_sampled(prob, q, boxes)


def test_rhs_full_size_cfg3_stretched_sampled():
    """The benchmarked stretched configuration (bench.py extra_configs: cfg3 on the Eq. 15 grid, 256^3, default launch
    configuration) against the oracle on sampled boxes, the strongly stretched region and the finest cells included."""
    prob, q = wl.cfg3()
    prob = wl.with_stretched_grid(prob)
    rng = np.random.default_rng(5)
    boxes = [tuple(int(v) for v in rng.integers(3, 256 - 13, size=3)) for _ in range(10)]
    boxes += [(3, 3, 3), (243, 243, 243), (123, 123, 123), (3, 123, 243)]
    check_full_size_sampled(prob, q, boxes)


# ---------------------------------------------------------------------------------------------
# a5: 10 RK3 steps, same dt sequence on both sides (taken from the oracle's CFL)
# ---------------------------------------------------------------------------------------------
def check_rk(prob, q, steps=10, **kw):
    orc = oracle.Oracle(prob)
    qo = q.copy()
    dts = []
    for _ in range(steps):
        dt = orc.cfl_dt(qo, prob.cfl)
        dts.append(dt)
        orc.rk3_step(qo, dt)
    with Gpu(prob, **kw) as g:
        got = g.rk3(q, dts)
    err = parity_errors(prob, got, qo)
    assert np.all(err <= RK_TOL), f"{prob.name}: per-equation error after {steps} RK3 steps {err}"
    return err


@pytest.mark.parametrize("ndim,nf", TEMPLATE_SET)
@pytest.mark.parametrize("rough", [False, True])
def test_rk3_parity_random_states(ndim, nf, rough):
    """rough = True: jumps, spikes and cell noise; within a few steps the unlimited WENO reconstruction (no positivity fix,
    reading B19) overshoots to face states with negative partial densities and pressures, which both sides must carry
    through the Riemann solver in the same way (this is what caught c = n rsqrt(..) vs sqrt(n / ..) for n, rho < 0)."""
    n = {1: (600,), 2: (130, 45), 3: (40, 29, 33)}[ndim]
    prob, q = wl.random_state(ndim, n, nf, seed=20 * ndim + nf, periodic=(nf != 2), rough=rough)
    check_rk(prob, q, march_segment=8)


@pytest.mark.parametrize("rough", [False, True])
def test_rk3_parity_kapila_source(rough):
    import dataclasses
    prob, q = wl.random_state(3, (40, 29, 33), 2, seed=91, periodic=False, rough=rough)
    check_rk(dataclasses.replace(prob, kapila=True), q, march_segment=8)


def test_rk3_parity_cfg0():
    prob, q = wl.cfg0()
    check_rk(prob, q)


def test_rk3_parity_cfg1():
    prob, q = wl.cfg1()
    check_rk(prob, q)


def test_rk3_parity_cfg2():
    prob, q = wl.cfg2()
    check_rk(prob, q)


def test_rk3_parity_cfg3_reduced():
    prob, q = wl.cfg3(n=96)
    check_rk(prob, q)


def test_rk3_parity_cfg4_reduced():
    prob, q = wl.cfg4(n=64)
    check_rk(prob, q)


def test_rk3_parity_cfg4_half_size():
    """cfg4 at 192^3 (three fluids; 16 x 16 tiles x several z segments, the launch shape of the 384^3 the bench times, not
    the two tile rows of the 64^3 case above) for the 10 steps north_star names.  192^3 rather than 384^3: the oracle
    needs about 2.5 s per step here against 20 s and 21 GB of host memory at full size."""
    prob, q = wl.cfg4(n=192)
    check_rk(prob, q)


def test_rhs_and_rk3_parity_kapila_on_a_stretched_grid():
    import dataclasses
    prob, q = wl.random_state(3, (40, 29, 33), 2, seed=92, periodic=False)
    prob = dataclasses.replace(wl.with_stretched_grid(prob), kapila=True)
    check_rhs(prob, q)
    check_rk(prob, q)


def test_results_are_bitwise_reproducible_from_run_to_run():
    """A data race between the warps of a block (exchange buffers, ring slots, staged plane) would show up as run-to-run
    differences: the same five steps, three times, must give the same bits (compute-sanitizer is not available on the
    GPU pool, so this and the parity tests are the race checks)."""
    prob, q = wl.random_state(3, (97, 50, 41), 2, seed=123, periodic=False)
    orc = oracle.Oracle(prob)
    dts = [0.5 * orc.cfl_dt(q.copy(), prob.cfl)] * 5
    runs = []
    for _ in range(3):
        with Gpu(prob) as g:
            runs.append(g.rk3(q, dts))
    assert np.array_equal(runs[0], runs[1]) and np.array_equal(runs[0], runs[2])
    assert np.all(np.isfinite(runs[0][prob.interior()]))


def test_rk3_full_size_cfg3_whole_state():
    """The headline workload at its full size, in the launch configuration bench.py times (default segment heuristic):
    the 10 steps north_star names (CFL + 3 stages each) compared cell by cell with the oracle over the whole 256^3
    state (about a minute of oracle time on the box's host cores)."""
    prob, q = wl.cfg3()
    check_rk(prob, q, steps=10)


def test_single_stage_combination_matches_forward_euler_of_rhs():
    """q + dt L(q) assembled by the last sweep equals the separately returned L (same kernels, two output modes)."""
    prob, q = wl.random_state(3, (30, 20, 25), 2, seed=9, periodic=True)
    with Gpu(prob) as g:
        L = g.rhs(q)
    # after a full step the state must differ from q by O(dt): a smoke check that the in-place stages ran
    orc = oracle.Oracle(prob)
    dt = orc.cfl_dt(q.copy(), 0.3)
    with Gpu(prob) as g:
        q1 = g.rk3(q, [dt])
    it = prob.interior()
    assert np.all(np.isfinite(q1[it]))
    lin = q[it] + dt * L[it]
    # RK3 = Euler + O(dt^2): the difference is far smaller than the increment itself
    assert np.max(np.abs(q1[it][0] - lin[0])) < 0.5 * np.max(np.abs(dt * L[it][0]))


# ---------------------------------------------------------------------------------------------
# a6: CFL
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ndim,nf", TEMPLATE_SET)
def test_cfl_dt_parity(ndim, nf):
    prob, q = wl.random_state(ndim, SIZES[ndim], nf, seed=4, periodic=True)
    ref = oracle.Oracle(prob).cfl_dt(q, prob.cfl)
    with Gpu(prob) as g:
        got = g.cfl_dt(q)
    assert abs(got - ref) <= 1e-13 * ref


def test_cfl_dt_parity_cfg3():
    prob, q = wl.cfg3(n=128)
    ref = oracle.Oracle(prob).cfl_dt(q, prob.cfl)
    with Gpu(prob) as g:
        got = g.cfl_dt(q)
    assert abs(got - ref) <= 1e-13 * ref


def test_cfl_dt_propagates_nan_and_advance_host_stops():
    """An inadmissible cell (NaN energy; negative c^2) must not be dropped by the max-reduction: dt is NaN, and
    mfc_advance_host refuses to step on."""
    prob, q = wl.random_state(3, (20, 12, 9), 2, seed=4, periodic=True)
    it = prob.interior()
    for poison in ("nan", "negative_c2"):
        qb = q.copy()
        if poison == "nan":
            qb[it][prob.nf + prob.ndim][3, 5, 7] = np.nan
        else:
            qb[it][prob.nf + prob.ndim][3, 5, 7] = -1.0e12          # p so negative that (Gamma + 1) p + Pi < 0
        with Gpu(prob) as g:
            assert np.isnan(g.cfl_dt(qb))
            qh = g.torch.from_numpy(qb.copy()).pin_memory()
            with pytest.raises(B.MfcError) as ei:
                B.mfc_advance_host(g.ctx, qh.data_ptr(), 1, 0.0, g.stream)
            assert ei.value.code == B.MFC_ENONFINITE
            assert np.array_equal(qh.numpy(), qb, equal_nan=True)


def test_step_runs_beside_a_tensor_core_kernel_on_another_stream():
    """The 3D kernel takes all 512 TMEM columns of a multiprocessor (mfc.h "Tensor memory"); a tcgen05 GEMM on another
    stream is serialised against it by the hardware allocator, in either order, without deadlock and without changing a bit."""
    prob, q = wl.random_state(3, (96, 72, 64), 2, seed=31, periodic=False, rough=False)
    orc = oracle.Oracle(prob)
    dts = [0.5 * orc.cfl_dt(q.copy(), prob.cfl)] * 4
    with Gpu(prob) as g:
        torch = g.torch
        alone = g.rk3(q, dts)
        a = torch.randn(4096, 4096, device=g.dev, dtype=torch.bfloat16)
        b = torch.randn(4096, 4096, device=g.dev, dtype=torch.bfloat16)
        side = torch.cuda.Stream()
        qd = g.to_dev(q)
        torch.cuda.synchronize()
        with torch.cuda.stream(side):
            for _ in range(40):
                c = a @ b
        for dt in dts:
            B.mfc_rk3_step(g.ctx, qd.data_ptr(), float(dt), g.stream)
            with torch.cuda.stream(side):
                for _ in range(10):
                    c = a @ b
        torch.cuda.synchronize()
        assert torch.isfinite(c.float()).all()
        assert np.array_equal(qd.cpu().numpy()[prob.interior()], alone[prob.interior()])


# ---------------------------------------------------------------------------------------------
# block decomposition: one block that is its own neighbour == the single-block solver
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ndim,n,periodic_dims", [(2, (70, 45), (0,)), (3, (40, 29, 33), (0, 1, 2)), (3, (41, 30, 33), (1,)), (3, (40, 29, 33), ())])
def test_block_solver_with_halo_ghosts_reproduces_the_single_block_solver(ndim, n, periodic_dims):
    """MFC_BC_HALO on every side + halo.fill_ghosts (local wrap / edge copies for a 1 x 1 x 1 decomposition) through
    mfc_rhs and the per-stage mfc_rk3_stage gives the bits of the ordinary context: the kernels read the ghost cells the
    caller filled, whatever the staging path (TMA at n[0] = 40, cp.async at 41)."""
    import dataclasses
    from paper_2305_09163_b200 import halo
    prob, q = wl.random_state(ndim, n, 2, seed=90 + ndim, periodic=True)
    bc = tuple(wl.BC_PERIODIC if d in periodic_dims else wl.BC_EXTRAP for d in range(3))
    prob = dataclasses.replace(prob, bc_lo=bc, bc_hi=bc)
    orc = oracle.Oracle(prob)
    dts = [0.7 * orc.cfl_dt(q.copy(), prob.cfl)] * 3
    it = prob.interior()
    with Gpu(prob) as g:
        torch = g.torch
        L_ref = g.rhs(q)[it]
        q_ref = g.rk3(q, dts)[it]
        dt_ref = g.cfl_dt(q)
        dec = halo.Decomposition((1, 1, 1), prob.bc_lo, prob.bc_hi)
        blk = halo.BlockSolver(prob, dec, 0)
        try:
            qd = g.to_dev(q)
            out = torch.zeros_like(qd)
            blk.rhs(qd, out)
            assert blk.cfl_dt(qd) == dt_ref
            for dt in dts:
                blk.rk3_step(qd, dt)
            torch.cuda.synchronize()
            assert np.array_equal(out.cpu().numpy()[it], L_ref)
            assert np.array_equal(qd.cpu().numpy()[it], q_ref)
        finally:
            blk.close()


def test_halo_sides_are_refused_in_a_non_uniform_dimension():
    import dataclasses
    prob, q = wl.random_state(2, (20, 12), 2, seed=1)
    ps = dataclasses.replace(wl.with_stretched_grid(prob), bc_lo=(B.MFC_BC_HALO,) * 3, bc_hi=(B.MFC_BC_HALO,) * 3)
    with pytest.raises(B.MfcError) as ei:
        Gpu(ps)
    assert ei.value.code == B.MFC_EUNSUPPORTED


# ---------------------------------------------------------------------------------------------
# host-buffer entry point and measurement hooks
# ---------------------------------------------------------------------------------------------
def test_advance_host_equals_device_path():
    prob, q = wl.random_state(2, (90, 40), 2, seed=12, periodic=True, rough=False)
    with Gpu(prob) as g:
        torch = g.torch
        qd = g.to_dev(q)
        t_dev = 0.0
        for _ in range(3):
            dt = B.mfc_cfl_dt(g.ctx, qd.data_ptr(), g.stream)
            B.mfc_rk3_step(g.ctx, qd.data_ptr(), dt, g.stream)
            t_dev += dt
        torch.cuda.synchronize()
        ref = qd.cpu().numpy()
        qh = torch.from_numpy(q.copy()).pin_memory()
        t_host = B.mfc_advance_host(g.ctx, qh.data_ptr(), 3, 0.0, g.stream)
        it = prob.interior()
        assert np.array_equal(qh.numpy()[it], ref[it])
        assert t_host == pytest.approx(t_dev, rel=1e-15)
        # fixed dt, pageable memory
        qp = q.copy()
        B.mfc_advance_host(g.ctx, qp.ctypes.data, 1, 1e-7, g.stream)
        ref1 = g.rk3(q, [1e-7])
        assert np.array_equal(qp[it], ref1[it])


def test_step_cfl_equals_cfl_dt_followed_by_rk3_step():
    """mfc_step_cfl only reorders the enqueue (first ghost fill before the wait for dt): same dt, same bits; an inadmissible
    state is refused with MFC_ENONFINITE and its interior left alone."""
    prob, q = wl.random_state(3, (40, 29, 33), 2, seed=33, periodic=False)
    it = prob.interior()
    with Gpu(prob) as g:
        qa, qb = g.to_dev(q), g.to_dev(q)
        dts_a, dts_b = [], []
        for _ in range(4):
            dts_a.append(B.mfc_cfl_dt(g.ctx, qa.data_ptr(), g.stream))
            B.mfc_rk3_step(g.ctx, qa.data_ptr(), dts_a[-1], g.stream)
            dts_b.append(B.mfc_step_cfl(g.ctx, qb.data_ptr(), g.stream))
        g.torch.cuda.synchronize()
        assert dts_a == dts_b
        assert np.array_equal(qa.cpu().numpy()[it], qb.cpu().numpy()[it])
        bad = q.copy()
        bad[it][prob.nf + prob.ndim][3, 5, 7] = np.nan
        qc = g.to_dev(bad)
        with pytest.raises(B.MfcError) as ei:
            B.mfc_step_cfl(g.ctx, qc.data_ptr(), g.stream)
        assert ei.value.code == B.MFC_ENONFINITE
        g.torch.cuda.synchronize()
        assert np.array_equal(qc.cpu().numpy()[it], bad[it], equal_nan=True)


def test_profile_hooks_count_launches_and_time():
    prob, q = wl.random_state(3, (32, 32, 32), 2, seed=1)
    with Gpu(prob) as g:
        qd = g.to_dev(q)
        n0 = B.mfc_launch_count(g.ctx)
        B.mfc_profile_enable(g.ctx, True)
        B.mfc_rk3_step(g.ctx, qd.data_ptr(), 1e-9, g.stream)
        B.mfc_cfl_dt(g.ctx, qd.data_ptr(), g.stream)
        assert B.mfc_launch_count(g.ctx) - n0 == 3 * 2 + 1    # per stage: ghost fill + one fused launch; the CFL reduction
        for kid, want in [(B.MFC_K_RHS, 3), (B.MFC_K_GHOST, 3), (B.MFC_K_CFL, 1)]:
            n, ms = B.mfc_profile_get(g.ctx, kid, reset=True)
            assert n == want and ms > 0.0
        n, ms = B.mfc_profile_get(g.ctx, B.MFC_K_RHS)
        assert n == 0 and ms == 0.0
        B.mfc_profile_enable(g.ctx, False)


def test_dfma_probe_reports_a_plausible_fp64_rate():
    from paper_2305_09163_b200 import build
    build.build()
    tf, ms = B.mfc_probe_dfma(-1)
    assert 5.0 < tf < 80.0 and ms > 0.0


def test_long_run_stays_finite_and_is_bitwise_reproducible():
    """150 steps (CFL + RK3 each) of the shock-bubble workload at 64^3 through the default 3D kernel, twice: finite state, the
    same bits both times (the two warp kinds of the split kernel meet only through mbarriers; a race would show here)."""
    prob, q = wl.cfg2(n=64)
    outs = []
    for _ in range(2):
        with Gpu(prob) as g:
            qd = g.to_dev(q)
            for _s in range(150):
                dt = B.mfc_cfl_dt(g.ctx, qd.data_ptr(), g.stream)
                B.mfc_rk3_step(g.ctx, qd.data_ptr(), dt, g.stream)
            g.torch.cuda.synchronize()
            outs.append(qd.cpu().numpy()[prob.interior()])
    assert np.all(np.isfinite(outs[0]))
    assert np.array_equal(outs[0], outs[1])


# ---------------------------------------------------------------------------------------------
# contexts on several devices of one process (mfc_opts.device): the opt-in to large dynamic shared
# memory is per kernel AND device, so the second device's first launch must set it again
# ---------------------------------------------------------------------------------------------
def test_contexts_on_two_devices_in_one_process():
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two visible GPUs")
    prob, q = wl.random_state(3, (40, 20, 12), 2, seed=9, periodic=True)
    outs = []
    for dev in (0, 1):
        with torch.cuda.device(dev):
            with Gpu(prob, device=dev) as g:
                outs.append(g.rhs(q)[prob.interior()])
    assert np.array_equal(outs[0], outs[1])


# ---------------------------------------------------------------------------------------------
# a decomposed run on ONE GPU -- every block a context of its own in this process,
# ghost cells moved between the blocks' arrays by the same slab logic the P2P exchange uses (halo.fill_ghosts_in_process)
# -- against the undivided GPU run (bit for bit: same kernels, same arithmetic per cell, identical 1 / dx) and against
# the oracle on the global array.
# ---------------------------------------------------------------------------------------------
DECOMPOSITIONS = [((2, 1, 1), "2x1x1"), ((1, 2, 2), "1x2x2"), ((2, 2, 2), "2x2x2")]
BOUNDARIES = [((0, 1, 2), "periodic"), ((), "extrapolation"), ((1,), "mixed")]


@pytest.mark.parametrize("dims,_dn", DECOMPOSITIONS)
@pytest.mark.parametrize("periodic_dims,_bn", BOUNDARIES)
def test_decomposed_run_equals_the_single_block_run_and_the_oracle(dims, _dn, periodic_dims, _bn):
    import dataclasses
    from paper_2305_09163_b200 import halo
    # even block extents in x on both levels (the undivided grid and every block take the kernel with Z warps), ragged
    # tiles, blocks of different sizes in y and z (45 = 23 + 22, 37 = 19 + 18)
    prob, q = wl.random_state(3, (72, 45, 37), 2, seed=77, periodic=True)
    bc = tuple(wl.BC_PERIODIC if d in periodic_dims else wl.BC_EXTRAP for d in range(3))
    prob = dataclasses.replace(prob, bc_lo=bc, bc_hi=bc)
    it = prob.interior()
    nsteps = 10
    with Gpu(prob) as g:
        L_one = g.rhs(q)[it]
        qd = g.to_dev(q)
        dts = []
        for _ in range(nsteps):
            dts.append(B.mfc_cfl_dt(g.ctx, qd.data_ptr(), g.stream))
            B.mfc_rk3_step(g.ctx, qd.data_ptr(), dts[-1], g.stream)
        g.torch.cuda.synchronize()
        q_one = qd.cpu().numpy()[it]
    dec = halo.Decomposition(dims, prob.bc_lo, prob.bc_hi)
    with halo.LocalBlocks(prob, q, dec) as blocks:
        L_dec = blocks.gather(blocks.rhs())[it]
        dts_dec = []
        for _ in range(nsteps):
            dts_dec.append(blocks.cfl_dt())              # the global minimum over the blocks
            blocks.rk3_step(dts_dec[-1])
        q_dec = blocks.gather()[it]
    assert np.array_equal(L_dec, L_one)
    assert dts_dec == dts
    assert np.array_equal(q_dec, q_one)
    # ... and the oracle on the global array, at the usual bars
    orc = oracle.Oracle(prob)
    qo = q.copy()
    L_ref = orc.rhs(qo)
    err = parity_errors(prob, _pad_like(prob, L_dec), L_ref, rhs_floors(prob, orc, qo))
    assert np.all(err <= RHS_TOL), err
    for dt in dts:
        orc.rk3_step(qo, dt)
    S = row_scales(prob, qo[it])
    e_rk = max(float(np.max(np.abs(q_dec[k] - qo[it][k])) / S[k]) for k in range(prob.neq))
    assert e_rk <= RK_TOL, e_rk


def _pad_like(prob, interior_values):
    a = np.zeros(prob.shape())
    a[prob.interior()] = interior_values
    return a
