"""Pins of the oracle's non-uniform-grid path (Listing 1, Eq. 15
PAPER.md:396-399) against things other than itself.  CPU only (`-m "not gpu"`)."""
from __future__ import annotations

import dataclasses

import numpy as np
import pytest
from numpy.polynomial import Polynomial
from numpy.polynomial.legendre import leggauss

import oracle
from paper_2305_09163_b200 import workloads as wl

NG = wl.NG


def random_edges(rng, n=5, ratio=3.0):
    w = rng.uniform(1.0, ratio, size=n)
    return np.concatenate([[0.0], np.cumsum(w)]) * rng.uniform(0.01, 10.0) + rng.uniform(-5, 5)


def cell_averages(poly: Polynomial, e):
    P = poly.integ()
    return (P(e[1:]) - P(e[:-1])) / np.diff(e)


def test_nonuniform_weno_reduces_to_the_uniform_scheme():
    """Uniform edges: the general-stencil definitions give the Jiang-Shu constants (1/3, -7/6, 11/6; 1/10, 6/10, 3/10;
    13/12, 1/4) -- i.e. orc_weno5 -- to round-off, for rough and smooth data."""
    rng = np.random.default_rng(3)
    for _ in range(300):
        h = rng.uniform(1e-3, 10.0)
        xe = rng.uniform(-3, 3) + h * np.arange(6.0)
        v = rng.normal(size=5) * 10.0 ** rng.uniform(-3, 6) + rng.normal() * 10.0 ** rng.uniform(-3, 6)
        a = oracle.weno5_nonuniform(xe, v)
        b = oracle.weno5(*v)
        s = np.max(np.abs(v))
        assert abs(a[0] - b[0]) <= 2e-13 * s and abs(a[1] - b[1]) <= 2e-13 * s


def test_nonuniform_weno_polynomial_exactness():
    """Cell averages of a polynomial of degree <= 2 on a random monotone grid: both face values exact with ANY weights
    (every candidate is exact); degree 3 and 4: exact at the ideal weights (eps huge), i.e. the ideal weights computed from
    the outermost cells reproduce the five-cell reconstruction; a quartic with Jiang-Shu weights is not exact."""
    rng = np.random.default_rng(5)
    worst = 0.0
    for _ in range(200):
        xe = random_edges(rng)
        L = xe[-1] - xe[0]
        for deg in range(5):
            poly = Polynomial(rng.normal(size=deg + 1), domain=[xe[0], xe[-1]], window=[-1, 1])
            v = cell_averages(poly, xe)
            s = np.max(np.abs(v)) + 1e-300
            for eps in ([1e-16, 1e-6, 1e10] if deg <= 2 else [1e14 * s * s]):
                vL, vR = oracle.weno5_nonuniform(xe, v, eps)
                assert abs(vL - poly(xe[3])) <= 2e-11 * s, (deg, eps)
                assert abs(vR - poly(xe[2])) <= 2e-11 * s, (deg, eps)
            if deg == 4:
                vL, _ = oracle.weno5_nonuniform(xe, v, 1e-16)
                worst = max(worst, abs(vL - poly(xe[3])) / s)
    assert worst > 1e-4          # the nonlinear weights are really in use


def test_nonuniform_smoothness_indicators_follow_the_jiang_shu_integral():
    """beta_r is not exposed; its definition is pinned through the weights it produces: with eps = 0-like and data whose
    candidates differ, the oracle's value must equal sum omega_r p_r with beta_r evaluated INDEPENDENTLY here by Gauss
    quadrature of  sum_l dx^(2l-1) int (d^l p_r/dx^l)^2 dx  over the centre cell, p_r fitted by a linear solve."""
    rng = np.random.default_rng(9)
    gx, gw = leggauss(6)
    for _ in range(100):
        xe = random_edges(rng, ratio=2.5)
        v = rng.normal(size=5)
        xm, xp = xe[2], xe[3]
        dx = xp - xm
        pL, pR, beta = [], [], []
        for r in range(3):
            e = xe[r:r + 4]
            # quadratic with the three cell averages: solve for monomial coefficients about the cell centre
            xc = 0.5 * (xm + xp)
            A = np.array([[((e[j + 1] - xc) ** (k + 1) - (e[j] - xc) ** (k + 1)) / ((k + 1) * (e[j + 1] - e[j])) for k in range(3)]
                          for j in range(3)])
            a = np.linalg.solve(A, v[r:r + 3])
            p = Polynomial(a)
            xs = 0.5 * dx * gx                                   # nodes about the centre
            b = dx * np.sum(0.5 * dx * gw * p.deriv(1)(xs) ** 2) + dx ** 3 * np.sum(0.5 * dx * gw * p.deriv(2)(xs) ** 2)
            beta.append(b)
            pL.append(p(xp - xc))
            pR.append(p(xm - xc))
        # ideal weights from five-cell exactness, independently: solve sum_r d_r p_r(face) = p5(face) on monomial data
        def ideal(face):
            rows, rhs = [], []
            for deg in (3, 4, 2):
                poly = Polynomial.basis(deg, domain=[xe[0], xe[-1]], window=[-1, 1])
                vv = cell_averages(poly, xe)
                cand = []
                for r in range(3):
                    e = xe[r:r + 4]
                    xc = 0.5 * (xm + xp)
                    A = np.array([[((e[j + 1] - xc) ** (k + 1) - (e[j] - xc) ** (k + 1)) / ((k + 1) * (e[j + 1] - e[j])) for k in range(3)]
                                  for j in range(3)])
                    cand.append(Polynomial(np.linalg.solve(A, vv[r:r + 3]))(face - xc))
                if deg == 2:
                    rows.append([1.0, 1.0, 1.0]); rhs.append(1.0)
                else:
                    rows.append(cand); rhs.append(poly(face))
            return np.linalg.solve(np.array(rows), np.array(rhs))
        eps = 1e-16
        for face, cands, got in ((xp, pL, 0), (xm, pR, 1)):
            d = ideal(face)
            al = d / (np.array(beta) + eps) ** 2
            want = np.sum(al / al.sum() * np.array(cands))
            have = oracle.weno5_nonuniform(xe, v, eps)[got]
            assert abs(have - want) <= 1e-9 * np.max(np.abs(v)), (have, want)


def test_nonuniform_weno_mirror_symmetry():
    rng = np.random.default_rng(11)
    for _ in range(100):
        xe = random_edges(rng)
        v = rng.normal(size=5)
        vL, vR = oracle.weno5_nonuniform(xe, v)
        mL, mR = oracle.weno5_nonuniform(-xe[::-1], v[::-1].copy())
        assert abs(vL - mR) <= 1e-12 and abs(vR - mL) <= 1e-12


def test_padded_edges_follow_the_source_cell_reading():
    e = np.array([0.0, 1.0, 3.0, 6.0, 10.0, 15.0])
    per = oracle.padded_edges(e, 0, 0)
    assert np.allclose(np.diff(per), [3, 4, 5, 1, 2, 3, 4, 5, 1, 2, 3])
    ext = oracle.padded_edges(e, 1, 1)
    assert np.allclose(np.diff(ext), [1, 1, 1, 1, 2, 3, 4, 5, 5, 5, 5])
    assert per[NG] == 0.0 and ext[NG] == 0.0 and per[-NG - 1] == 15.0


@pytest.mark.parametrize("ndim", [1, 2, 3])
def test_rhs_with_uniform_edges_equals_the_uniform_rhs(ndim):
    n = {1: (41,), 2: (17, 13), 3: (9, 8, 7)}[ndim]
    prob, q = wl.random_state(ndim, n, 2, seed=4, periodic=(ndim != 2))
    pe = dataclasses.replace(prob, edges=tuple(np.linspace(prob.lo[d], prob.hi[d], prob.n[d] + 1) if d < ndim else None for d in range(3)))
    a = oracle.Oracle(prob).rhs(q.copy())[prob.interior()]
    b = oracle.Oracle(pe).rhs(q.copy())[prob.interior()]
    for k in range(prob.neq):
        assert np.max(np.abs(a[k] - b[k])) <= 1e-11 * np.max(np.abs(a[k]))
    assert oracle.Oracle(pe).cfl_dt(q, 0.3) == pytest.approx(oracle.Oracle(prob).cfl_dt(q, 0.3), rel=1e-13)


@pytest.mark.parametrize("ndim,periodic", [(1, True), (2, False), (3, True)])
def test_stretched_grid_uniform_state_and_conservation(ndim, periodic):
    """Uniform state => L vanishes to round-off on a stretched grid (the general-stencil coefficients sum to 1 only to an
    ulp, so unlike the uniform scheme it is not bitwise zero): 1e-12 of the RHS of a non-uniform state on the same grid;
    periodic conservative rows satisfy sum L_k dV = 0 (fluxes telescope with the cell's own width in Eq. 9)."""
    n = {1: (40,), 2: (18, 14), 3: (10, 9, 8)}[ndim]
    prob, q = wl.random_state(ndim, n, 2, seed=6, periodic=periodic)
    prob = wl.with_stretched_grid(prob)
    orc = oracle.Oracle(prob)
    it = prob.interior()
    qu = q.copy()
    qu[it] = qu[it][:, :1, :1, :1]
    L = orc.rhs(q.copy())[it]
    Lu = orc.rhs(qu)[it]
    for k in range(prob.neq):
        assert np.max(np.abs(Lu[k])) <= 1e-12 * np.max(np.abs(L[k]))
    if periodic:
        dV = np.ones(())
        W = [prob.widths(d) if d < ndim else np.ones(1) for d in range(3)]
        dV = W[2][:, None, None] * W[1][None, :, None] * W[0][None, None, :]
        for k in range(prob.nf + ndim + 1):
            assert abs(np.sum(L[k] * dV)) <= 1e-11 * np.sum(np.abs(L[k]) * dV)


def test_stretched_grid_advection_converges_at_fifth_order():
    """C3 on the Eq. 15 grid: 1-D periodic advection of a smooth density wave (single fluid, u = p = 1), initialised and
    compared with EXACT cell averages on the stretched cells, dt ~ dx^(5/3) so that RK3 does not mask the spatial order."""
    errs = []
    ns = (40, 80, 160)
    for n in ns:
        prob, _ = wl.random_state(1, (n,), 1, seed=1, periodic=True)
        prob = dataclasses.replace(prob, fluids=[(1.4, 0.0)])
        prob = wl.with_stretched_grid(prob)
        e = np.asarray(prob.edges[0])
        Lx = e[-1] - e[0]
        k = 2 * np.pi / Lx
        avg = lambda shift: 1.0 + 0.2 * (np.cos(k * (e[:-1] - shift)) - np.cos(k * (e[1:] - shift))) / (k * np.diff(e))
        rho = avg(0.0)[None, None, :]
        q = wl.assemble(prob, [np.ones_like(rho)], [rho], [np.ones_like(rho)], np.ones_like(rho))
        orc = oracle.Oracle(prob)
        T, t = 0.25 * Lx, 0.0
        dt = 0.2 * np.min(np.diff(e)) * (40.0 / n) ** (2.0 / 3.0)
        while t < T - 1e-14:
            step = min(dt, T - t)
            orc.rk3_step(q, step)
            t += step
        errs.append(np.sum(np.abs(q[prob.interior()][0, 0, 0] - avg(T)) * np.diff(e)) / Lx)
    rates = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    assert np.all(rates > 4.6), (rates, errs)


def test_eq15_stretching_is_the_papers_formula_at_a_point():
    """PAPER.md:396-399 (Eq. 15) evaluated by hand at x = 0.3 (L = 1, a = 4, x_a = -0.12, x_b = 0.12):
    x + x/a [log cosh(1.68) + log cosh(0.72) - 2 log cosh(0.48)] = 0.3 + 0.075 (1.0209984 + 0.2394835 - 2 x 0.1110304)."""
    e = wl.stretched_edges(10, -0.5, 0.5)           # uniform edges -0.5, -0.4, .., 0.5 in the centred coordinate
    x = 0.3
    want = x + x / 4.0 * (np.log(np.cosh(4 * (x + 0.12))) + np.log(np.cosh(4 * (x - 0.12))) - 2 * np.log(np.cosh(0.48)))
    assert e[8] == pytest.approx(want, rel=1e-14)
    assert want == pytest.approx(0.3 + 0.075 * (1.0209984 + 0.2394835 - 2 * 0.1110304), rel=1e-6)
    assert np.allclose(e, -e[::-1])                 # odd map: the refinement is centred
