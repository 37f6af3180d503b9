"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs 0-4).

This module serves BOTH the CPU oracle (tests, bench cpu_baseline) and the CUDA path (tests,
bench).  It imports neither.  It holds no step of the method (no cons->prim, no WENO, no HLLC,
no RHS, no RK, no CFL): it only *defines initial data*.  Initial data are stated in primitive
variables (alpha_i, rho_i, u, p); the single piece of physics used to turn them into the
conservative input array is the stiffened-gas total energy, PAPER.md:54-58 (Eq. 1) with the
alpha-weighted mixture rule and the kinetic energy added (reading B2):

    rho E = sum_i alpha_i/(gamma_i-1) * p + sum_i alpha_i*gamma_i*pi_inf_i/(gamma_i-1) + rho |u|^2 / 2

The paper's case files (3D two-component air/water, bubble clouds) are not
available; these inputs stand in for them.

State layout (PAPER.md:238 flattened arrays, equation index slowest):
    q[eq, z, y, x], x fastest, padded by ng=3 ghost layers on both sides of every ACTIVE dimension
    (inactive dimensions have extent 1).  Equation order:
    alpha_i rho_i (i=1..N_f), rho u_d (d=1..D), rho E, alpha_i (i=1..N_f-1).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Sequence, Tuple

import numpy as np

NG = 3  # ghost layers, PAPER.md:168 (buffer size set by the WENO order; WENO5 -> 3)

BC_PERIODIC = 0
BC_EXTRAP = 1

# stiffened-gas parameters named by BASELINE.json
WATER = (4.4, 6.0e8)
AIR = (1.4, 0.0)
VAPOUR = (1.33, 0.0)


@dataclass
class Problem:
    """Everything mfc_init needs (grid, fluids, BCs, options); plain data only."""

    name: str
    ndim: int
    n: Tuple[int, int, int]  # interior cells per dimension (1 for inactive dims)
    lo: Tuple[float, float, float]
    hi: Tuple[float, float, float]
    fluids: List[Tuple[float, float]]  # (gamma, pi_inf) per fluid
    bc_lo: Tuple[int, int, int]
    bc_hi: Tuple[int, int, int]
    weno_eps: float = 1.0e-16
    cfl: float = 0.3
    steps: int = 1
    seed: int | None = None
    notes: str = ""
    weno_order: int = 5  # 5: WENO5-JS (the paper's default), 3: WENO3-JS, 1: piecewise constant
    kapila: bool = False  # K div(u) source of PAPER.md Eq. 2 on the alpha row (two fluids); False = Allaire
    # non-uniform Cartesian spacing: per dimension the n + 1 edges of the interior cells, or None (uniform)
    edges: Tuple | None = None
    # per dimension the reciprocal cell width to hand to mfc_init instead of n / (hi - lo) (mfc_grid.inv_dx): set on the
    # blocks of a decomposed grid to the global value, so that every block divides by the identical number
    inv_dx: Tuple | None = None

    @property
    def nf(self) -> int:
        return len(self.fluids)

    @property
    def neq(self) -> int:
        return 2 * self.nf + self.ndim

    @property
    def padded(self) -> Tuple[int, int, int]:
        return tuple(self.n[d] + 2 * NG if d < self.ndim else 1 for d in range(3))

    @property
    def dx(self) -> Tuple[float, float, float]:
        return tuple((self.hi[d] - self.lo[d]) / self.n[d] if d < self.ndim else 1.0 for d in range(3))

    @property
    def cells(self) -> int:
        return int(self.n[0]) * int(self.n[1]) * int(self.n[2])

    def shape(self) -> Tuple[int, int, int, int]:
        px, py, pz = self.padded
        return (self.neq, pz, py, px)

    def interior(self) -> Tuple[slice, slice, slice, slice]:
        sl = [slice(NG, NG + self.n[d]) if d < self.ndim else slice(0, 1) for d in range(3)]
        return (slice(None), sl[2], sl[1], sl[0])

    def centers(self, d: int) -> np.ndarray:
        if self.edges is not None and self.edges[d] is not None:
            e = np.asarray(self.edges[d], dtype=np.float64)
            return 0.5 * (e[:-1] + e[1:])
        h = self.dx[d]
        return self.lo[d] + (np.arange(self.n[d], dtype=np.float64) + 0.5) * h

    def widths(self, d: int) -> np.ndarray:
        """Widths of the interior cells of dimension d."""
        if self.edges is not None and self.edges[d] is not None:
            return np.diff(np.asarray(self.edges[d], dtype=np.float64))
        return np.full(self.n[d], self.dx[d])


def _grid(ndim: int, n: Sequence[int]) -> Tuple[Tuple[int, int, int], Tuple[float, ...], Tuple[float, ...]]:
    nn = tuple(int(n[d]) if d < ndim else 1 for d in range(3))
    return nn, (0.0, 0.0, 0.0), (1.0, 1.0, 1.0)


def stretched_edges(n: int, lo: float = 0.0, hi: float = 1.0, a: float = 4.0, xa: float = -0.12, xb: float = 0.12) -> np.ndarray:
    """The n + 1 cell edges of a grid refined near the middle of [lo, hi] by the hyperbolic-tangent stretching of
    PAPER.md:396-399 (Eq. 15), applied to the uniform edges in the centred coordinate x = (xi - mid) (the paper's droplet
    sits at the origin, x_a = -1.2 D, x_b = 1.2 D, a_x = 4):
        x_s = x + (x / a) [log cosh(a (x - x_a) / L) + log cosh(a (x - x_b) / L) - 2 log cosh(a (x_b - x_a) / (2 L))]
    L = hi - lo.  Cells at the ends are about 2.6 x wider than in the middle for the defaults.  Input definition only."""
    L = hi - lo
    mid = 0.5 * (lo + hi)
    x = np.linspace(lo, hi, n + 1) - mid
    lc = lambda t: np.log(np.cosh(t))
    xs = x + (x / a) * (lc(a * (x - xa) / L) + lc(a * (x - xb) / L) - 2.0 * lc(a * (xb - xa) / (2.0 * L)))
    assert np.all(np.diff(xs) > 0.0)
    return xs + mid


def with_stretched_grid(prob: Problem, dims=None, **kw) -> Problem:
    """The same problem on the Eq. 15 grid in the given dimensions (default: all active ones).  Initial data are defined
    per cell index, so the state array is reused as it is: same per-cell values on the stretched cells."""
    import dataclasses
    dims = range(prob.ndim) if dims is None else dims
    edges = [None, None, None]
    for d in dims:
        edges[d] = stretched_edges(prob.n[d], prob.lo[d], prob.hi[d], **kw)
    return dataclasses.replace(prob, name=prob.name + "_stretched", edges=tuple(edges))


def assemble(prob: Problem, alpha: Sequence[np.ndarray], rho_i: Sequence, vel: Sequence, p) -> np.ndarray:
    """Build the padded conservative array from primitive fields given on the interior.

    alpha: N_f arrays (z,y,x) summing to 1; rho_i: N_f densities (scalars or arrays);
    vel: D velocity components; p: pressure.  Ghost cells are left at zero (the solver fills them).
    """
    nf, D = prob.nf, prob.ndim
    nz, ny, nx = prob.n[2], prob.n[1], prob.n[0]
    shp = (nz, ny, nx)
    q = np.zeros(prob.shape(), dtype=np.float64)
    it = prob.interior()
    rho = np.zeros(shp)
    Gam = np.zeros(shp)
    Pi = np.zeros(shp)
    for i in range(nf):
        a = np.broadcast_to(np.asarray(alpha[i], dtype=np.float64), shp)
        ar = a * np.broadcast_to(np.asarray(rho_i[i], dtype=np.float64), shp)
        q[(i,) + it[1:]] = ar
        rho += ar
        g, pinf = prob.fluids[i]
        Gam += a / (g - 1.0)
        Pi += a * g * pinf / (g - 1.0)
        if i < nf - 1:
            q[(nf + D + 1 + i,) + it[1:]] = a
    ke = np.zeros(shp)
    for d in range(D):
        u = np.broadcast_to(np.asarray(vel[d], dtype=np.float64), shp)
        q[(nf + d,) + it[1:]] = rho * u
        ke += 0.5 * rho * u * u
    q[(nf + D,) + it[1:]] = Gam * np.broadcast_to(np.asarray(p, dtype=np.float64), shp) + Pi + ke
    return q


# --------------------------------------------------------------------------------------------
# config 0: 1D two-fluid air/water shock tube
# --------------------------------------------------------------------------------------------
def cfg0(n: int = 1000) -> Tuple[Problem, np.ndarray]:
    nn, lo, hi = _grid(1, (n,))
    prob = Problem("cfg0_shocktube_1d", 1, nn, lo, hi, [WATER, AIR], (BC_EXTRAP,) * 3, (BC_EXTRAP,) * 3,
                   steps=200, notes="x<0.7 water p=1e9, else air rho=50 p=1e5")
    x = prob.centers(0)[None, None, :]
    left = x < 0.7
    aw = np.where(left, 1.0 - 1.0e-6, 1.0e-6)
    p = np.where(left, 1.0e9, 1.0e5)
    q = assemble(prob, [aw, 1.0 - aw], [1000.0, 50.0], [0.0], p)
    return prob, q


# --------------------------------------------------------------------------------------------
# config 1: 2D periodic two-fluid smooth advection
# --------------------------------------------------------------------------------------------
def cfg1(n: int = 512, seed: int = 1001) -> Tuple[Problem, np.ndarray]:
    nn, lo, hi = _grid(2, (n, n))
    prob = Problem("cfg1_advection_2d", 2, nn, lo, hi, [WATER, AIR], (BC_PERIODIC,) * 3, (BC_PERIODIC,) * 3,
                   steps=100, seed=seed, notes="alpha_air=0.5+0.4 sin sin + U(-1e-3,1e-3); u=(1,0.5); p=1e5")
    rng = np.random.default_rng(seed)
    x = prob.centers(0)[None, None, :]
    y = prob.centers(1)[None, :, None]
    a_air = 0.5 + 0.4 * np.sin(2 * np.pi * x) * np.sin(2 * np.pi * y) + rng.uniform(-1e-3, 1e-3, size=(1, n, n))
    q = assemble(prob, [1.0 - a_air, a_air], [1000.0, 50.0], [1.0, 0.5], 1.0e5)
    return prob, q


# --------------------------------------------------------------------------------------------
# config 2: 3D shock-bubble
# --------------------------------------------------------------------------------------------
def rankine_hugoniot_stiffened(rho1: float, p1: float, gamma: float, pi_inf: float, mach: float):
    """Post-shock state behind a planar shock of Mach number `mach` running into fluid at rest.

    Ideal-gas normal-shock relations with p -> p + pi_inf (textbook; a stiffened gas is an ideal gas
    in the shifted pressure).  Returns (rho2, u2, p2).  Part of the *input definition* of config 2.
    """
    c1 = np.sqrt(gamma * (p1 + pi_inf) / rho1)
    m2 = mach * mach
    pr = 1.0 + 2.0 * gamma / (gamma + 1.0) * (m2 - 1.0)
    rr = (gamma + 1.0) * m2 / ((gamma - 1.0) * m2 + 2.0)
    p2 = pr * (p1 + pi_inf) - pi_inf
    rho2 = rr * rho1
    u2 = mach * c1 * (1.0 - 1.0 / rr)
    return float(rho2), float(u2), float(p2)


def diffuse_interface(dist: np.ndarray, h: float, cells: float) -> np.ndarray:
    """Volume fraction of the fluid on the negative side of a signed distance `dist`: a tanh profile
    `cells` grid cells wide, floored to [1e-6, 1-1e-6].  A diffuse-interface method needs the interface
    resolved over a few cells; a one-cell staircase of alpha = 1e-6 | 1-1e-6 on a sphere makes WENO5
    overshoot alpha below 0 at the single-cell caps and the unlimited scheme of the paper (no positivity
    fix is mentioned) then produces NaN in the ORACLE itself within a few steps."""
    a = 0.5 * (1.0 - np.tanh(dist / (cells * h)))
    return np.clip(a, 1.0e-6, 1.0 - 1.0e-6)


INTERFACE_CELLS = 1.5


def cfg2(n: int = 128) -> Tuple[Problem, np.ndarray]:
    nn, lo, hi = _grid(3, (n, n, n))
    prob = Problem("cfg2_shock_bubble_3d", 3, nn, lo, hi, [WATER, AIR], (BC_EXTRAP,) * 3, (BC_EXTRAP,) * 3,
                   steps=50, notes="air bubble r=0.15 in water, Mach-1.5 water shock at x=0.1")
    x = prob.centers(0)[None, None, :]
    y = prob.centers(1)[None, :, None]
    z = prob.centers(2)[:, None, None]
    dist = np.sqrt((x - 0.5) ** 2 + (y - 0.5) ** 2 + (z - 0.5) ** 2) - 0.15
    a_air = diffuse_interface(dist, prob.dx[0], INTERFACE_CELLS)
    inside = dist < 0.0
    rho2, u2, p2 = rankine_hugoniot_stiffened(1000.0, 1.0e5, WATER[0], WATER[1], 1.5)
    post = np.broadcast_to(x < 0.1, inside.shape)
    rho_w = np.where(post, rho2, 1000.0)
    ux = np.where(post, u2, 0.0)
    p = np.where(post, p2, 1.0e5)
    q = assemble(prob, [1.0 - a_air, a_air], [rho_w, 1.2], [ux, 0.0, 0.0], p)
    return prob, q


# --------------------------------------------------------------------------------------------
# config 3 (headline): 3D bubble cloud
# --------------------------------------------------------------------------------------------
def cfg3(n: int = 256, seed: int = 2002, nbubbles: int = 64) -> Tuple[Problem, np.ndarray]:
    nn, lo, hi = _grid(3, (n, n, n))
    prob = Problem("cfg3_bubble_cloud_3d", 3, nn, lo, hi, [WATER, AIR], (BC_EXTRAP,) * 3, (BC_EXTRAP,) * 3,
                   steps=20, seed=seed, notes="64 air bubbles in water, p=1e7 pulse on x<0.05")
    rng = np.random.default_rng(seed)
    centers = rng.uniform(0.2, 0.8, size=(nbubbles, 3))
    radii = np.exp(rng.normal(np.log(0.03), 0.3, size=nbubbles))
    xc, yc, zc = prob.centers(0), prob.centers(1), prob.centers(2)
    # signed distance to the union of the spheres (min over bubbles), evaluated in a box around each bubble
    h = prob.dx[0]
    pad = 8.0 * INTERFACE_CELLS * h            # tanh(8) = 1 - 2e-7: beyond this the floor 1e-6 applies anyway
    dist = np.full((n, n, n), pad)
    for (cx, cy, cz), r in zip(centers, radii):
        ix = np.nonzero(np.abs(xc - cx) < r + pad)[0]
        iy = np.nonzero(np.abs(yc - cy) < r + pad)[0]
        iz = np.nonzero(np.abs(zc - cz) < r + pad)[0]
        if len(ix) == 0 or len(iy) == 0 or len(iz) == 0:
            continue
        sx, sy, sz = (slice(ix[0], ix[-1] + 1), slice(iy[0], iy[-1] + 1), slice(iz[0], iz[-1] + 1))
        d = np.sqrt((xc[sx][None, None, :] - cx) ** 2 + (yc[sy][None, :, None] - cy) ** 2
                    + (zc[sz][:, None, None] - cz) ** 2) - r
        dist[sz, sy, sx] = np.minimum(dist[sz, sy, sx], d)
    a_air = diffuse_interface(dist, h, INTERFACE_CELLS)
    inside = dist < 0.0
    p = np.where(np.broadcast_to(xc[None, None, :] < 0.05, inside.shape), 1.0e7, 1.0e5)
    q = assemble(prob, [1.0 - a_air, a_air], [1000.0, 1.2], [0.0, 0.0, 0.0], p)
    return prob, q


# --------------------------------------------------------------------------------------------
# config 4: 3D three-fluid, periodic
# --------------------------------------------------------------------------------------------
def _periodic_gaussian(f: np.ndarray, sigma: float) -> np.ndarray:
    """Periodic Gaussian smoothing by FFT (input generation only)."""
    out = f
    for ax in range(f.ndim):
        k = np.fft.rfftfreq(f.shape[ax]) * 2.0 * np.pi
        g = np.exp(-0.5 * (k * sigma) ** 2)
        shape = [1] * f.ndim
        shape[ax] = g.size
        out = np.fft.irfft(np.fft.rfft(out, axis=ax) * g.reshape(shape), n=f.shape[ax], axis=ax)
    return out


def cfg4(n: int = 384, seed: int = 3003, sigma: float = 8.0) -> Tuple[Problem, np.ndarray]:
    nn, lo, hi = _grid(3, (n, n, n))
    prob = Problem("cfg4_three_fluid_3d", 3, nn, lo, hi, [WATER, AIR, VAPOUR], (BC_PERIODIC,) * 3,
                   (BC_PERIODIC,) * 3, steps=10, seed=seed,
                   notes="softmax of standardised smoothed random fields; p=1e5; u=U(-1,1) per cell")
    rng = np.random.default_rng(seed)
    zs = []
    for _ in range(3):
        f = _periodic_gaussian(rng.uniform(0.0, 1.0, size=(n, n, n)), sigma)
        zs.append((f - f.mean()) / f.std())
    e = [np.exp(0.5 * z) for z in zs]
    tot = e[0] + e[1] + e[2]
    alpha = [ei / tot for ei in e]
    # make the stored N_f-1 fractions and the implied last one consistent: alpha_3 = 1 - a1 - a2
    alpha[2] = 1.0 - alpha[0] - alpha[1]
    vel = [rng.uniform(-1.0, 1.0, size=(n, n, n)) for _ in range(3)]
    q = assemble(prob, alpha, [1000.0, 1.2, 0.6], vel, 1.0e5)
    return prob, q


# --------------------------------------------------------------------------------------------
# generic seeded random admissible state (parity tests of every <D, N_f> instantiation)
# --------------------------------------------------------------------------------------------
def random_state(ndim: int, n: Sequence[int], nf: int, seed: int, periodic: bool = True,
                 rough: bool = True) -> Tuple[Problem, np.ndarray]:
    """Random admissible mixture state: smooth background + (optionally) jumps and cell noise."""
    nn, lo, hi = _grid(ndim, n)
    fl = [WATER, AIR, VAPOUR][:nf]
    bc = (BC_PERIODIC,) * 3 if periodic else (BC_EXTRAP,) * 3
    prob = Problem(f"random_d{ndim}_f{nf}_s{seed}", ndim, nn, lo, hi, fl, bc, bc, seed=seed)
    rng = np.random.default_rng(seed)
    shp = (nn[2], nn[1], nn[0])
    X = np.meshgrid(*[prob.centers(d) for d in (2, 1, 0)], indexing="ij")

    def field(amp_noise):
        ph = rng.uniform(0, 2 * np.pi, size=3)
        f = sum(np.sin(2 * np.pi * X[2 - d] * (1 + d) + ph[d]) for d in range(ndim)) / ndim
        if rough:
            f = f + amp_noise * rng.uniform(-1, 1, size=shp)
            f = f + 0.7 * (rng.uniform(size=shp) < 0.02)  # isolated spikes
            f = f + 0.5 * np.sign(np.sin(2 * np.pi * (X[2] + 0.13)))  # a jump in x
        return f

    zs = [field(0.2) for _ in range(nf)]
    e = [np.exp(1.5 * z) for z in zs]
    tot = sum(e)
    alpha = [np.clip(ei / tot, 1e-6, 1.0) for ei in e]
    if nf > 1:
        alpha[-1] = 1.0 - sum(alpha[:-1])
    else:
        alpha = [np.ones(shp)]
    rho0 = [1000.0, 1.2, 0.6][:nf]
    rho_i = [r * (1.0 + 0.1 * field(0.05)) for r in rho0]
    vel = [30.0 * field(0.3) for _ in range(ndim)]
    p = 1.0e5 * np.exp(0.8 * field(0.1))
    q = assemble(prob, alpha, rho_i, vel, p)
    return prob, q


CONFIGS = {0: cfg0, 1: cfg1, 2: cfg2, 3: cfg3, 4: cfg4}
