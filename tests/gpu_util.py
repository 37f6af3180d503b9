"""Helpers of the GPU parity tests: device buffers through torch, calls through the C-ABI binding, and the
parity norm of DESIGN.md ("Parity norm").  Nothing of the method is computed here."""
from __future__ import annotations

import numpy as np

from paper_2305_09163_b200 import binding as B


def torch_mod():
    import torch
    return torch


class Gpu:
    """One mfc context plus the torch plumbing (device memory, stream)."""

    def __init__(self, prob, **kw):
        torch = torch_mod()
        from paper_2305_09163_b200 import build
        build.build()
        self.torch = torch
        self.prob = prob
        self.dev = torch.device("cuda", torch.cuda.current_device())
        self.ctx = B.init_from_problem(prob, **kw)
        self.neq, self.ng, self.padded, self.elems = B.mfc_layout(self.ctx)

    def close(self):
        if self.ctx is not None:
            B.mfc_destroy(self.ctx)
            self.ctx = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    @property
    def stream(self) -> int:
        return self.torch.cuda.current_stream().cuda_stream

    def to_dev(self, a: np.ndarray):
        return self.torch.from_numpy(np.ascontiguousarray(a)).to(self.dev)

    def rhs(self, q: np.ndarray) -> np.ndarray:
        qd = self.to_dev(q)
        out = self.torch.full_like(qd, float("nan"))
        B.mfc_rhs(self.ctx, qd.data_ptr(), out.data_ptr(), self.stream)
        self.torch.cuda.synchronize()
        return out.cpu().numpy()

    def prim(self, q: np.ndarray) -> np.ndarray:
        qd = self.to_dev(q)
        out = self.torch.full_like(qd, float("nan"))
        B.mfc_cons_to_prim(self.ctx, qd.data_ptr(), out.data_ptr(), self.stream)
        self.torch.cuda.synchronize()
        return out.cpu().numpy()

    def rk3(self, q: np.ndarray, dts) -> np.ndarray:
        qd = self.to_dev(q)
        for dt in dts:
            B.mfc_rk3_step(self.ctx, qd.data_ptr(), float(dt), self.stream)
        self.torch.cuda.synchronize()
        return qd.cpu().numpy()

    def cfl_dt(self, q: np.ndarray) -> float:
        qd = self.to_dev(q)
        return B.mfc_cfl_dt(self.ctx, qd.data_ptr(), self.stream)

    def line(self, direction: int, w: np.ndarray):
        torch = self.torch
        n = w.shape[1] - 2 * B.MFC_NG
        wd = self.to_dev(w)
        mk = lambda *s: torch.full(s, float("nan"), dtype=torch.float64, device=self.dev)
        vL, vR, F, uf = mk(self.neq, n + 2), mk(self.neq, n + 2), mk(self.neq, n + 1), mk(n + 1)
        B.mfc_line_fluxes(self.ctx, direction, n, wd.data_ptr(), vL.data_ptr(), vR.data_ptr(), F.data_ptr(), uf.data_ptr(),
                          self.stream)
        torch.cuda.synchronize()
        return vL.cpu().numpy(), vR.cpu().numpy(), F.cpu().numpy(), uf.cpu().numpy()


EPS_MACH = 2.0 ** -52
RHS_TOL = 1.0e-10
ROUNDOFF_K = 12.0          # "a few ulp": measured, tests/test_parity_norm.py (two CPU builds: <= 2.2) and the GPU suite (<= 3.8)


def rhs_floors(prob, orc, q: np.ndarray) -> np.ndarray:
    """Round-off floors of the per-equation RHS scales, from oracle quantities only.

    Two correct fp64 evaluations of one face flux differ by a few ulp of every reconstructed state.  The face
    velocity u_face is built from u -/+ c and p/(rho c), so it carries an absolute error of a few eps * lam,
    lam = max(|u| + c), however small u_face itself is.  Each flux row inherits it at its own flux scale
        alpha_i rho_i : max(alpha_i rho_i) lam       alpha_i : max(alpha_i) lam
        rho u_d       : max|p| + max(rho) lam max|u| (acoustic coupling rho c du)
        rho E         : max|E + p| lam
    and the RHS at that scale / dx, whatever the magnitude of the RHS itself (which can vanish identically: a
    quiescent bubble, a transverse momentum row).  S_k is floored at K eps / tol times that scale, K = 12, so
    that `tol relative` never asks for less than K ulp of the flux terms that cancel.
    """
    it = prob.interior()
    w = orc.cons_to_prim(q)[it]
    nf, D = prob.nf, prob.ndim
    dxmin = min(float(np.min(prob.widths(d))) for d in range(D))
    dxmax = max(float(np.max(prob.widths(d))) for d in range(D))
    lam = dxmax / orc.cfl_dt(q, 1.0)                           # >= max_d max_cells (|u_d| + c)
    rho = w[:nf].sum(axis=0)
    umax = max(float(np.max(np.abs(w[nf + d]))) for d in range(D))
    pmax = float(np.max(np.abs(w[nf + D])))
    F = np.zeros(prob.neq)
    for i in range(nf):
        F[i] = float(np.max(np.abs(w[i]))) * lam
    F[nf:nf + D] = pmax + float(rho.max()) * lam * umax
    F[nf + D] = float(np.max(np.abs(q[it][nf + D]) + np.abs(w[nf + D]))) * lam
    for k in range(nf + D + 1, prob.neq):
        F[k] = float(np.max(np.abs(w[k]))) * lam
    return ROUNDOFF_K * EPS_MACH / RHS_TOL * F / dxmin


def row_scales(prob, ref_int: np.ndarray, floors=None) -> np.ndarray:
    """S_k = max(max |ref_k| over the interior, floor_k); the D momentum rows share one scale (a transverse
    momentum RHS can be pure cancellation noise)."""
    nf, D = prob.nf, prob.ndim
    S = np.array([np.max(np.abs(ref_int[k])) for k in range(prob.neq)])
    S[nf:nf + D] = S[nf:nf + D].max()
    if floors is not None:
        S = np.maximum(S, floors)
    return S


def _ratio(d: float, s: float) -> float:
    return 0.0 if d == 0.0 else (np.inf if s == 0.0 else d / s)


def parity_errors(prob, got: np.ndarray, ref: np.ndarray, floors=None) -> np.ndarray:
    """max_cells |got_k - ref_k| / S_k per equation, interior cells only."""
    it = prob.interior()
    g, r = got[it], ref[it]
    assert np.all(np.isfinite(g)), "non-finite values in the GPU result"
    S = row_scales(prob, r, floors)
    return np.array([_ratio(float(np.max(np.abs(g[k] - r[k]))), S[k]) for k in range(prob.neq)])


def parity_report(prob, got: np.ndarray, ref: np.ndarray, floors: np.ndarray):
    """The RHS parity error three ways, per equation: with the round-off floors (the asserted norm), WITHOUT them
    (SURVEY.md 8(c)-D read literally: S_k = max |oracle_k|) and in units of eps_mach * (flux scale) / dx, i.e. in
    "ulp of the terms that cancel" -- the quantity the floor bounds at ROUNDOFF_K."""
    it = prob.interior()
    g, r = got[it], ref[it]
    assert np.all(np.isfinite(g)), "non-finite values in the GPU result"
    d = np.array([float(np.max(np.abs(g[k] - r[k]))) for k in range(prob.neq)])
    S0, S = row_scales(prob, r), row_scales(prob, r, floors)
    floored = np.array([_ratio(d[k], S[k]) for k in range(prob.neq)])
    unfloored = np.array([_ratio(d[k], S0[k]) for k in range(prob.neq)])
    ulps = d / (floors * RHS_TOL / ROUNDOFF_K)            # floors = K eps / tol * Phi / dx
    return floored, unfloored, ulps
