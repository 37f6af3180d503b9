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


def row_scales(prob, ref_int: np.ndarray, alpha_floor: float = 0.0) -> np.ndarray:
    """S_k = max |ref_k| over the interior; the D momentum rows share one scale (a transverse momentum RHS can be
    pure cancellation noise); alpha rows are floored (an alpha RHS can vanish identically)."""
    nf, D = prob.nf, prob.ndim
    S = np.array([np.max(np.abs(ref_int[k])) for k in range(prob.neq)])
    S[nf:nf + D] = S[nf:nf + D].max()
    for k in range(nf + D + 1, prob.neq):
        S[k] = max(S[k], alpha_floor)
    return S


def parity_errors(prob, got: np.ndarray, ref: np.ndarray, alpha_floor: float = 0.0) -> np.ndarray:
    """max_cells |got_k - ref_k| / S_k per equation, interior cells only."""
    it = prob.interior()
    g, r = got[it], ref[it]
    assert np.all(np.isfinite(g)), "non-finite values in the GPU result"
    S = row_scales(prob, r, alpha_floor)
    err = np.zeros(prob.neq)
    for k in range(prob.neq):
        d = np.max(np.abs(g[k] - r[k]))
        err[k] = 0.0 if d == 0.0 else (np.inf if S[k] == 0.0 else d / S[k])
    return err
