"""CPU oracle (TEST INFRASTRUCTURE, not the product).

ctypes front end of oracle/mfc_oracle.c.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It imports nothing from the CUDA
package; it takes a plain description of the problem (any object with the attributes ndim, n, dx,
fluids, bc_lo, bc_hi, weno_eps) and numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "mfc_oracle.c"
_LIB = _HERE / "libmfc_oracle.so"
NG = 3
MAXF = 4


class _Problem(C.Structure):
    _fields_ = [
        ("ndim", C.c_int),
        ("nf", C.c_int),
        ("n", C.c_int * 3),
        ("dx", C.c_double * 3),
        ("gamma", C.c_double * MAXF),
        ("pi_inf", C.c_double * MAXF),
        ("bc_lo", C.c_int * 3),
        ("bc_hi", C.c_int * 3),
        ("weno_eps", C.c_double),
        ("weno_order", C.c_int),
        ("kapila", C.c_int),
        ("xe", C.POINTER(C.c_double) * 3),
    ]


def padded_edges(edges, bc_lo: int, bc_hi: int) -> np.ndarray:
    """Cell edges of the padded line from the n + 1 edges of the interior cells (non-uniform spacing).

    A ghost cell has the width of the cell its value is copied from (reading B20b; the paper is silent):
    periodic -> the widths wrap around; extrapolation -> the boundary cell's width repeated."""
    e = np.asarray(edges, dtype=np.float64)
    w = np.diff(e)
    assert e.ndim == 1 and e.size >= NG + 1 and np.all(w > 0.0), "edges must increase"
    lo = w[-NG:] if bc_lo == 0 else np.full(NG, w[0])
    hi = w[:NG] if bc_hi == 0 else np.full(NG, w[-1])
    left = e[0] - np.cumsum(lo[::-1])[::-1]
    right = e[-1] + np.cumsum(hi)
    return np.ascontiguousarray(np.concatenate([left, e, right]))


STRICT_FLAGS = ["-O2", "-ffp-contract=off"]


def _compile(target: Path, float_flags, force: bool = False) -> Path:
    if force or not target.exists() or target.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = target.with_suffix(f".so.tmp{os.getpid()}")
        cmd = ["gcc"] + list(float_flags) + ["-fopenmp", "-shared", "-fPIC", "-std=c99", str(_SRC), "-o", str(tmp), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, target)
    return target


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (-O2, no FMA contraction, OpenMP on the outer loops only)."""
    return _compile(_LIB, STRICT_FLAGS, force)


def variant_flags():
    """Floating-point flags of the SECOND build of the same source (tests/test_parity_norm.py): another correct
    fp64 evaluation of the same formulas, used to measure how far two correct evaluations differ.  With FMA
    hardware: contraction of every a*b+c (what nvcc does by default); without: reassociation and reciprocals."""
    try:
        with open("/proc/cpuinfo") as f:
            has_fma = " fma " in f.read()
    except OSError:
        has_fma = False
    if has_fma:
        return ["-O2", "-ffp-contract=fast", "-mfma"], "fma"
    return ["-O2", "-fassociative-math", "-fno-signed-zeros", "-fno-trapping-math", "-freciprocal-math"], "reassoc"


def build_variant(force: bool = False):
    flags, tag = variant_flags()
    return _compile(_HERE / f"libmfc_oracle_{tag}.so", flags, force), tag


_libs = {}


def lib(path: Path | None = None):
    """The strict build (default) or, with `path`, another build of the same source (build_variant)."""
    key = str(path) if path is not None else ""
    if key not in _libs:
        if path is None:
            build()
        L = C.CDLL(str(path if path is not None else _LIB))
        dp = C.POINTER(C.c_double)
        pp = C.POINTER(_Problem)
        L.orc_neq.argtypes = [pp]; L.orc_neq.restype = C.c_int
        L.orc_elems.argtypes = [pp]; L.orc_elems.restype = C.c_longlong
        L.orc_fill_ghosts.argtypes = [pp, dp]; L.orc_fill_ghosts.restype = None
        L.orc_cons_to_prim.argtypes = [pp, dp, dp]; L.orc_cons_to_prim.restype = None
        L.orc_cons_to_prim_cell.argtypes = [pp, dp, dp]; L.orc_cons_to_prim_cell.restype = None
        L.orc_weno5.argtypes = [C.c_double] * 6 + [dp, dp]; L.orc_weno5.restype = None
        L.orc_hllc.argtypes = [pp, C.c_int, dp, dp, dp, dp]; L.orc_hllc.restype = None
        L.orc_line.argtypes = [pp, C.c_int, C.c_int, dp, dp, dp, dp, dp]; L.orc_line.restype = None
        L.orc_rhs.argtypes = [pp, dp, dp]; L.orc_rhs.restype = None
        L.orc_rk3_step.argtypes = [pp, dp, C.c_double]; L.orc_rk3_step.restype = None
        L.orc_cfl_dt.argtypes = [pp, dp, C.c_double]; L.orc_cfl_dt.restype = C.c_double
        L.orc_weno3.argtypes = [C.c_double] * 4 + [dp, dp]; L.orc_weno3.restype = None
        L.orc_weno5_nonuniform.argtypes = [dp, dp, C.c_double, dp, dp]; L.orc_weno5_nonuniform.restype = None
        L.orc_kapila_K.argtypes = [pp, C.c_double, C.c_double]; L.orc_kapila_K.restype = C.c_double
        L.orc_threads.argtypes = []; L.orc_threads.restype = C.c_int
        L.orc_set_threads.argtypes = [C.c_int]; L.orc_set_threads.restype = None
        _libs[key] = L
    return _libs[key]


def _dp(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.POINTER(C.c_double))


class Oracle:
    """The oracle bound to one problem description."""

    def __init__(self, prob, lib_path: Path | None = None):
        self.L = lib(lib_path)
        P = _Problem()
        P.ndim = int(prob.ndim)
        P.nf = len(prob.fluids)
        assert 1 <= P.nf <= MAXF
        for d in range(3):
            P.n[d] = int(prob.n[d]) if d < prob.ndim else 1
            P.dx[d] = float(prob.dx[d])
            P.bc_lo[d] = int(prob.bc_lo[d])
            P.bc_hi[d] = int(prob.bc_hi[d])
        for i, (g, pinf) in enumerate(prob.fluids):
            P.gamma[i] = float(g)
            P.pi_inf[i] = float(pinf)
        P.weno_eps = float(prob.weno_eps)
        P.weno_order = int(getattr(prob, "weno_order", 5))
        assert P.weno_order in (1, 3, 5)
        P.kapila = 1 if getattr(prob, "kapila", False) else 0
        assert not P.kapila or P.nf == 2, "the Kapila coefficient of Eq. 2 is the two-fluid one"
        # non-uniform Cartesian spacing: prob.edges[d] = the n[d] + 1 edges of the interior cells, or None
        self.xe = [None, None, None]
        edges = getattr(prob, "edges", None)
        for d in range(3):
            P.xe[d] = None
            if edges is not None and d < prob.ndim and edges[d] is not None:
                assert P.weno_order in (1, 5), "non-uniform spacing: WENO5 (or first order) only"
                assert len(edges[d]) == P.n[d] + 1
                self.xe[d] = padded_edges(edges[d], P.bc_lo[d], P.bc_hi[d])
                P.xe[d] = self.xe[d].ctypes.data_as(C.POINTER(C.c_double))
        self.P = P
        self.neq = self.L.orc_neq(C.byref(P))
        self.elems = self.L.orc_elems(C.byref(P))
        self.ndim = P.ndim
        self.nf = P.nf

    def kapila_K(self, alpha1: float, p: float) -> float:
        """K of PAPER.md Eq. 2 at one state (two fluids)."""
        return float(self.L.orc_kapila_K(C.byref(self.P), float(alpha1), float(p)))

    # -- whole-array operations (q is [neq, pz, py, px], modified in place where noted) --
    def fill_ghosts(self, q: np.ndarray) -> None:
        assert q.size == self.elems
        self.L.orc_fill_ghosts(C.byref(self.P), _dp(q))

    def cons_to_prim(self, q: np.ndarray) -> np.ndarray:
        assert q.size == self.elems
        w = np.empty_like(q)
        self.L.orc_cons_to_prim(C.byref(self.P), _dp(q), _dp(w))
        return w

    def rhs(self, q: np.ndarray) -> np.ndarray:
        """Returns L(q); fills q's ghost cells in place (as the C-ABI's mfc_rhs does)."""
        assert q.size == self.elems
        out = np.zeros_like(q)
        self.L.orc_rhs(C.byref(self.P), _dp(q), _dp(out))
        return out

    def rk3_step(self, q: np.ndarray, dt: float) -> None:
        assert q.size == self.elems
        self.L.orc_rk3_step(C.byref(self.P), _dp(q), float(dt))

    def cfl_dt(self, q: np.ndarray, cfl: float) -> float:
        assert q.size == self.elems
        return float(self.L.orc_cfl_dt(C.byref(self.P), _dp(q), float(cfl)))

    # -- pieces, for pins --
    def cons_to_prim_cell(self, qc) -> np.ndarray:
        qc = np.ascontiguousarray(qc, dtype=np.float64)
        w = np.empty(self.neq)
        self.L.orc_cons_to_prim_cell(C.byref(self.P), _dp(qc), _dp(w))
        return w

    def hllc(self, direction: int, wL, wR):
        wL = np.ascontiguousarray(wL, dtype=np.float64)
        wR = np.ascontiguousarray(wR, dtype=np.float64)
        F = np.empty(self.neq)
        u = np.empty(1)
        self.L.orc_hllc(C.byref(self.P), int(direction), _dp(wL), _dp(wR), _dp(F), _dp(u))
        return F, float(u[0])

    def line(self, direction: int, w: np.ndarray):
        """w: [neq, n + 6] primitives on one line -> vL, vR [neq, n+2], F [neq, n+1], uf [n+1]."""
        w = np.ascontiguousarray(w, dtype=np.float64)
        n = w.shape[1] - 2 * NG
        vL = np.empty((self.neq, n + 2)); vR = np.empty((self.neq, n + 2))
        F = np.empty((self.neq, n + 1)); uf = np.empty(n + 1)
        self.L.orc_line(C.byref(self.P), int(direction), n, _dp(w), _dp(vL), _dp(vR), _dp(F), _dp(uf))
        return vL, vR, F, uf


def weno5(a, b, c, d, e, eps=1e-16):
    vL = C.c_double()
    vR = C.c_double()
    lib().orc_weno5(float(a), float(b), float(c), float(d), float(e), float(eps), C.byref(vL), C.byref(vR))
    return vL.value, vR.value


def weno5_nonuniform(xe, v, eps=1e-16):
    """xe: the six edges of cells i-2..i+2, v: their five values -> (vL at x_{i+1/2}, vR at x_{i-1/2})."""
    xe = np.ascontiguousarray(xe, dtype=np.float64)
    v = np.ascontiguousarray(v, dtype=np.float64)
    assert xe.size == 6 and v.size == 5
    vL = C.c_double()
    vR = C.c_double()
    lib().orc_weno5_nonuniform(_dp(xe), _dp(v), float(eps), C.byref(vL), C.byref(vR))
    return vL.value, vR.value


def weno3(b, c, d, eps=1e-16):
    vL = C.c_double()
    vR = C.c_double()
    lib().orc_weno3(float(b), float(c), float(d), float(eps), C.byref(vL), C.byref(vR))
    return vL.value, vR.value


def threads() -> int:
    return int(lib().orc_threads())


def set_threads(n: int) -> None:
    lib().orc_set_threads(int(n))
