"""Thin ctypes binding of libmfc_b200.so (include/mfc.h): same names, argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI.  Device buffers are plain integer
addresses (e.g. ``tensor.data_ptr()``); streams are ``cudaStream_t`` handles as integers
(``torch.cuda.current_stream().cuda_stream``).  There is no CPU fallback: a missing library raises
``MfcLibraryError`` and a missing device makes ``mfc_init`` fail with ``MFC_ECUDA``.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "libmfc_b200.so"

MFC_NG = 3
MFC_ABI_VERSION = 3   # of include/mfc.h as this binding marshals it; checked against the library when it is loaded
MFC_OK, MFC_EINVAL, MFC_EUNSUPPORTED, MFC_ECUDA, MFC_ENOMEM, MFC_ENONFINITE, MFC_ELIMIT = 0, -1, -2, -3, -4, -5, -6
MFC_STATIC_MAX_CELLS = 4096 * 8192   # mfc_cfl_dt_static: most interior cells its fixed workspace serves
MFC_BC_PERIODIC, MFC_BC_EXTRAP, MFC_BC_HALO = 0, 1, 2
MFC_K_RHS, MFC_K_CFL, MFC_K_PRIM, MFC_K_GHOST, MFC_K_COUNT = 0, 1, 2, 3, 4
KERNEL_NAMES = {MFC_K_RHS: "rhs_fused", MFC_K_CFL: "cfl", MFC_K_PRIM: "prim", MFC_K_GHOST: "ghost_fill"}
MFC_STAGING_AUTO, MFC_STAGING_TMA, MFC_STAGING_CPASYNC, MFC_STAGING_ROLES = 0, 1, 2, 3

# every symbol include/mfc.h declares
EXPORTS = [
    "mfc_init", "mfc_destroy", "mfc_layout", "mfc_rhs", "mfc_rk3_step", "mfc_rk3_stage", "mfc_stage_array", "mfc_cfl_dt",
    "mfc_advance_host", "mfc_cfl_dt_static", "mfc_step_cfl",
    "mfc_cons_to_prim", "mfc_line_fluxes", "mfc_profile_enable", "mfc_profile_get", "mfc_launch_count",
    "mfc_probe_dfma", "mfc_strerror", "mfc_version", "mfc_cuda_error", "mfc_abi_version",
]


class MfcLibraryError(RuntimeError):
    pass


class MfcError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {mfc_strerror(code)} ({code})")


class mfc_grid(C.Structure):
    _fields_ = [("ndim", C.c_int), ("n", C.c_int * 3), ("lo", C.c_double * 3), ("hi", C.c_double * 3),
                ("edges_host", C.POINTER(C.c_double) * 3), ("inv_dx", C.c_double * 3)]


class mfc_fluid(C.Structure):
    _fields_ = [("gamma", C.c_double), ("pi_inf", C.c_double)]


class mfc_bc(C.Structure):
    _fields_ = [("lo", C.c_int * 3), ("hi", C.c_int * 3)]


class mfc_opts(C.Structure):
    _fields_ = [("weno_eps", C.c_double), ("cfl", C.c_double), ("device", C.c_int), ("march_segment", C.c_int),
                ("weno_order", C.c_int), ("kapila", C.c_int), ("staging", C.c_int), ("abi_version", C.c_int)]


_lib = None


def lib():
    """Loads the CUDA library; raises if it has not been built (python -m paper_2305_09163_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise MfcLibraryError(f"{LIB_PATH} is missing: build it with `python -m paper_2305_09163_b200.build` "
                              "(nvcc, sm_100a); there is no CPU fallback")
    try:
        L = C.CDLL(str(LIB_PATH))
    except OSError as exc:  # pragma: no cover
        raise MfcLibraryError(f"cannot load {LIB_PATH}: {exc}") from exc
    vp, dp, ip, llp = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int), C.POINTER(C.c_longlong)
    L.mfc_init.argtypes = [C.POINTER(vp), C.POINTER(mfc_grid), C.c_int, C.POINTER(mfc_fluid), C.POINTER(mfc_bc),
                           C.POINTER(mfc_opts)]
    L.mfc_init.restype = C.c_int
    L.mfc_destroy.argtypes = [vp]; L.mfc_destroy.restype = None
    L.mfc_layout.argtypes = [vp, ip, ip, llp, llp]; L.mfc_layout.restype = C.c_int
    L.mfc_rhs.argtypes = [vp, vp, vp, vp]; L.mfc_rhs.restype = C.c_int
    L.mfc_rk3_step.argtypes = [vp, vp, C.c_double, vp]; L.mfc_rk3_step.restype = C.c_int
    L.mfc_cfl_dt.argtypes = [vp, vp, dp, vp]; L.mfc_cfl_dt.restype = C.c_int
    L.mfc_cfl_dt_static.argtypes = [C.POINTER(mfc_grid), C.c_int, C.POINTER(mfc_fluid), C.c_double, C.c_int, vp, vp, vp]
    L.mfc_cfl_dt_static.restype = C.c_int
    L.mfc_step_cfl.argtypes = [vp, vp, dp, vp]; L.mfc_step_cfl.restype = C.c_int
    L.mfc_rk3_stage.argtypes = [vp, C.c_int, vp, C.c_double, vp]; L.mfc_rk3_stage.restype = C.c_int
    L.mfc_stage_array.argtypes = [vp, C.c_int, C.POINTER(vp)]; L.mfc_stage_array.restype = C.c_int
    L.mfc_advance_host.argtypes = [vp, vp, C.c_int, C.c_double, dp, vp]; L.mfc_advance_host.restype = C.c_int
    L.mfc_cons_to_prim.argtypes = [vp, vp, vp, vp]; L.mfc_cons_to_prim.restype = C.c_int
    L.mfc_line_fluxes.argtypes = [vp, C.c_int, C.c_int, vp, vp, vp, vp, vp, vp]; L.mfc_line_fluxes.restype = C.c_int
    L.mfc_profile_enable.argtypes = [vp, C.c_int]; L.mfc_profile_enable.restype = C.c_int
    L.mfc_profile_get.argtypes = [vp, C.c_int, llp, dp, C.c_int]; L.mfc_profile_get.restype = C.c_int
    L.mfc_launch_count.argtypes = [vp]; L.mfc_launch_count.restype = C.c_longlong
    L.mfc_probe_dfma.argtypes = [C.c_int, dp, dp]; L.mfc_probe_dfma.restype = C.c_int
    L.mfc_strerror.argtypes = [C.c_int]; L.mfc_strerror.restype = C.c_char_p
    L.mfc_version.argtypes = []; L.mfc_version.restype = C.c_char_p
    L.mfc_cuda_error.argtypes = [vp]; L.mfc_cuda_error.restype = C.c_char_p
    L.mfc_abi_version.argtypes = []; L.mfc_abi_version.restype = C.c_int
    if L.mfc_abi_version() != MFC_ABI_VERSION:
        raise MfcLibraryError(f"{LIB_PATH} was built with MFC_ABI_VERSION {L.mfc_abi_version()}, this binding marshals "
                              f"version {MFC_ABI_VERSION}: rebuild with `python -m paper_2305_09163_b200.build --force`")
    _lib = L
    return L


def _check(code: int, where: str) -> None:
    if code != MFC_OK:
        raise MfcError(code, where)


def mfc_strerror(code: int) -> str:
    return lib().mfc_strerror(int(code)).decode()


def mfc_version() -> str:
    return lib().mfc_version().decode()


def mfc_init(grid_n, lo, hi, fluids, bc_lo, bc_hi, *, weno_eps=1e-16, cfl=0.3, device=-1, march_segment=0, weno_order=5,
             kapila=False, staging=MFC_STAGING_AUTO, edges=None, inv_dx=None):
    """grid_n / lo / hi: one entry per active dimension; fluids: [(gamma, pi_inf), ...]; edges: per dimension the
    n + 1 cell edges (any sequence of floats) or None for uniform spacing; inv_dx: per dimension the reciprocal cell width
    to use instead of n / (hi - lo) (blocks of a decomposed grid pass the global one), 0 or None for the default;
    returns the context handle."""
    ndim = len(grid_n)
    g = mfc_grid()
    g.ndim = ndim
    b = mfc_bc()
    for d in range(3):
        g.n[d] = int(grid_n[d]) if d < ndim else 1
        g.lo[d] = float(lo[d]) if d < ndim else 0.0
        g.hi[d] = float(hi[d]) if d < ndim else 1.0
        b.lo[d] = int(bc_lo[d]) if d < ndim else MFC_BC_EXTRAP
        b.hi[d] = int(bc_hi[d]) if d < ndim else MFC_BC_EXTRAP
        g.inv_dx[d] = float(inv_dx[d]) if inv_dx is not None and d < ndim and d < len(inv_dx) and inv_dx[d] else 0.0
    keep = []                                    # host edge arrays, alive until mfc_init has copied them
    for d in range(3):
        e = edges[d] if edges is not None and d < ndim and d < len(edges) else None
        if e is None:
            g.edges_host[d] = None
        else:
            arr = (C.c_double * (int(grid_n[d]) + 1))(*[float(v) for v in e])
            keep.append(arr)
            g.edges_host[d] = C.cast(arr, C.POINTER(C.c_double))
    fl = (mfc_fluid * max(1, len(fluids)))()
    for i, (gam, pinf) in enumerate(fluids):
        fl[i].gamma, fl[i].pi_inf = float(gam), float(pinf)
    o = mfc_opts(float(weno_eps), float(cfl), int(device), int(march_segment), int(weno_order), 1 if kapila else 0,
                 int(staging), MFC_ABI_VERSION)
    h = C.c_void_p()
    _check(lib().mfc_init(C.byref(h), C.byref(g), len(fluids), fl, C.byref(b), C.byref(o)), "mfc_init")
    return h


def mfc_destroy(ctx) -> None:
    lib().mfc_destroy(ctx)


def mfc_layout(ctx):
    """-> (neq, ng, (px, py, pz), elems)"""
    neq, ng, el = C.c_int(), C.c_int(), C.c_longlong()
    pn = (C.c_longlong * 3)()
    _check(lib().mfc_layout(ctx, C.byref(neq), C.byref(ng), pn, C.byref(el)), "mfc_layout")
    return neq.value, ng.value, (pn[0], pn[1], pn[2]), el.value


def mfc_cuda_error(ctx) -> str:
    return lib().mfc_cuda_error(ctx).decode()


def _check_ctx(code: int, where: str, ctx) -> None:
    if code in (MFC_ECUDA, MFC_ENOMEM):
        raise MfcError(code, f"{where} [{mfc_cuda_error(ctx)}]")
    _check(code, where)


def mfc_rhs(ctx, q_dev: int, rhs_dev: int, stream: int = 0) -> None:
    _check_ctx(lib().mfc_rhs(ctx, q_dev, rhs_dev, stream), "mfc_rhs", ctx)


def mfc_rk3_step(ctx, q_dev: int, dt: float, stream: int = 0) -> None:
    _check_ctx(lib().mfc_rk3_step(ctx, q_dev, float(dt), stream), "mfc_rk3_step", ctx)


def mfc_rk3_stage(ctx, stage: int, q_dev: int, dt: float, stream: int = 0) -> None:
    _check_ctx(lib().mfc_rk3_stage(ctx, int(stage), q_dev, float(dt), stream), "mfc_rk3_stage", ctx)


def mfc_stage_array(ctx, k: int) -> int:
    """-> device address of the library's stage array q1 (k = 1) or q2 (k = 2)"""
    p = C.c_void_p()
    _check(lib().mfc_stage_array(ctx, int(k), C.byref(p)), "mfc_stage_array")
    return int(p.value)


def mfc_cfl_dt(ctx, q_dev: int, stream: int = 0) -> float:
    dt = C.c_double()
    _check(lib().mfc_cfl_dt(ctx, q_dev, C.byref(dt), stream), "mfc_cfl_dt")
    return dt.value


def mfc_step_cfl(ctx, q_dev: int, stream: int = 0) -> float:
    """One step at the CFL time step of the current state (mfc_cfl_dt + mfc_rk3_step as one call); -> the step taken."""
    dt = C.c_double()
    _check_ctx(lib().mfc_step_cfl(ctx, q_dev, C.byref(dt), stream), "mfc_step_cfl", ctx)
    return dt.value


def mfc_cfl_dt_static(grid_n, lo, hi, fluids, q_dev: int, dt_dev: int, *, cfl: float = 0.3, device: int = -1,
                      stream: int = 0) -> None:
    """The CFL time step without a context and without any allocation by the library, for callers that cannot let a
    library call cudaMalloc (see include/mfc.h).  q_dev: the state; dt_dev: address of ONE device double that the kernel
    writes on `stream` (the call does not wait).  Uniform grids of at most MFC_STATIC_MAX_CELLS interior cells."""
    ndim = len(grid_n)
    g = mfc_grid()
    g.ndim = ndim
    for d in range(3):
        g.n[d] = int(grid_n[d]) if d < ndim else 1
        g.lo[d] = float(lo[d]) if d < ndim else 0.0
        g.hi[d] = float(hi[d]) if d < ndim else 1.0
        g.edges_host[d] = None
        g.inv_dx[d] = 0.0
    fl = (mfc_fluid * max(1, len(fluids)))()
    for i, (gam, pinf) in enumerate(fluids):
        fl[i].gamma, fl[i].pi_inf = float(gam), float(pinf)
    _check(lib().mfc_cfl_dt_static(C.byref(g), len(fluids), fl, float(cfl), int(device), q_dev, dt_dev, stream),
           "mfc_cfl_dt_static")


def mfc_advance_host(ctx, q_host: int, nsteps: int, dt_fixed: float = 0.0, stream: int = 0) -> float:
    t = C.c_double()
    _check(lib().mfc_advance_host(ctx, q_host, int(nsteps), float(dt_fixed), C.byref(t), stream), "mfc_advance_host")
    return t.value


def mfc_cons_to_prim(ctx, q_dev: int, w_dev: int, stream: int = 0) -> None:
    _check(lib().mfc_cons_to_prim(ctx, q_dev, w_dev, stream), "mfc_cons_to_prim")


def mfc_line_fluxes(ctx, direction: int, n: int, w_dev: int, vL_dev: int, vR_dev: int, F_dev: int, uface_dev: int,
                    stream: int = 0) -> None:
    _check(lib().mfc_line_fluxes(ctx, int(direction), int(n), w_dev, vL_dev, vR_dev, F_dev, uface_dev, stream),
           "mfc_line_fluxes")


def mfc_profile_enable(ctx, on: bool) -> None:
    _check(lib().mfc_profile_enable(ctx, 1 if on else 0), "mfc_profile_enable")


def mfc_profile_get(ctx, kernel_id: int, reset: bool = False):
    """-> (launches, total_ms)"""
    n, ms = C.c_longlong(), C.c_double()
    _check(lib().mfc_profile_get(ctx, int(kernel_id), C.byref(n), C.byref(ms), 1 if reset else 0), "mfc_profile_get")
    return n.value, ms.value


def mfc_launch_count(ctx) -> int:
    return int(lib().mfc_launch_count(ctx))


def mfc_probe_dfma(device: int = -1):
    """-> (TFLOP/s, ms) of the register-resident DFMA micro-benchmark"""
    tf, ms = C.c_double(), C.c_double()
    _check(lib().mfc_probe_dfma(int(device), C.byref(tf), C.byref(ms)), "mfc_probe_dfma")
    return tf.value, ms.value


def init_from_problem(prob, **kw):
    """mfc_init from a workloads.Problem-like object (ndim, n, lo, hi, fluids, bc_lo, bc_hi, weno_eps, cfl)."""
    D = prob.ndim
    return mfc_init(prob.n[:D], prob.lo[:D], prob.hi[:D], prob.fluids, prob.bc_lo[:D], prob.bc_hi[:D],
                    weno_eps=prob.weno_eps, cfl=prob.cfl, weno_order=getattr(prob, "weno_order", 5),
                    kapila=getattr(prob, "kapila", False), edges=getattr(prob, "edges", None),
                    inv_dx=getattr(prob, "inv_dx", None), **kw)
