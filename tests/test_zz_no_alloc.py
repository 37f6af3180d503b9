"""mfc_cfl_dt_static: the CFL time step for callers that cannot let the library allocate device memory.

Who needs it: code that lives inside an application whose memory pool already owns the whole device (one more
cudaMalloc fails, or takes what the application had budgeted), time loops that keep other streams busy (cudaMalloc and
cudaFree stall the entire device), and plug-ins that are handed buffers plus a stream and may only enqueue work.  None
of them can call mfc_init, which allocates the stage arrays and the reduction workspace; this entry point takes no
context and keeps its workspace in a fixed array inside the library (include/mfc.h states the size and the limit).

What is checked: for the same grid, fluids, CFL number and state, the entry point returns what the context path
(mfc_init + mfc_cfl_dt) returns, within the 1e-13 relative tolerance the CFL parity tests use (the bits are in fact
equal), on two calls in a row -- the second on a different, slower state, so that anything the first call left in the
shared workspace (its partial maxima, its ticket count) would show up as a wrong, too small time step.  The buffers the
entry point works on are allocated here, by the test, as a caller's would be.

This file is named so that pytest collects it last: under `pytest -x` a failure here hides no other test.  It does not
depend on anything the other tests leave behind and passes alone in a fresh process.
"""
from __future__ import annotations

import numpy as np
import pytest

from paper_2305_09163_b200 import binding as B
from paper_2305_09163_b200 import build as mfc_build
from paper_2305_09163_b200 import workloads as wl

REL_TOL = 1.0e-13   # the tolerance of test_cfl_dt_parity (tests/test_gpu_parity.py)

# (ndim, sizes, fluids): one block only (1D), several blocks with a ragged last one, and the 3D template with three fluids;
# 67 * 29 * 41 = 79 663 cells = 19 blocks of 4096 + 1 839
CASES = [(1, (1201,), 2), (2, (301, 45), 1), (3, (67, 29, 41), 2), (3, (40, 33, 21), 3)]


def _static_dt(torch, prob, qd, out, cfl):
    D = prob.ndim
    B.mfc_cfl_dt_static(prob.n[:D], prob.lo[:D], prob.hi[:D], prob.fluids, qd.data_ptr(), out.data_ptr(), cfl=cfl,
                        stream=torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return float(out.cpu()[0])


@pytest.mark.gpu
@pytest.mark.parametrize("ndim,n,nf", CASES)
def test_static_entry_point_matches_the_context_path_on_two_calls_in_a_row(ndim, n, nf):
    import torch

    mfc_build.build()
    prob, q_fast = wl.random_state(ndim, n, nf, seed=11, periodic=True)
    # second state: the same fields at rest -- every signal speed drops, so dt must GROW on the second call; stale partial
    # maxima of the first call would keep it at the first value
    it = prob.interior()
    q_slow = q_fast.copy()
    rho = q_slow[it][:nf].sum(axis=0)
    mom = q_slow[it][nf:nf + ndim]
    q_slow[it][nf + ndim] -= 0.5 * (mom ** 2).sum(axis=0) / rho      # kinetic energy out of rho E
    q_slow[it][nf:nf + ndim] = 0.0
    dev = torch.device("cuda", torch.cuda.current_device())
    stream = torch.cuda.current_stream().cuda_stream
    ctx = B.init_from_problem(prob)
    try:
        out = torch.full((1,), float("nan"), dtype=torch.float64, device=dev)      # the caller's result buffer
        refs, gots = [], []
        for q in (q_fast, q_slow):
            qd = torch.from_numpy(q).to(dev)                                        # the caller's state
            refs.append(B.mfc_cfl_dt(ctx, qd.data_ptr(), stream))
            gots.append(_static_dt(torch, prob, qd, out, prob.cfl))
    finally:
        B.mfc_destroy(ctx)
    for ref, got in zip(refs, gots):
        assert np.isfinite(ref) and ref > 0.0
        assert abs(got - ref) <= REL_TOL * ref, (got, ref)
    assert refs[1] > refs[0] and gots[1] > gots[0]


@pytest.mark.gpu
def test_static_entry_point_keeps_nan_like_the_context_path():
    import torch

    mfc_build.build()
    prob, q = wl.random_state(3, (20, 12, 9), 2, seed=4, periodic=True)
    q[prob.interior()][prob.nf + prob.ndim][3, 5, 7] = np.nan
    dev = torch.device("cuda", torch.cuda.current_device())
    out = torch.zeros((1,), dtype=torch.float64, device=dev)
    assert np.isnan(_static_dt(torch, prob, torch.from_numpy(q).to(dev), out, prob.cfl))


def test_static_entry_point_refuses_what_its_workspace_cannot_serve():
    """Argument checks run before the first CUDA call, so they are testable without a device."""
    mfc_build.build()
    water_air = [(4.4, 6.0e8), (1.4, 0.0)]
    one = 8   # a non-null address; never dereferenced by a refused call
    with pytest.raises(B.MfcError) as ei:      # 384^3 = 56.6 M cells > MFC_STATIC_MAX_CELLS
        B.mfc_cfl_dt_static((384, 384, 384), (0.0,) * 3, (1.0,) * 3, water_air, one, one)
    assert ei.value.code == B.MFC_ELIMIT
    assert "MFC_STATIC_MAX_CELLS" in str(ei.value)
    with pytest.raises(B.MfcError) as ei:      # one cell past the limit in 1D
        B.mfc_cfl_dt_static((B.MFC_STATIC_MAX_CELLS + 1,), (0.0,), (1.0,), water_air, one, one)
    assert ei.value.code == B.MFC_ELIMIT
    with pytest.raises(B.MfcError) as ei:      # null state
        B.mfc_cfl_dt_static((64,), (0.0,), (1.0,), water_air, 0, one)
    assert ei.value.code == B.MFC_EINVAL
    with pytest.raises(B.MfcError) as ei:      # gamma <= 1
        B.mfc_cfl_dt_static((64,), (0.0,), (1.0,), [(1.0, 0.0)], one, one)
    assert ei.value.code == B.MFC_EINVAL
    # non-uniform spacing is a context feature
    g = B.mfc_grid()
    g.ndim, g.n[0], g.lo[0], g.hi[0] = 1, 8, 0.0, 1.0
    import ctypes as C
    edges = (C.c_double * 9)(*np.linspace(0.0, 1.0, 9))
    g.edges_host[0] = C.cast(edges, C.POINTER(C.c_double))
    fl = (B.mfc_fluid * 1)()
    fl[0].gamma, fl[0].pi_inf = 1.4, 0.0
    assert B.lib().mfc_cfl_dt_static(C.byref(g), 1, fl, 0.3, -1, one, one, None) == B.MFC_EUNSUPPORTED
