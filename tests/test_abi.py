"""The C-ABI library: builds, loads, exports every symbol include/mfc.h declares, validates arguments before
touching the GPU, and fails loudly (no CPU fallback) when there is no device.  CPU only."""
from __future__ import annotations

import ctypes as C
import re
from pathlib import Path

import pytest

from paper_2305_09163_b200 import binding as B
from paper_2305_09163_b200 import build as mfc_build

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lib():
    mfc_build.build()
    return B.lib()


def declared_symbols():
    text = (ROOT / "include" / "mfc.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mfc_[a-z0-9_]+)\s*\(", text)))


def test_header_and_binding_list_the_same_entry_points():
    assert declared_symbols() == sorted(B.EXPORTS)


def test_library_exports_every_declared_symbol(lib):
    for name in declared_symbols():
        assert hasattr(lib, name), name


def test_north_star_entry_points_present(lib):
    for name in ("mfc_init", "mfc_rhs", "mfc_rk3_step", "mfc_cfl_dt"):
        assert hasattr(lib, name)


def test_strerror_and_version(lib):
    assert B.mfc_strerror(B.MFC_OK) == "ok"
    assert "invalid" in B.mfc_strerror(B.MFC_EINVAL)
    assert "sm_100a" in B.mfc_version()


@pytest.mark.parametrize("kw,code", [
    (dict(grid_n=(2,)), B.MFC_EINVAL),                                   # fewer cells than ghost layers
    (dict(fluids=[(1.0, 0.0)]), B.MFC_EINVAL),                           # gamma <= 1
    (dict(fluids=[(1.4, 0.0)] * 4), B.MFC_EUNSUPPORTED),                 # outside the template set
    (dict(bc_lo=(0,), bc_hi=(1,)), B.MFC_EINVAL),                        # periodic on one side only
    (dict(bc_lo=(7,), bc_hi=(7,)), B.MFC_EINVAL),
    (dict(lo=(1.0,), hi=(1.0,)), B.MFC_EINVAL),
    (dict(weno_order=4), B.MFC_EINVAL),                                   # reconstruction order 1, 3 or 5
    (dict(weno_order=7), B.MFC_EINVAL),
    (dict(fluids=[(1.4, 0.0)], kapila=True), B.MFC_EUNSUPPORTED),         # Eq. 2 is the two-fluid coefficient
    (dict(fluids=[(4.4, 6e8), (1.4, 0.0), (1.33, 0.0)], kapila=True), B.MFC_EUNSUPPORTED),
])
def test_init_rejects_bad_arguments_before_touching_cuda(lib, kw, code):
    args = dict(grid_n=(16,), lo=(0.0,), hi=(1.0,), fluids=[(4.4, 6e8), (1.4, 0.0)], bc_lo=(1,), bc_hi=(1,))
    args.update(kw)
    with pytest.raises(B.MfcError) as ei:
        B.mfc_init(**args)
    assert ei.value.code == code


def test_null_pointers_are_rejected(lib):
    assert lib.mfc_init(None, None, 2, None, None, None) == B.MFC_EINVAL
    assert lib.mfc_rhs(None, None, None, None) == B.MFC_EINVAL
    assert lib.mfc_rk3_step(None, None, 0.1, None) == B.MFC_EINVAL
    assert lib.mfc_cfl_dt(None, None, None, None) == B.MFC_EINVAL
    assert lib.mfc_layout(None, None, None, None, None) == B.MFC_EINVAL
    assert lib.mfc_launch_count(None) == 0
    lib.mfc_destroy(None)


def test_no_cpu_fallback_without_a_device(lib):
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if has_gpu:
        pytest.skip("a CUDA device is present")
    with pytest.raises(B.MfcError) as ei:
        B.mfc_init((16,), (0.0,), (1.0,), [(1.4, 0.0)], (1,), (1,))
    assert ei.value.code == B.MFC_ECUDA


def test_abi_version_of_header_binding_and_library_agree(lib):
    text = (ROOT / "include" / "mfc.h").read_text()
    assert int(re.search(r"#define\s+MFC_ABI_VERSION\s+(\d+)", text).group(1)) == B.MFC_ABI_VERSION == lib.mfc_abi_version()


def test_init_refuses_a_caller_compiled_against_another_abi(lib):
    g, b = B.mfc_grid(), B.mfc_bc()
    g.ndim, g.n[0], g.lo[0], g.hi[0] = 1, 16, 0.0, 1.0
    b.lo[0] = b.hi[0] = B.MFC_BC_EXTRAP
    fl = (B.mfc_fluid * 1)()
    fl[0].gamma, fl[0].pi_inf = 1.4, 0.0
    o = B.mfc_opts()
    o.device, o.abi_version = -1, B.MFC_ABI_VERSION - 1
    h = C.c_void_p()
    assert lib.mfc_init(C.byref(h), C.byref(g), 1, fl, C.byref(b), C.byref(o)) == B.MFC_EINVAL
    assert not h.value


def test_init_rejects_a_bad_reciprocal_width(lib):
    for bad in (-1.0, float("inf"), float("nan")):
        with pytest.raises(B.MfcError) as ei:
            B.mfc_init((16,), (0.0,), (1.0,), [(1.4, 0.0)], (1,), (1,), inv_dx=(bad,))
        assert ei.value.code == B.MFC_EINVAL
