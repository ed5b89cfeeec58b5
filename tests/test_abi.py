"""Host-side checks of the C-ABI boundary (no GPU): libstag.so builds for sm_100a, loads, and
exports every function include/stag.h declares; the binding's signature table names exactly
those functions; the pure-host entry points behave."""
import ctypes
import os
import re

import pytest

import paper_1111_0125_b200 as stag

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "stag.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(stag_[A-Za-z0-9_]+)\s*\(", text)))


def test_header_declares_the_north_star_entry_points():
    names = _declared_functions()
    for must in ("stag_dslash", "stag_apply_A", "stag_cg_solve"):
        assert must in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    path = stag.build()
    assert os.path.exists(path) and path.endswith("libstag.so")
    h = ctypes.CDLL(path)
    for name in _declared_functions():
        assert hasattr(h, name), "libstag.so does not export %s" % name


def test_binding_covers_exactly_the_declared_functions():
    assert sorted(stag.SIGNATURES) == _declared_functions()


def test_library_is_built_for_sm_100a():
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", stag.build()], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_spinor_bytes_and_argument_checks_on_host():
    assert stag.spinor_bytes((4, 4, 4, 4), stag.PREC_F64) == 3 * 128 * 16
    assert stag.spinor_bytes((4, 4, 4, 4), stag.PREC_F32) == 3 * 128 * 8
    assert stag.spinor_bytes((4, 4, 4, 4), stag.PREC_F32_R12) == 3 * 128 * 8
    # Vh = 6*4*2*10/2 = 240 -> padded to 256
    assert stag.spinor_bytes((6, 4, 2, 10), stag.PREC_F64) == 3 * 256 * 16
    assert stag.spinor_bytes((3, 4, 4, 4), stag.PREC_F64) == 0      # odd extent
    assert stag.spinor_bytes((4, 4, 4, 0), stag.PREC_F64) == 0
    assert stag.spinor_bytes((4, 4, 4, 4), 7) == 0                  # bad enum


def test_workspace_bytes_is_pure_arithmetic_on_host():
    """stag_cg_workspace_bytes needs no device: control block + partial-sum
    slots + the vectors of Fig. 1 the mode needs."""
    d = (28, 28, 28, 96)
    sp64, sp32 = stag.spinor_bytes(d, stag.PREC_F64), stag.spinor_bytes(d, stag.PREC_F32)
    w0, w1, w3 = (stag.cg_workspace_bytes(d, m) for m in (stag.CG_F64, stag.CG_F32, stag.CG_RELIABLE))
    fixed = w0 - 7 * sp64           # b_e, 2 staging, r, q, tmp, d in fp64
    assert 0 < fixed < (1 << 20)
    assert w3 == w1 == fixed + 6 * sp64 + 5 * sp32      # no fp64 d; y, r, d, q, tmp in fp32
    assert stag.cg_workspace_bytes(d, stag.CG_DEFECT) == w3
    op = stag.cg_workspace_bytes(d, -1)
    assert fixed - 2 * 256 <= op - sp64 <= fixed        # operator only: one odd-site intermediate
    # right-hand sides scale the vectors, not the fixed part
    w3_4 = stag.cg_workspace_bytes(d, stag.CG_RELIABLE, 4)
    assert 4 * (4 * sp64 + 5 * sp32) + 2 * sp64 <= w3_4 <= 4 * (4 * sp64 + 5 * sp32) + 2 * sp64 + (1 << 20)
    assert stag.cg_workspace_bytes(d, 4) == 0 and stag.cg_workspace_bytes(d, 0, 0) == 0
    assert stag.cg_workspace_bytes(d, 0, stag.MAX_RHS + 1) == 0
    assert stag.cg_workspace_bytes((28, 28, 28, 95), 0) == 0
    # the setter checks its arguments before it touches the device
    assert stag.lib().stag_set_workspace(None, 0) == stag.OK
    assert stag.lib().stag_set_workspace(None, 64) == stag.EINVAL


def test_strerror_and_null_arguments():
    lib = stag.lib()
    assert lib.stag_strerror(0) == b"ok"
    assert b"invalid" in lib.stag_strerror(stag.EINVAL)
    dims = (ctypes.c_int * 4)(4, 4, 4, 4)
    assert lib.stag_dslash(None, None, None, 0, dims, 0) == stag.EINVAL
    assert lib.stag_apply_A(None, None, None, 0.1, 0) == stag.EINVAL
    assert lib.stag_cg_solve(None, None, None, 0.1, 1e-10, 10, 0, None, None) == stag.EINVAL
    h = ctypes.c_void_p()
    assert lib.stag_links_create(ctypes.byref(h), dims, 1, None, 0) == stag.EINVAL
    bad = (ctypes.c_int * 4)(4, 5, 4, 4)
    buf = (ctypes.c_double * 8)()
    assert lib.stag_links_create(ctypes.byref(h), bad, 1, ctypes.cast(buf, ctypes.c_void_p), 0) == stag.EINVAL


def test_compute_entry_points_refuse_to_run_without_cuda(have_cuda):
    if have_cuda:
        pytest.skip("CUDA present")
    with pytest.raises(RuntimeError):
        stag.empty_spinor((4, 4, 4, 4), stag.PREC_F64)
