"""stag_apply_A_noalloc: the operator A = m^2 - D_eo D_oe (eq. 2.3) for callers that cannot
allocate device memory -- a program whose own pool owns the whole device (a cudaMalloc inside a
library fails there), code that runs where cudaMalloc / cudaFree are banned because they stall
every stream, or a caller that only holds the spinors it was given.  The odd-site intermediate
lives in an 8 MiB array inside the library image instead of a workspace (include/stag.h).

What is checked: the entry point writes, bit for bit, what stag_apply_A writes (it launches the
same two kernels), on two calls in a row with DIFFERENT inputs -- the second call finds the
first one's intermediate still in the shared array and must not be affected by it -- and it also
meets the oracle at the tolerances the other operator tests use.  Its refusals (lattice too
large for the array, link form not built yet, aliased output) launch nothing and say why.

This file is named to be collected last: pytest -x stops at the first failure, and a failure here
must not hide the rest of the suite.  It passes alone in a fresh process (the first call does the
per-device address lookup) and after the other tests (which leave the array unused).
"""
import ctypes

import numpy as np
import pytest

import fieldgen
import oracle
import paper_1111_0125_b200 as stag
from tests.parity import rel_err

pytestmark = pytest.mark.gpu

TOL = {stag.PREC_F64: 1e-13, stag.PREC_F32: 2e-6, stag.PREC_F64_R12: 1e-13, stag.PREC_F32_R12: 2e-6}


def _raw(v):
    import torch
    return v.view(torch.uint8).cpu().numpy()


@pytest.mark.parametrize("prec", sorted(TOL))
@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (6, 4, 2, 10)])      # Vh = 2048; Vh = 240 -> 16 pad lanes
def test_noalloc_equals_apply_A_on_two_calls_in_a_row(dims, prec):
    import torch
    m = 0.05
    W = fieldgen.links(dims, "random", seed=11)
    L = stag.Links(dims, W)
    chi1 = fieldgen.spinor_gaussian(dims, 0, seed=21)
    chi2 = fieldgen.spinor_gaussian(dims, 0, seed=22)
    v1, v2 = stag.spinor_pack(chi1, dims, prec), stag.spinor_pack(chi2, dims, prec)
    # the existing path; it also builds the links of `prec`, which the new entry point will not do
    ref1, ref2 = stag.apply_A(v1, L, m, prec), stag.apply_A(v2, L, m, prec)
    out1 = torch.full_like(v1, float("nan"))
    out2 = torch.full_like(v2, float("nan"))
    stag.apply_A_noalloc(v1, out1, L, m, prec)
    stag.apply_A_noalloc(v2, out2, L, m, prec)        # straight after, same stream, stale scratch
    torch.cuda.synchronize()
    assert np.array_equal(_raw(out1), _raw(ref1))
    assert np.array_equal(_raw(out2), _raw(ref2))
    # and against the oracle, at the tolerance of tests/test_gpu_dslash.py
    for chi, out in ((chi1, out1), (chi2, out2)):
        got = stag.spinor_unpack(out, dims, prec)
        assert rel_err(got, oracle.apply_A(chi, W, dims, m)) <= TOL[prec]
    # a third call with the first input again: what call two left behind changes nothing
    out3 = torch.full_like(v1, float("nan"))
    stag.apply_A_noalloc(v1, out3, L, m, prec)
    torch.cuda.synchronize()
    assert np.array_equal(_raw(out3), _raw(ref1))
    L.close()


def test_noalloc_at_the_largest_baseline_lattice_that_fits():
    """16^3 x 32 (BASELINE configs[2]): 3 MiB of fp64 intermediate, several hundred tiles."""
    import torch
    cfg = fieldgen.CONFIGS["c3_16^3x32"]
    W, b = cfg.links(), cfg.source()
    L = stag.Links(cfg.dims, W)
    refA = oracle.apply_A(b, W, cfg.dims, cfg.mass)
    for prec in (stag.PREC_F64, stag.PREC_F32_R12):
        v = stag.spinor_pack(b, cfg.dims, prec)
        ref = stag.apply_A(v, L, cfg.mass, prec)
        for _ in range(2):
            out = torch.full_like(v, float("nan"))
            stag.apply_A_noalloc(v, out, L, cfg.mass, prec)
            torch.cuda.synchronize()
            assert np.array_equal(_raw(out), _raw(ref))
        assert rel_err(stag.spinor_unpack(out, cfg.dims, prec), refA) <= TOL[prec]
    L.close()


def test_noalloc_refuses_what_it_cannot_do_without_allocating():
    import torch
    dims = (4, 4, 4, 4)
    L = stag.Links(dims, fieldgen.links(dims, "random", seed=3))
    chi = fieldgen.spinor_gaussian(dims, 0, seed=4)
    # links of fp32/12 do not exist on a fresh handle and building them would allocate
    v = stag.spinor_pack(chi, dims, stag.PREC_F32_R12)
    out = torch.zeros_like(v)
    with pytest.raises(stag.StagError) as e:
        stag.apply_A_noalloc(v, out, L, 0.1, stag.PREC_F32_R12)
    assert e.value.status == stag.EINVAL and "not built" in str(e.value)
    assert not out.any()                                   # nothing was launched
    stag.apply_A(v, L, 0.1, stag.PREC_F32_R12)             # set-up: an ordinary call builds them
    stag.apply_A_noalloc(v, out, L, 0.1, stag.PREC_F32_R12)
    assert out.any()
    # out must not alias in; null pointers
    with pytest.raises(stag.StagError):
        stag.apply_A_noalloc(v, v, L, 0.1, stag.PREC_F32_R12)
    assert stag.lib().stag_apply_A_noalloc(None, None, None, 0.1, 0) == stag.EINVAL
    L.close()

    # a lattice whose fp64 intermediate (10.1 MiB) is beyond the 8 MiB array: refused in fp64 with
    # both sizes in the text, accepted in fp32 (5.1 MiB)
    big = (24, 24, 24, 32)
    vh = 24 * 24 * 24 * 32 // 2
    assert 3 * vh * 16 > stag.NOALLOC_SCRATCH_BYTES >= 3 * vh * 8
    Wb = np.broadcast_to(np.eye(3, dtype=np.complex128), (4, 2, vh, 3, 3))
    Lb = stag.Links(big, Wb)
    x64 = stag.empty_spinor(big, stag.PREC_F64).zero_()
    o64 = torch.zeros_like(x64)
    with pytest.raises(stag.StagError) as e:
        stag.apply_A_noalloc(x64, o64, Lb, 0.1, stag.PREC_F64)
    assert e.value.status == stag.EINVAL
    assert str(3 * vh * 16) in str(e.value) and str(stag.NOALLOC_SCRATCH_BYTES) in str(e.value)
    x32 = stag.empty_spinor(big, stag.PREC_F32).fill_(1.0)
    ref = stag.apply_A(x32, Lb, 0.1, stag.PREC_F32)
    o32 = torch.zeros_like(x32)
    stag.apply_A_noalloc(x32, o32, Lb, 0.1, stag.PREC_F32)
    torch.cuda.synchronize()
    assert np.array_equal(_raw(o32), _raw(ref))
    Lb.close()
