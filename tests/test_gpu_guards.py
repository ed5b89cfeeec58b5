"""Out-of-bounds writes, checked without a sanitizer (compute-sanitizer is not available on this
GPU pool): every caller-owned output lives inside a larger allocation whose guard zones before
and after it hold a sentinel bit pattern; after each entry point the guards must be untouched and
the input must be bit-identical.  Ragged volumes (pads), extents of 2, batches and slabs."""
import numpy as np
import pytest

import fieldgen
import paper_1111_0125_b200 as stag
from paper_1111_0125_b200 import slab

pytestmark = pytest.mark.gpu

GUARD = 4096          # elements on each side
SENT = -1.2345678e30


def guarded(n, dtype):
    import torch
    big = torch.full((n + 2 * GUARD,), SENT, dtype=dtype, device="cuda")
    return big, big[GUARD:GUARD + n]


def guards_intact(big, n):
    return bool((big[:GUARD] == SENT).all()) and bool((big[GUARD + n:] == SENT).all())


@pytest.mark.parametrize("dims", [(6, 4, 2, 10), (2, 2, 2, 2), (4, 4, 4, 4), (10, 6, 4, 6)])
@pytest.mark.parametrize("prec", [0, 1, 2, 3, 4, 5])
def test_hop_and_A_write_only_their_output(dims, prec):
    import torch
    W = fieldgen.links(dims, "random", seed=3)
    L = stag.Links(dims, W)
    v = stag.spinor_pack(fieldgen.spinor_gaussian(dims, 0, seed=4), dims, prec)
    v0 = v.clone()
    big, out = guarded(v.numel(), v.dtype)
    stag.dslash(v, L, 1, prec, out=out)
    assert guards_intact(big, v.numel()) and torch.equal(v, v0) and bool(torch.isfinite(out).all())
    vh = dims[0] * dims[1] * dims[2] * dims[3] // 2
    planes = out.view(3, -1, 2)
    assert planes.shape[1] == vh or float(planes[:, vh:, :].abs().max()) == 0.0      # pads stay zero
    big2, out2 = guarded(v.numel(), v.dtype)
    stag.apply_A(v, L, 0.1, prec, out=out2)
    assert guards_intact(big2, v.numel()) and torch.equal(v, v0) and bool(torch.isfinite(out2).all())


@pytest.mark.parametrize("nrhs", [1, 3, 5])
def test_batch_entries_write_only_their_output(nrhs):
    import torch
    dims = (6, 4, 2, 10)
    L = stag.Links(dims, fieldgen.links(dims, "random", seed=3))
    for prec in (0, 3):
        vs = stag.spinor_pack_mrhs([fieldgen.spinor_gaussian(dims, 0, seed=10 + k) for k in range(nrhs)], dims, prec)
        vs0 = vs.clone()
        big, flat = guarded(vs.numel(), vs.dtype)
        out = flat.view(nrhs, -1)
        stag.dslash_mrhs(vs, L, 1, prec, out=out)
        assert guards_intact(big, vs.numel()) and torch.equal(vs, vs0)
        stag.apply_A_mrhs(vs, L, 0.1, prec, out=out)
        assert guards_intact(big, vs.numel()) and torch.equal(vs, vs0)
    bs = stag.spinor_pack_mrhs([fieldgen.spinor_gaussian(dims, 0, seed=20 + k) for k in range(nrhs)], dims, 0)
    bs0 = bs.clone()
    big, flat = guarded(bs.numel(), bs.dtype)
    flat.zero_()
    x0 = flat.view(nrhs, -1)
    # the solver works in place on its x argument: call the C entry on the guarded buffer directly
    import ctypes
    sts = (stag._Stats * nrhs)()
    rc = stag.lib().stag_cg_solve_mrhs(ctypes.c_void_p(x0.data_ptr()), ctypes.c_void_p(bs.data_ptr()), L.handle,
                                       0.1, 1e-10, 2000, stag.CG_RELIABLE, nrhs, None, sts)
    torch.cuda.synchronize()
    assert rc == stag.OK and guards_intact(big, bs.numel()) and torch.equal(bs, bs0)


def test_slab_hop_and_pack_unpack_write_only_their_output():
    import torch
    dims = (6, 2, 2, 8)
    W = fieldgen.links(dims, "random", seed=3)
    slabs = [slab.SlabLinks(dims, W, r, 2) for r in range(2)]
    slab.connect_in_process(slabs)
    chi = fieldgen.spinor_gaussian(dims, 0, seed=4)
    for prec in (0, 3):
        vs = [stag.spinor_pack(np.ascontiguousarray(slab.scatter_spinor(chi, dims, r, 2)), slabs[r].dims, prec) for r in range(2)]
        for r in range(2):
            slabs[r].push(vs[r], prec)
        for r in range(2):
            big, out = guarded(vs[r].numel(), vs[r].dtype)
            slabs[r].hop(vs[r], 1, prec, out=out)
            assert guards_intact(big, vs[r].numel())
    # pack / unpack on a ragged volume
    d2 = (6, 4, 2, 10)
    c = fieldgen.spinor_gaussian(d2, 0, seed=5)
    src = torch.from_numpy(c.view(np.float64).reshape(-1)).cuda()
    n = stag.spinor_bytes(d2, 0) // 8
    big, dst = guarded(n, torch.float64)
    import ctypes
    assert stag.lib().stag_spinor_pack(ctypes.c_void_p(dst.data_ptr()), ctypes.c_void_p(src.data_ptr()), stag._cdims(d2), 0) == 0
    big2, back = guarded(src.numel(), torch.float64)
    assert stag.lib().stag_spinor_unpack(ctypes.c_void_p(back.data_ptr()), ctypes.c_void_p(dst.data_ptr()), stag._cdims(d2), 0) == 0
    torch.cuda.synchronize()
    assert guards_intact(big, n) and guards_intact(big2, src.numel()) and torch.equal(back, src)
