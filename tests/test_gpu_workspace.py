"""The caller-owned workspace (stag_cg_workspace_bytes / stag_set_workspace)
and the immutable link handle: several host threads, each with its own stream and workspace, solve
on ONE handle at the same time (the production pattern of P:L145: many sources per gauge field);
the handle-owned default is safe -- serialised -- from several threads; pad lanes handed in dirty
cannot reach an inner product."""
import ctypes
import threading

import numpy as np
import pytest

import fieldgen
import oracle
import paper_1111_0125_b200 as stag
from tests.parity import rel_err

pytestmark = pytest.mark.gpu


def _setup(name="c2_8^4", nsrc=2):
    cfg = fieldgen.CONFIGS[name]
    W = cfg.links()
    L = stag.Links(cfg.dims, W)
    bs = [fieldgen.spinor_gaussian(cfg.dims, 0, seed=500 + k) for k in range(nsrc)]
    return cfg, W, L, bs


def _solve_in_threads(cfg, L, bds, mode, own_workspace, **kw):
    import torch
    torch.cuda.synchronize()
    out, err = [None] * len(bds), []

    def work(k):
        try:
            s = torch.cuda.Stream()
            with torch.cuda.stream(s):
                ws = None
                if own_workspace:
                    ws = torch.empty(stag.cg_workspace_bytes(cfg.dims, mode), dtype=torch.uint8, device="cuda")
                    stag.set_workspace(ws)
                for _ in range(3):                      # repeated: the cached graph is replayed
                    out[k] = stag.cg_solve(bds[k], L, cfg.mass, cfg.tol, cfg.maxiter, mode, **kw)
                s.synchronize()
                if own_workspace:
                    stag.set_workspace(None)
        except Exception as e:                          # surface it in the parent
            err.append(e)

    ts = [threading.Thread(target=work, args=(k,)) for k in range(len(bds))]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    assert not err, err
    return out


@pytest.mark.parametrize("mode", [stag.CG_F64, stag.CG_RELIABLE])
@pytest.mark.parametrize("own_workspace", [True, False])
def test_two_threads_two_streams_one_handle_equal_the_sequential_solves_bitwise(mode, own_workspace):
    import torch
    cfg, W, L, bs = _setup()
    bds = [stag.spinor_pack(b, cfg.dims, 0) for b in bs]
    seq = [stag.cg_solve(bd, L, cfg.mass, cfg.tol, cfg.maxiter, mode, recon12=True) for bd in bds]
    par = _solve_in_threads(cfg, L, bds, mode, own_workspace, recon12=True)
    for (xs, ss), (xp, sp), b in zip(seq, par, bs):
        assert ss["status"] == sp["status"] == stag.OK
        assert ss["iters"] == sp["iters"] and ss["true_resid"] == sp["true_resid"]
        assert torch.equal(xs, xp)                      # fixed-order reductions: the same bits
        x_ref, _, _, _, rc = oracle.cg(b, W, cfg.dims, cfg.mass, 1e-12, 10 * cfg.maxiter)
        assert rc == 0 and rel_err(stag.spinor_unpack(xp, cfg.dims, 0), x_ref) <= 1e-8


def test_with_a_caller_workspace_the_library_allocates_nothing_and_leaves_the_handle_alone():
    import torch
    cfg, W, L, bs = _setup(nsrc=3)
    L3 = stag.Links(cfg.dims, W)
    for prec in (stag.PREC_F64, stag.PREC_F32, stag.PREC_F32_R12):          # derived link forms exist already
        stag.dslash(stag.spinor_pack(bs[0], cfg.dims, prec), L3, 1, prec)
    bd = stag.spinor_pack_mrhs(bs, cfg.dims, 0)
    ws = torch.empty(stag.cg_workspace_bytes(cfg.dims, stag.CG_RELIABLE, 3), dtype=torch.uint8, device="cuda")
    stag.set_workspace(ws)
    try:
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        xs, sts = stag.cg_solve_mrhs(bd, L3, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE, recon12=True)
        a = stag.apply_A_mrhs(bd, L3, cfg.mass, stag.PREC_F64)
        torch.cuda.synchronize()
        # torch's own allocations (xs, a) come from its cached pool or are accounted here:
        grown = free0 - torch.cuda.mem_get_info()[0]
        assert grown <= 2 * bd.numel() * 8 + (4 << 20), grown       # nothing of workspace size was cudaMalloc'ed
        assert all(t["status"] == stag.OK for t in sts)
        for k in range(3):
            assert rel_err(stag.spinor_unpack(a[k], cfg.dims, 0), oracle.apply_A(bs[k], W, cfg.dims, cfg.mass)) <= 1e-13
        # the same calls on the handle-owned default give the same bits
        stag.set_workspace(None)
        xs2, _ = stag.cg_solve_mrhs(bd, L3, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE, recon12=True)
        assert torch.equal(xs, xs2)
    finally:
        stag.set_workspace(None)


def test_workspace_too_small_or_misaligned_is_refused():
    import torch
    cfg, W, L, bs = _setup(nsrc=1)
    bd = stag.spinor_pack(bs[0], cfg.dims, 0)
    need = stag.cg_workspace_bytes(cfg.dims, stag.CG_RELIABLE)
    small = torch.empty(need - 256, dtype=torch.uint8, device="cuda")
    stag.set_workspace(small)
    try:
        with pytest.raises(stag.StagError) as e:
            stag.cg_solve(bd, L, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE)
        assert e.value.status == stag.EINVAL and str(need) in str(e.value)
        # a workspace sized for the operator alone serves stag_apply_A, not a solve
        op = torch.empty(stag.cg_workspace_bytes(cfg.dims, -1), dtype=torch.uint8, device="cuda")
        stag.set_workspace(op)
        out = stag.apply_A(bd, L, cfg.mass, stag.PREC_F64)
        assert rel_err(stag.spinor_unpack(out, cfg.dims, 0), oracle.apply_A(bs[0], W, cfg.dims, cfg.mass)) <= 1e-13
        with pytest.raises(stag.StagError):
            stag.cg_solve(bd, L, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_F64)
        big = torch.empty(need + 512, dtype=torch.uint8, device="cuda")
        assert stag.lib().stag_set_workspace(ctypes.c_void_p(big.data_ptr() + 8), need) == stag.EINVAL   # alignment
        assert stag.lib().stag_set_workspace(None, 16) == stag.EINVAL
    finally:
        stag.set_workspace(None)


@pytest.mark.parametrize("mode", [stag.CG_F64, stag.CG_RELIABLE, stag.CG_DEFECT])
def test_dirty_pad_lanes_of_b_and_x0_cannot_reach_the_inner_products(mode):
    """Vh = 240 is padded to 256: a caller that builds b or x0 with torch ops instead of
    stag_spinor_pack may leave anything in the 16 pad lanes of each colour plane."""
    import torch
    dims, m = (6, 4, 2, 10), 0.1
    W = fieldgen.links(dims, "random", seed=41)
    b = fieldgen.spinor_gaussian(dims, 0, seed=42)
    L = stag.Links(dims, W)
    bd = stag.spinor_pack(b, dims, 0)
    x_clean, s_clean = stag.cg_solve(bd, L, m, 1e-10, 5000, mode)
    dirty_b = bd.clone()
    dirty_b.view(3, 256, 2)[:, 240:, :] = 1e6
    x0 = torch.zeros_like(bd)
    x0.view(3, 256, 2)[:, 240:, :] = -3e5
    x, st = stag.cg_solve(dirty_b, L, m, 1e-10, 5000, mode, x0=x0)
    assert st["status"] == stag.OK and st["iters"] == s_clean["iters"] and st["true_resid"] == s_clean["true_resid"]
    assert torch.equal(x, x_clean)
    assert float(x.view(3, 256, 2)[:, 240:, :].abs().max()) == 0.0
    x_ref, _, _, _, rc = oracle.cg(b, W, dims, m, 1e-12, 50000)
    assert rc == 0 and rel_err(stag.spinor_unpack(x, dims, 0), x_ref) <= 1e-8


def test_dirty_pad_lanes_in_the_propagator_wrapper():
    import torch
    dims, m = (6, 4, 2, 10), 0.2
    W = fieldgen.links(dims, "random", seed=43)
    h = np.stack([fieldgen.spinor_gaussian(dims, p, seed=44 + p) for p in (0, 1)])
    L = stag.Links(dims, W)
    he, ho = (stag.spinor_pack_mrhs([h[p]], dims, 0) for p in (0, 1))
    pe, po, _ = stag.solve_M(he, ho, L, m, 1e-11, 5000)
    he2, ho2 = he.clone(), ho.clone()
    he2.view(1, 3, 256, 2)[:, :, 240:, :] = 7e4
    ho2.view(1, 3, 256, 2)[:, :, 240:, :] = -2e4
    pe2, po2, sts = stag.solve_M(he2, ho2, L, m, 1e-11, 5000)
    assert sts[0]["status"] == stag.OK
    assert torch.equal(pe, pe2) and torch.equal(po, po2)
    assert float(po2.view(1, 3, 256, 2)[:, :, 240:, :].abs().max()) == 0.0
    psi_ref, _, _, rc = oracle.solve_M(h, W, dims, m, 1e-13, 50000)
    got = np.stack([stag.spinor_unpack(pe2[0], dims, 0), stag.spinor_unpack(po2[0], dims, 0)])
    assert rc == 0 and rel_err(got, psi_ref) <= 1e-8
