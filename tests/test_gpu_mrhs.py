"""GPU parity of the several-right-hand-sides entry points (stag_dslash_mrhs, stag_apply_A_mrhs,
stag_cg_solve_mrhs) and of the propagator wrapper stag_solve_M against the CPU oracle, through
the C ABI.  A batch is nothing new mathematically: right-hand side k of every result must equal
the oracle's single-vector result for input k (same tolerances as the single entry points)."""
import ctypes

import numpy as np
import pytest

import fieldgen
import oracle
import paper_1111_0125_b200 as stag

pytestmark = pytest.mark.gpu

TOL = {stag.PREC_F64: 1e-13, stag.PREC_F64_R12: 1e-13, stag.PREC_F32: 2e-6, stag.PREC_F32_R12: 2e-6}
ALL_PREC = [stag.PREC_F64, stag.PREC_F32, stag.PREC_F64_R12, stag.PREC_F32_R12]


from tests.parity import rel_err as rel_l2  # L2 AND worst-site bound (tests/parity.py)


# nrhs values cover every chunking: 1..4 in one fp32 launch, 5 = 4+1, 7 = 4+3, 12 = the cap;
# in fp64 (chunks of 2) they cover 2, 2+1, 2+2, ...
@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (6, 4, 2, 10), (2, 2, 2, 2)])
@pytest.mark.parametrize("prec", ALL_PREC)
@pytest.mark.parametrize("nrhs", [1, 2, 3, 4, 5, 7, 12])
def test_dslash_mrhs_matches_oracle(dims, prec, nrhs):
    W = fieldgen.links(dims, "random", seed=31)
    L = stag.Links(dims, W)
    for parity in (0, 1):
        chis = [fieldgen.spinor_gaussian(dims, 1 - parity, seed=40 + k) for k in range(nrhs)]
        outs = stag.dslash_mrhs(stag.spinor_pack_mrhs(chis, dims, prec), L, parity, prec)
        for k, o in enumerate(stag.spinor_unpack_mrhs(outs, dims, prec)):
            assert rel_l2(o, oracle.dslash(chis[k], W, dims, parity)) <= TOL[prec], (k, parity)


@pytest.mark.parametrize("prec", ALL_PREC)
def test_mrhs_hop_equals_single_hop_bitwise_and_keeps_pads_zero(prec):
    """Same arithmetic in the same order per right-hand side: the batch kernel must give the
    bits of the single kernel; pad lanes of every spinor of the batch stay zero."""
    import torch
    dims = (6, 4, 2, 10)          # Vh = 240, Vh_pad = 256
    W = fieldgen.links(dims, "random", seed=3)
    L = stag.Links(dims, W)
    chis = [fieldgen.spinor_gaussian(dims, 0, seed=50 + k) for k in range(3)]
    vs = stag.spinor_pack_mrhs(chis, dims, prec)
    outs = torch.full_like(vs, float("nan"))
    stag.dslash_mrhs(vs, L, 1, prec, out=outs)
    for k in range(3):
        single = stag.dslash(vs[k].contiguous(), L, 1, prec)
        assert torch.equal(outs[k], single)
        assert float(outs[k].view(3, 256, 2)[:, 240:, :].abs().max()) == 0.0


@pytest.mark.parametrize("prec", ALL_PREC)
@pytest.mark.parametrize("nrhs", [2, 3, 5])
def test_apply_A_mrhs_matches_oracle(prec, nrhs):
    cfg = fieldgen.CONFIGS["c2_8^4"]
    W = cfg.links()
    L = stag.Links(cfg.dims, W)
    chis = [fieldgen.spinor_gaussian(cfg.dims, 0, seed=60 + k) for k in range(nrhs)]
    outs = stag.apply_A_mrhs(stag.spinor_pack_mrhs(chis, cfg.dims, prec), L, cfg.mass, prec)
    for k, o in enumerate(stag.spinor_unpack_mrhs(outs, cfg.dims, prec)):
        assert rel_l2(o, oracle.apply_A(chis[k], W, cfg.dims, cfg.mass)) <= TOL[prec]


def _check_solution(x, b, W, cfg, x_ref, tol):
    res = np.linalg.norm((b - oracle.apply_A(x, W, cfg.dims, cfg.mass)).ravel()) / np.linalg.norm(b.ravel())
    assert res <= tol * (1 + 1e-3), res
    assert rel_l2(x, x_ref) <= 1e-8


@pytest.mark.parametrize("mode", [stag.CG_F64, stag.CG_DEFECT, stag.CG_RELIABLE])
@pytest.mark.parametrize("recon12", [False, True])
def test_cg_mrhs_each_solution_matches_oracle(mode, recon12):
    """Three Gaussian sources on config 1: each x_k against the oracle's own solve of b_k
    (to 1e-12), true residual recomputed with the oracle's A, iteration counts within a few %
    of the oracle's (Q17)."""
    cfg = fieldgen.CONFIGS["c1_4^4"]
    W = cfg.links()
    L = stag.Links(cfg.dims, W)
    bs = [fieldgen.spinor_gaussian(cfg.dims, 0, seed=70 + k) for k in range(3)]
    xs, sts = stag.cg_solve_mrhs(stag.spinor_pack_mrhs(bs, cfg.dims, 0), L, cfg.mass, cfg.tol, cfg.maxiter,
                                 mode, recon12=recon12)
    for k, x in enumerate(stag.spinor_unpack_mrhs(xs, cfg.dims, 0)):
        x_ref, it_ref, _, _, rc = oracle.cg(bs[k], W, cfg.dims, cfg.mass, 1e-12, 10 * cfg.maxiter)
        assert rc == 0
        assert sts[k]["status"] == stag.OK and sts[k]["true_resid"] <= cfg.tol
        _check_solution(x, bs[k], W, cfg, x_ref, cfg.tol)
        _, it10, _, _, _ = oracle.cg(bs[k], W, cfg.dims, cfg.mass, cfg.tol, cfg.maxiter)
        if mode != stag.CG_DEFECT:
            assert abs(sts[k]["iters"] - it10) <= 0.1 * it10 + 3, (sts[k]["iters"], it10)


def test_cg_mrhs_freezes_finished_right_hand_sides_and_handles_zero_source():
    """Free field: a plane wave is an eigenvector of A (one iteration), a Gaussian source needs
    many, a zero source none.  Each must come out right although they share the loop."""
    cfg = fieldgen.CONFIGS["c2_8^4_free"]
    W = cfg.links()
    L = stag.Links(cfg.dims, W)
    pw = fieldgen.spinor_planewave(cfg.dims, (1, 2, 3, 0))
    ga = fieldgen.spinor_gaussian(cfg.dims, 0, seed=80)
    ze = np.zeros_like(ga)
    for mode in (stag.CG_F64, stag.CG_RELIABLE):
        xs, sts = stag.cg_solve_mrhs(stag.spinor_pack_mrhs([pw, ga, ze], cfg.dims, 0), L, cfg.mass, cfg.tol,
                                     cfg.maxiter, mode)
        x = stag.spinor_unpack_mrhs(xs, cfg.dims, 0)
        lam = cfg.mass ** 2 + 4 * sum(np.sin(2 * np.pi * (n + (0.5 if mu == 3 else 0.0)) / cfg.dims[mu]) ** 2
                                      for mu, n in enumerate((1, 2, 3, 0)))
        assert rel_l2(x[0], pw / lam) <= 1e-9
        x_ref, it_ref, _, _, _ = oracle.cg(ga, W, cfg.dims, cfg.mass, 1e-12, 10 * cfg.maxiter)
        _check_solution(x[1], ga, W, cfg, x_ref, cfg.tol)
        assert not x[2].any() and sts[2]["iters"] == 0 and sts[2]["true_resid"] == 0.0
        assert sts[0]["iters"] <= 3 < sts[1]["iters"]
        assert all(s["status"] == stag.OK for s in sts)


def test_cg_mrhs_one_rhs_equals_single_entry_bitwise():
    import torch
    cfg = fieldgen.CONFIGS["c1_4^4"]
    L = stag.Links(cfg.dims, cfg.links())
    b = stag.spinor_pack(cfg.source(), cfg.dims, 0)
    x1, st1 = stag.cg_solve(b, L, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE)
    xs, sts = stag.cg_solve_mrhs(b.view(1, -1), L, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE)
    assert torch.equal(xs[0], x1) and sts[0]["iters"] == st1["iters"]


def test_cg_mrhs_batch_reproduces_single_solves_bitwise():
    """Lockstep does not couple the recurrences: in pure fp64 CG (no shared trigger) every
    right-hand side of a batch goes through exactly the arithmetic of its own single solve (on the
    kernel-per-step path the batch runs on; the persistent kernel sums in another order)."""
    import torch
    cfg = fieldgen.CONFIGS["c1_4^4"]
    L = stag.Links(cfg.dims, cfg.links())
    bs = [fieldgen.spinor_gaussian(cfg.dims, 0, seed=90 + k) for k in range(3)]
    vb = stag.spinor_pack_mrhs(bs, cfg.dims, 0)
    xs, sts = stag.cg_solve_mrhs(vb, L, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_F64)
    for k in range(3):
        x1, st1 = stag.cg_solve(vb[k].contiguous(), L, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_F64, persistent=False)
        assert sts[k]["iters"] == st1["iters"]
        assert torch.equal(xs[k], x1)


@pytest.mark.parametrize("mode", [stag.CG_F64, stag.CG_RELIABLE])
def test_solve_M_propagator_matches_oracle(mode):
    """The staggered propagator from a point source, three colours at once (Q23):
    psi against the oracle's solve_M (to 1e-12) and |h - (D+m) psi| with the oracle's M."""
    cfg = fieldgen.CONFIGS["c1_4^4"]
    W = cfg.links()
    L = stag.Links(cfg.dims, W)
    vh = cfg.vh
    hs = []
    for c in range(3):
        h = np.zeros((2, vh, 3), dtype=np.complex128)
        h[1, 5, c] = 1.0                      # an odd site: exercises the D_eo h_o term
        h[0, 0, c] = 0.5
        hs.append(h)
    he = stag.spinor_pack_mrhs([np.ascontiguousarray(h[0]) for h in hs], cfg.dims, 0)
    ho = stag.spinor_pack_mrhs([np.ascontiguousarray(h[1]) for h in hs], cfg.dims, 0)
    pe, po, sts = stag.solve_M(he, ho, L, cfg.mass, cfg.tol, cfg.maxiter, mode)
    pe, po = stag.spinor_unpack_mrhs(pe, cfg.dims, 0), stag.spinor_unpack_mrhs(po, cfg.dims, 0)
    for c in range(3):
        psi = np.ascontiguousarray(np.stack([pe[c], po[c]]))
        ref, _, _, rc = oracle.solve_M(hs[c], W, cfg.dims, cfg.mass, 1e-12, 10 * cfg.maxiter)
        assert rc == 0 and sts[c]["status"] == stag.OK
        assert rel_l2(psi, ref) <= 1e-8
        b_e = cfg.mass * hs[c][0] - oracle.dslash(np.ascontiguousarray(hs[c][1]), W, cfg.dims, 0)
        res = rel_l2(oracle.apply_M(psi, W, cfg.dims, cfg.mass), hs[c])
        assert res <= cfg.tol * np.linalg.norm(b_e) / (cfg.mass * np.linalg.norm(hs[c])) * (1 + 1e-3)


def test_mrhs_argument_errors():
    cfg = fieldgen.CONFIGS["c1_4^4"]
    L = stag.Links(cfg.dims, cfg.links())
    b = stag.spinor_pack(cfg.source(), cfg.dims, 0)
    x = stag.empty_spinor(cfg.dims, 0)
    lib = stag.lib()
    vp = ctypes.c_void_p
    cd = (ctypes.c_int * 4)(*cfg.dims)
    assert lib.stag_dslash_mrhs(vp(x.data_ptr()), vp(b.data_ptr()), L.handle, 1, cd, 0, 0) == stag.EINVAL
    assert lib.stag_apply_A_mrhs(vp(x.data_ptr()), vp(b.data_ptr()), L.handle, 0.1, 0, 0) == stag.EINVAL
    for bad in (0, stag.MAX_RHS + 1):
        assert lib.stag_cg_solve_mrhs(vp(x.data_ptr()), vp(b.data_ptr()), L.handle, 0.1, 1e-10, 10, 3, bad,
                                      None, None) == stag.EINVAL
    assert lib.stag_solve_M(vp(x.data_ptr()), vp(x.data_ptr()), vp(b.data_ptr()), vp(b.data_ptr()), L.handle,
                            0.0, 1e-10, 10, 3, 1, None, None) == stag.EINVAL      # mass = 0


@pytest.mark.slow
def test_mrhs_full_size_hop_matches_oracle():
    """bench configuration: three right-hand sides through the fp32/12 and fp64/18 batch hops in the
    blocked layout, then 2, 3 and 4 right-hand sides through the PAIRED layout -- the instantiations
    dslash_batch_kernel<.., PAIRED = true> that bench.py's `mrhs.dslash` rows time and the fp32
    iteration of stag_cg_solve_mrhs runs on -- every output site against the oracle (eq. 2.5),
    relative L2 error and worst component (tests/parity.py)."""
    import torch
    cfg = fieldgen.CONFIGS["c4_28^3x96"]
    W = cfg.links()
    L = stag.Links(cfg.dims, W)
    chis = [fieldgen.spinor_gaussian(cfg.dims, 0, seed=100 + k) for k in range(4)]
    refs = [oracle.dslash(c, W, cfg.dims, 1) for c in chis]
    for prec in (stag.PREC_F32_R12, stag.PREC_F32, stag.PREC_F64):
        outs = stag.dslash_mrhs(stag.spinor_pack_mrhs(chis[:3], cfg.dims, prec), L, 1, prec)
        for k, o in enumerate(stag.spinor_unpack_mrhs(outs, cfg.dims, prec)):
            assert rel_l2(o, refs[k]) <= TOL[prec]
    for prec in (stag.PREC_F32_R12, stag.PREC_F32):
        for n in (2, 3, 4):
            pv = stag.batch_convert(stag.spinor_pack_mrhs(chis[:n], cfg.dims, prec), cfg.dims, prec, stag.BATCH_PAIRED)
            po = torch.full_like(pv, float("nan"))
            stag.dslash_mrhs(pv, L, 1, prec, out=po, layout=stag.BATCH_PAIRED)
            outs = stag.batch_convert(po, cfg.dims, prec, stag.BATCH_BLOCKED)
            for k, o in enumerate(stag.spinor_unpack_mrhs(outs, cfg.dims, prec)):
                assert rel_l2(o, refs[k]) <= TOL[prec], (prec, n, k)
    L.close()


@pytest.mark.slow
def test_batched_solve_and_propagator_full_size_with_oracle_operators():
    """bench configuration (28^3 x 96): three sources in lockstep (mode 3, 12-real fp32 links), each
    solution checked through the ORACLE's A; right-hand side 0 is the config's own source, so its
    solution is also held to north_star's "within 1e-8 relative of the oracle solve" (eq. 2.1-2.3,
    P:L27-37) against the oracle's stored solve (tests/golden/refsol_c4_283x96.npz, tests/refsol.py);
    then the propagator wrapper for a point source in the three colours, checked through the oracle's
    M = D + m on the whole lattice."""
    from tests import refsol
    cfg = fieldgen.CONFIGS["c4_28^3x96"]
    rec = refsol.load(cfg.name)
    W = cfg.links()
    L = stag.Links(cfg.dims, W)
    bs = [cfg.source()] + [fieldgen.spinor_gaussian(cfg.dims, 0, seed=500 + k) for k in (1, 2)]
    xs, sts = stag.cg_solve_mrhs(stag.spinor_pack_mrhs(bs, cfg.dims, 0), L, cfg.mass, cfg.tol, cfg.maxiter,
                                 stag.CG_RELIABLE, recon12=True)
    for k, x in enumerate(stag.spinor_unpack_mrhs(xs, cfg.dims, 0)):
        assert sts[k]["status"] == stag.OK and sts[k]["true_resid"] <= cfg.tol
        res = np.linalg.norm((bs[k] - oracle.apply_A(x, W, cfg.dims, cfg.mass)).ravel()) / np.linalg.norm(bs[k].ravel())
        assert res <= cfg.tol * (1 + 1e-3), (k, res)
        if k == 0:
            s = refsol.score(x, rec, cfg)
            print("batched solve, right-hand side 0 vs the oracle's solve: %r" % (s,))
            assert s["l2_sketch"] <= 1e-8 and s["l2_sites"] <= 1e-8 and s["max_site"] <= 1e-8 and s["norm"] <= 1e-8
    del xs
    hs = []
    for c in range(3):
        h = np.zeros((2, cfg.vh, 3), dtype=np.complex128)
        h[1, 12345, c] = 1.0
        hs.append(h)
    he = stag.spinor_pack_mrhs([np.ascontiguousarray(h[0]) for h in hs], cfg.dims, 0)
    ho = stag.spinor_pack_mrhs([np.ascontiguousarray(h[1]) for h in hs], cfg.dims, 0)
    pe, po, sts = stag.solve_M(he, ho, L, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE, recon12=True)
    pe, po = stag.spinor_unpack_mrhs(pe, cfg.dims, 0), stag.spinor_unpack_mrhs(po, cfg.dims, 0)
    for c in range(3):
        assert sts[c]["status"] == stag.OK
        psi = np.ascontiguousarray(np.stack([pe[c], po[c]]))
        b_e = cfg.mass * hs[c][0] - oracle.dslash(np.ascontiguousarray(hs[c][1]), W, cfg.dims, 0)
        res = rel_l2(oracle.apply_M(psi, W, cfg.dims, cfg.mass), hs[c])
        assert res <= cfg.tol * np.linalg.norm(b_e) / (cfg.mass * np.linalg.norm(hs[c])) * (1 + 1e-3), (c, res)
    L.close()


# ---- the paired fp32 batch layout (include/stag.h "batch layouts") ---------

F32_PREC = [stag.PREC_F32, stag.PREC_F32_R12]


@pytest.mark.parametrize("nrhs", [1, 2, 3, 4, 5, 7, 12])
def test_batch_convert_is_the_documented_permutation_and_round_trips(nrhs):
    """paired[j][c][cb] = (re_2j, im_2j, re_2j+1, im_2j+1); an odd last right-hand side stays an
    ordinary spinor; pure data movement, so the round trip is exact."""
    import torch
    dims = (6, 4, 2, 10)          # Vh_pad = 256
    chis = [fieldgen.spinor_gaussian(dims, 0, seed=90 + k) for k in range(nrhs)]
    vs = stag.spinor_pack_mrhs(chis, dims, stag.PREC_F32)
    pv = stag.batch_convert(vs, dims, stag.PREC_F32, stag.BATCH_PAIRED)
    flat = pv.reshape(-1)
    n = vs.shape[1]                                  # 6 * Vh_pad reals per spinor
    for j in range(nrhs // 2):
        pair = flat[2 * j * n:(2 * j + 2) * n].view(3 * 256, 2, 2)       # [complex index][half][re,im]
        assert torch.equal(pair[:, 0, :].reshape(-1), vs[2 * j])
        assert torch.equal(pair[:, 1, :].reshape(-1), vs[2 * j + 1])
    if nrhs % 2:
        assert torch.equal(flat[(nrhs - 1) * n:], vs[nrhs - 1])
    assert torch.equal(stag.batch_convert(pv, dims, stag.PREC_F32, stag.BATCH_BLOCKED), vs)
    v64 = stag.spinor_pack_mrhs(chis, dims, stag.PREC_F64)
    assert torch.equal(stag.batch_convert(v64, dims, stag.PREC_F64, stag.BATCH_PAIRED), v64)   # fp64: one layout


@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (6, 4, 2, 10), (2, 2, 2, 2)])
@pytest.mark.parametrize("prec", F32_PREC)
@pytest.mark.parametrize("nrhs", [2, 3, 4, 5, 7, 12])
def test_paired_hop_matches_oracle_and_the_blocked_hop_bitwise(dims, prec, nrhs):
    import torch
    W = fieldgen.links(dims, "random", seed=31)
    L = stag.Links(dims, W)
    for parity in (0, 1):
        chis = [fieldgen.spinor_gaussian(dims, 1 - parity, seed=40 + k) for k in range(nrhs)]
        vs = stag.spinor_pack_mrhs(chis, dims, prec)
        pv = stag.batch_convert(vs, dims, prec, stag.BATCH_PAIRED)
        po = torch.full_like(pv, float("nan"))
        stag.dslash_mrhs(pv, L, parity, prec, out=po, layout=stag.BATCH_PAIRED)
        outs = stag.batch_convert(po, dims, prec, stag.BATCH_BLOCKED)
        assert torch.equal(outs, stag.dslash_mrhs(vs, L, parity, prec))       # same arithmetic per right-hand side
        for k, o in enumerate(stag.spinor_unpack_mrhs(outs, dims, prec)):
            assert rel_l2(o, oracle.dslash(chis[k], W, dims, parity)) <= TOL[prec], (k, parity)
        vh, vp = np.prod(dims) // 2, outs.shape[1] // 6
        if vp != vh:
            assert float(outs.view(nrhs, 3, vp, 2)[:, :, vh:, :].abs().max()) == 0.0   # pads stay zero


@pytest.mark.parametrize("prec", F32_PREC)
@pytest.mark.parametrize("nrhs", [2, 3, 5])
def test_paired_apply_A_matches_oracle(prec, nrhs):
    cfg = fieldgen.CONFIGS["c2_8^4"]
    W = cfg.links()
    L = stag.Links(cfg.dims, W)
    chis = [fieldgen.spinor_gaussian(cfg.dims, 0, seed=60 + k) for k in range(nrhs)]
    pv = stag.batch_convert(stag.spinor_pack_mrhs(chis, cfg.dims, prec), cfg.dims, prec, stag.BATCH_PAIRED)
    outs = stag.batch_convert(stag.apply_A_mrhs(pv, L, cfg.mass, prec, layout=stag.BATCH_PAIRED), cfg.dims, prec, stag.BATCH_BLOCKED)
    for k, o in enumerate(stag.spinor_unpack_mrhs(outs, cfg.dims, prec)):
        assert rel_l2(o, oracle.apply_A(chis[k], W, cfg.dims, cfg.mass)) <= TOL[prec]


def test_paired_layout_is_refused_for_fp64():
    import torch
    dims = (4, 4, 4, 4)
    L = stag.Links(dims, fieldgen.links(dims, "random", seed=1))
    vs = stag.spinor_pack_mrhs([fieldgen.spinor_gaussian(dims, 0, seed=k) for k in range(2)], dims, stag.PREC_F64)
    with pytest.raises(stag.StagError):
        stag.dslash_mrhs(vs, L, 1, stag.PREC_F64, layout=stag.BATCH_PAIRED)
    with pytest.raises(stag.StagError):
        stag.dslash_mrhs(vs, L, 1, stag.PREC_F64, layout=2)


@pytest.mark.parametrize("mode", [stag.CG_F32, stag.CG_DEFECT, stag.CG_RELIABLE])
@pytest.mark.parametrize("nrhs", [2, 3, 4, 5])
def test_cg_mrhs_on_paired_fp32_vectors_all_chunkings(mode, nrhs):
    """The fp32 iteration keeps its vectors paired when nrhs >= 2: pairs only (2, 4), pair + single
    (3), a full chunk + single (5); a ragged lattice so that pad lanes exist.  Each x_k against the
    oracle's solve of b_k."""
    dims, m = (6, 4, 2, 10), 0.1
    W = fieldgen.links(dims, "random", seed=51)
    L = stag.Links(dims, W)
    bs = [fieldgen.spinor_gaussian(dims, 0, seed=170 + k) for k in range(nrhs)]
    xs, sts = stag.cg_solve_mrhs(stag.spinor_pack_mrhs(bs, dims, 0), L, m, 1e-10, 5000, mode, recon12=True)
    for k, x in enumerate(stag.spinor_unpack_mrhs(xs, dims, 0)):
        x_ref, it_ref, _, _, rc = oracle.cg(bs[k], W, dims, m, 1e-12, 50000)
        assert rc == 0
        res = np.linalg.norm((bs[k] - oracle.apply_A(x, W, dims, m)).ravel()) / np.linalg.norm(bs[k].ravel())
        if mode == stag.CG_F32:                        # pure fp32 stalls (SURVEY pin 9) but must agree with its own report
            assert sts[k]["status"] == stag.ENOCONV and abs(res - sts[k]["true_resid"]) <= 1e-3 * res
            assert rel_l2(x, x_ref) <= 1e-3
            continue
        assert sts[k]["status"] == stag.OK and sts[k]["true_resid"] <= 1e-10
        assert res <= 1e-10 * (1 + 1e-3)
        assert rel_l2(x, x_ref) <= 1e-8
        assert sts[k]["iters"] <= 1.3 * it_ref + 5
