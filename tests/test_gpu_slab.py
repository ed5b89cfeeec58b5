"""GPU parity of the T-slab hop (stag_slab_push / stag_slab_hop) on ONE device: the slabs of a
decomposition live in one process, are wired with raw pointers, and run one after the other
(all pushes of an exchange, then all hops), so no kernel ever waits on a kernel that has not been
launched.  The data path -- links gathered per slab from the whole field, faces stored into the
neighbours' halo buffers, flags, halo reads, 12-real signs at the global time boundary -- is the
multi-GPU one.  Results must equal the whole-lattice kernel BITWISE (same arithmetic per site) and
the oracle within the usual tolerance."""
import numpy as np
import pytest

import fieldgen
import oracle
import paper_1111_0125_b200 as stag
from paper_1111_0125_b200 import slab

pytestmark = pytest.mark.gpu

TOL = {stag.PREC_F64: 1e-13, stag.PREC_F64_R12: 1e-13, stag.PREC_F32: 2e-6, stag.PREC_F32_R12: 2e-6}
ALL_PREC = [stag.PREC_F64, stag.PREC_F32, stag.PREC_F64_R12, stag.PREC_F32_R12]


from tests.parity import rel_err as rel_l2  # L2 AND worst-site bound (tests/parity.py)


def make_slabs(dims, W, nranks, antiperiodic=True):
    slabs = [slab.SlabLinks(dims, W, r, nranks, antiperiodic_t=antiperiodic) for r in range(nranks)]
    slab.connect_in_process(slabs)
    return slabs


def slab_hop_all(slabs, chi, dims, parity, prec):
    """One decomposed hop: scatter, all pushes, all hops, gather (canonical in, canonical out)."""
    n = len(slabs)
    vs = [stag.spinor_pack(np.ascontiguousarray(slab.scatter_spinor(chi, dims, r, n)), slabs[r].dims, prec)
          for r in range(n)]
    for r in range(n):
        slabs[r].push(vs[r], prec)
    outs = [slabs[r].hop(vs[r], parity, prec) for r in range(n)]
    return outs, slab.gather_spinor([stag.spinor_unpack(o, slabs[r].dims, prec) for r, o in enumerate(outs)], dims)


# (dims, nranks): several ranks, two ranks (both neighbours the same slab), one rank (its own
# neighbour), slabs of two slices (every slice is a boundary), ragged Vh (pads), X_mu = 2
CASES = [((4, 4, 4, 8), 2), ((4, 4, 4, 12), 3), ((4, 4, 4, 8), 4), ((4, 4, 4, 4), 1),
         ((6, 2, 2, 8), 2), ((2, 2, 2, 4), 2), ((8, 8, 8, 8), 2)]


@pytest.mark.parametrize("dims,nranks", CASES)
@pytest.mark.parametrize("prec", ALL_PREC)
def test_slab_hop_matches_oracle_and_whole_lattice_kernel(dims, nranks, prec):
    import torch
    W = fieldgen.links(dims, "random", seed=61)
    L = stag.Links(dims, W)
    slabs = make_slabs(dims, W, nranks)
    for parity in (0, 1):
        chi = fieldgen.spinor_gaussian(dims, 1 - parity, seed=62 + parity)
        outs, got = slab_hop_all(slabs, chi, dims, parity, prec)
        assert rel_l2(got, oracle.dslash(chi, W, dims, parity)) <= TOL[prec]
        whole = stag.spinor_unpack(stag.dslash(stag.spinor_pack(chi, dims, prec), L, parity, prec), dims, prec)
        assert np.array_equal(got, whole)
        for r, o in enumerate(outs):                      # pads of every slab's output stay zero
            vh = slabs[r].dims[0] * slabs[r].dims[1] * slabs[r].dims[2] * slabs[r].dims[3] // 2
            planes = o.view(3, -1, 2)
            assert float(planes[:, vh:, :].abs().max()) == 0.0 if planes.shape[1] > vh else True


@pytest.mark.parametrize("dims,nranks", [((4, 4, 4, 8), 2), ((6, 2, 2, 12), 3), ((4, 4, 4, 4), 1), ((2, 2, 2, 8), 4)])
def test_slab_from_its_own_time_slices_equals_slab_from_the_whole_field(dims, nranks):
    """stag_slab_create_local: a rank hands over only its own time slices of the links plus the
    t-links of the slice before them (slab.scatter_links), never the whole lattice.  Both hops, all
    four link forms: bitwise equal to the slabs made from the whole field, and within tolerance of
    the oracle (which only ever sees the whole field)."""
    W = fieldgen.links(dims, "random", seed=63)
    whole = make_slabs(dims, W, nranks)
    local = []
    for r in range(nranks):
        Wl, Wb = slab.scatter_links(W, dims, r, nranks)
        local.append(slab.SlabLinks(dims, Wl, r, nranks, W_back=Wb))
    slab.connect_in_process(local)
    for parity in (0, 1):
        chi = fieldgen.spinor_gaussian(dims, 1 - parity, seed=64 + parity)
        ref = oracle.dslash(chi, W, dims, parity)
        for prec in ALL_PREC:
            _, a = slab_hop_all(whole, chi, dims, parity, prec)
            _, b = slab_hop_all(local, chi, dims, parity, prec)
            assert np.array_equal(a, b)
            assert rel_l2(b, ref) <= TOL[prec]
    with pytest.raises(ValueError):
        slab.SlabLinks(dims, W[:, :, :7], 0, nranks)                    # neither whole nor local + back
    for s in whole + local:
        s.close()


@pytest.mark.parametrize("prec", ALL_PREC)
def test_slab_hop_periodic_time_boundary(prec):
    dims = (4, 4, 2, 8)
    W = fieldgen.links(dims, "random", seed=5, antiperiodic_t=False)
    slabs = make_slabs(dims, W, 2, antiperiodic=False)
    chi = fieldgen.spinor_gaussian(dims, 0, seed=6)
    _, got = slab_hop_all(slabs, chi, dims, 1, prec)
    assert rel_l2(got, oracle.dslash(chi, W, dims, 1)) <= TOL[prec]


@pytest.mark.parametrize("nranks", [1, 2, 4])
@pytest.mark.parametrize("prec", [stag.PREC_F64, stag.PREC_F32_R12])
def test_slab_apply_A_matches_oracle_over_repeated_exchanges(nranks, prec):
    """A = m^2 - D_eo D_oe through two exchanges per application, applied three times in a row so
    both halo buffers and the epoch flags are reused."""
    cfg = fieldgen.CONFIGS["c2_8^4"]
    W = cfg.links()
    slabs = make_slabs(cfg.dims, W, nranks)
    chi = cfg.source()
    for rep in range(3):
        ref = oracle.apply_A(chi, W, cfg.dims, cfg.mass)
        vs = [stag.spinor_pack(np.ascontiguousarray(slab.scatter_spinor(chi, cfg.dims, r, nranks)), slabs[r].dims, prec)
              for r in range(nranks)]
        for r in range(nranks):
            slabs[r].push(vs[r], prec)
        tmps = [slabs[r].hop(vs[r], 1, prec) for r in range(nranks)]
        for r in range(nranks):
            slabs[r].push(tmps[r], prec)
        outs = [slabs[r].hop(tmps[r], 0, prec, a=cfg.mass ** 2, own=vs[r]) for r in range(nranks)]
        got = slab.gather_spinor([stag.spinor_unpack(o, slabs[r].dims, prec) for r, o in enumerate(outs)], cfg.dims)
        assert rel_l2(got, ref) <= TOL[prec]
        chi = np.ascontiguousarray(ref / np.linalg.norm(ref) * np.linalg.norm(chi))


def test_single_rank_slab_dslash_entry_and_argument_errors():
    """nranks = 1: stag_slab_dslash (push + hop in one call) is safe on one device."""
    import ctypes
    dims = (4, 4, 4, 4)
    W = fieldgen.links(dims, "random", seed=1)
    chi = fieldgen.spinor_gaussian(dims, 0, seed=2)
    S = slab.SlabLinks(dims, W, 0, 1)
    v = stag.spinor_pack(chi, dims, 0)
    out = stag.empty_spinor(dims, 0)
    lib = stag.lib()
    vp = ctypes.c_void_p
    assert lib.stag_slab_hop(vp(out.data_ptr()), vp(v.data_ptr()), S.handle, 1, 0, 0.0, None) == stag.EINVAL  # no push yet
    got = stag.spinor_unpack(S.dslash(v, 1, 0), dims, 0)
    assert rel_l2(got, oracle.dslash(chi, W, dims, 1)) <= 1e-13
    # a slab handle is refused by the whole-lattice entry points, and vice versa
    cd = (ctypes.c_int * 4)(*dims)
    assert lib.stag_dslash(vp(out.data_ptr()), vp(v.data_ptr()), S.handle, 1, cd, 0) == stag.EINVAL
    L = stag.Links(dims, W)
    assert lib.stag_slab_push(vp(v.data_ptr()), L.handle, 0) == stag.EINVAL
    h = ctypes.c_void_p()
    for rank, n in ((0, 3), (2, 2), (0, 4)):     # 4/3 not integer; rank out of range; 1 slice each
        assert lib.stag_slab_create(ctypes.byref(h), cd, 1, vp(W.ctypes.data), 0, rank, n) == stag.EINVAL
    two = slab.SlabLinks((4, 4, 4, 8), fieldgen.links((4, 4, 4, 8), "random", seed=1), 0, 2)
    v8 = stag.empty_spinor(two.dims, 0)
    assert lib.stag_slab_push(vp(v8.data_ptr()), two.handle, 0) == stag.EINVAL   # not connected yet


# ---- CG over the slabs -------------------------------------------------------------------
def _slab_cg(cfg, W, b, nranks, mode, **kw):
    slabs = make_slabs(cfg.dims, W, nranks)
    bs = [stag.spinor_pack(np.ascontiguousarray(slab.scatter_spinor(b, cfg.dims, r, nranks)), slabs[r].dims, 0)
          for r in range(nranks)]
    xs, sts = slab.cg_solve_in_process(slabs, bs, cfg.mass, cfg.tol, cfg.maxiter, mode, **kw)
    x = slab.gather_spinor([stag.spinor_unpack(xs[r], slabs[r].dims, 0) for r in range(nranks)], cfg.dims)
    return x, sts


@pytest.mark.parametrize("nranks", [1, 2, 4])
@pytest.mark.parametrize("mode", [stag.CG_F64, stag.CG_RELIABLE])
def test_slab_cg_matches_oracle(nranks, mode):
    """The multi-GPU solve, all ranks on one device: x against the oracle's solve (to 1e-12),
    the fp64 true residual recomputed with the oracle's A, iteration count within a few % of
    the oracle's (Q17), and every rank reporting the same scalars."""
    cfg = fieldgen.CONFIGS["c2_8^4"]
    W, b = cfg.links(), cfg.source()
    x, sts = _slab_cg(cfg, W, b, nranks, mode)
    x_ref, _, _, _, rc = oracle.cg(b, W, cfg.dims, cfg.mass, 1e-12, 10 * cfg.maxiter)
    _, it10, _, _, _ = oracle.cg(b, W, cfg.dims, cfg.mass, cfg.tol, cfg.maxiter)
    assert rc == 0
    for st in sts:
        assert st["status"] == stag.OK and st["true_resid"] <= cfg.tol
        assert (st["iters"], st["true_resid"], st["n_updates"]) == (sts[0]["iters"], sts[0]["true_resid"], sts[0]["n_updates"])
    assert abs(sts[0]["iters"] - it10) <= 0.05 * it10 + 3
    res = np.linalg.norm((b - oracle.apply_A(x, W, cfg.dims, cfg.mass)).ravel()) / np.linalg.norm(b.ravel())
    assert res <= cfg.tol * (1 + 1e-3)
    assert rel_l2(x, x_ref) <= 1e-8
    if mode == stag.CG_RELIABLE:
        assert sts[0]["n_updates"] >= 1 and sts[0]["iters_f32"] == sts[0]["iters"]


def test_slab_cg_one_rank_equals_whole_lattice_solver_bitwise():
    """nranks = 1: the global sums have one term, so the slab path must reproduce the one-GPU
    solver's iterates exactly (same kernels' arithmetic, same reduction order) -- kernel-per-step
    paths on both sides; the persistent kernels sum in another order (tests/test_gpu_persistent.py)."""
    import torch
    cfg = fieldgen.CONFIGS["c1_4^4"]
    W, b = cfg.links(), cfg.source()
    L = stag.Links(cfg.dims, W)
    bd = stag.spinor_pack(b, cfg.dims, 0)
    for mode in (stag.CG_F64, stag.CG_RELIABLE):
        x1, st1 = stag.cg_solve(bd, L, cfg.mass, cfg.tol, cfg.maxiter, mode, persistent=False)
        S = make_slabs(cfg.dims, W, 1)
        xs, sts = slab.cg_solve_in_process(S, [bd], cfg.mass, cfg.tol, cfg.maxiter, mode)
        assert sts[0]["iters"] == st1["iters"] and sts[0]["n_updates"] == st1["n_updates"]
        assert torch.equal(xs[0], x1)


def test_slab_cg_degenerate_cases():
    cfg = fieldgen.CONFIGS["c1_4^4"]
    W, b = cfg.links(), cfg.source()
    # b = 0 -> x = 0, no iterations
    x, sts = _slab_cg(cfg, W, np.zeros_like(b), 2, stag.CG_RELIABLE)
    assert not x.any() and sts[0]["iters"] == 0 and sts[0]["status"] == stag.OK
    # maxiter = 3 -> ENOCONV with the true residual reported, same on both ranks
    slabs = make_slabs(cfg.dims, W, 2)
    bs = [stag.spinor_pack(np.ascontiguousarray(slab.scatter_spinor(b, cfg.dims, r, 2)), slabs[r].dims, 0) for r in range(2)]
    xs, sts = slab.cg_solve_in_process(slabs, bs, cfg.mass, cfg.tol, 3, stag.CG_RELIABLE)
    assert sts[0]["status"] == stag.ENOCONV and sts[0]["iters"] == 3 and sts[0]["true_resid"] > cfg.tol
    assert sts[0]["true_resid"] == sts[1]["true_resid"]
    x = slab.gather_spinor([stag.spinor_unpack(xs[r], slabs[r].dims, 0) for r in range(2)], cfg.dims)
    res = np.linalg.norm((b - oracle.apply_A(x, W, cfg.dims, cfg.mass)).ravel()) / np.linalg.norm(b.ravel())
    assert abs(res - sts[0]["true_resid"]) <= 1e-12 * max(1.0, res)
    # a plane-wave source on the free field converges in one iteration on four ranks
    cfgf = fieldgen.CONFIGS["c2_8^4_free"]
    pw = fieldgen.spinor_planewave(cfgf.dims, (1, 2, 3, 0))
    x, sts = _slab_cg(cfgf, cfgf.links(), pw, 4, stag.CG_F64)
    assert sts[0]["iters"] == 1 and rel_l2(x, pw / 8.588286437626904) <= 1e-12


def test_slab_cg_run_single_call_on_one_rank():
    """stag_slab_cg_run (the call of a one-process-per-GPU run) on a one-slab decomposition:
    same iterates as the stepped loop."""
    import torch
    cfg = fieldgen.CONFIGS["c1_4^4"]
    W, b = cfg.links(), cfg.source()
    bd = stag.spinor_pack(b, cfg.dims, 0)
    S = make_slabs(cfg.dims, W, 1)
    xs, sts = slab.cg_solve_in_process(S, [bd], cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE)
    x, st = S[0].cg_solve(bd, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE)
    assert st["iters"] == sts[0]["iters"] and torch.equal(x, xs[0])


@pytest.mark.slow
@pytest.mark.parametrize("nranks", [2, 4, 8])
def test_slab_hop_full_size_bitwise_against_whole_lattice(nranks):
    """bench configuration (28^3 x 96) split into 2, 4, 8 slabs on one device: both hops in the
    precisions of the timed solve must reproduce the whole-lattice kernel bit for bit."""
    import torch
    cfg = fieldgen.CONFIGS["c4_28^3x96"]
    W = cfg.links()
    L = stag.Links(cfg.dims, W)
    slabs = make_slabs(cfg.dims, W, nranks)
    del W
    chi = cfg.source()
    for prec in (stag.PREC_F32_R12, stag.PREC_F64):
        whole1 = stag.dslash(stag.spinor_pack(chi, cfg.dims, prec), L, 1, prec)
        w1 = stag.spinor_unpack(whole1, cfg.dims, prec)
        outs, got = slab_hop_all(slabs, chi, cfg.dims, 1, prec)
        assert np.array_equal(got, w1)
        whole0 = stag.spinor_unpack(stag.dslash(whole1, L, 0, prec), cfg.dims, prec)
        _, got0 = slab_hop_all(slabs, w1, cfg.dims, 0, prec)
        assert np.array_equal(got0, whole0)
    for s in slabs:
        s.close()
    L.close()


def test_watchdog_turns_a_missing_push_into_an_error_instead_of_a_hang():
    """Two slabs; only rank 0 pushes, then rank 0 hops: its boundary threads wait for flags rank 1
    never sets.  With the wait limit lowered the kernel must give up, the slab must report
    STAG_ETIMEOUT, and the interior of the result (which needs no neighbour) must still be right."""
    dims = (4, 4, 4, 8)
    W = fieldgen.links(dims, "random", seed=61)
    slabs = make_slabs(dims, W, 2)
    chi = fieldgen.spinor_gaussian(dims, 0, seed=62)
    prec = stag.PREC_F64
    v0 = stag.spinor_pack(np.ascontiguousarray(slab.scatter_spinor(chi, dims, 0, 2)), slabs[0].dims, prec)
    slabs[0].set_wait_limit(2000)                      # ~ a millisecond
    assert slabs[0].status() == stag.OK
    slabs[0].push(v0, prec)                            # rank 1 never pushes
    out = stag.spinor_unpack(slabs[0].hop(v0, 1, prec), slabs[0].dims, prec)
    assert slabs[0].status() == stag.ETIMEOUT
    ref = slab.scatter_spinor(oracle.dslash(chi, W, dims, 1), dims, 0, 2)
    s3 = slab.slice_sites(dims)
    assert rel_l2(out[s3:-s3], ref[s3:-s3]) <= 1e-13   # slices 1 .. Tl-2 need no halo
    # the CG entry points report it too
    import torch
    x = torch.zeros_like(v0)
    slabs[0].cg_begin(x, v0, 0.1, 1e-10, 10, stag.CG_F64)
    with pytest.raises(stag.StagError) as e:
        slabs[0].cg_control()      # ACT_NORM needs no status read; the next control call does
        ph = 0
        while slabs[0].cg_step(slab.ACT_NORM, ph):
            ph += 1
        slabs[0].cg_control()
    assert e.value.status == stag.ETIMEOUT


def _random_slab_cases(n, seed):
    rng = np.random.default_rng(seed)
    cases = []
    while len(cases) < n:
        dims = tuple(int(v) for v in rng.choice([2, 4, 6], size=3)) + (int(rng.choice([4, 8, 12, 16, 24])),)
        nranks = int(rng.choice([r for r in (1, 2, 3, 4, 6) if dims[3] % r == 0 and (dims[3] // r) % 2 == 0]))
        if np.prod(dims) <= 5000:
            cases.append((dims, nranks, int(rng.integers(1, 10**6))))
    return cases


@pytest.mark.parametrize("dims,nranks,seed", _random_slab_cases(12, 2011))
def test_slab_hop_and_cg_on_randomly_drawn_decompositions(dims, nranks, seed):
    """A dozen lattices and slab counts drawn with a fixed seed: both hops bitwise against the
    whole-lattice kernel, and the mixed slab CG against the oracle's A."""
    W = fieldgen.links(dims, "random", seed=seed)
    L = stag.Links(dims, W)
    slabs = make_slabs(dims, W, nranks)
    for parity in (0, 1):
        chi = fieldgen.spinor_gaussian(dims, 1 - parity, seed=seed + parity)
        for prec in (stag.PREC_F64, stag.PREC_F32_R12):
            _, got = slab_hop_all(slabs, chi, dims, parity, prec)
            whole = stag.spinor_unpack(stag.dslash(stag.spinor_pack(chi, dims, prec), L, parity, prec), dims, prec)
            assert np.array_equal(got, whole)
    b = fieldgen.spinor_gaussian(dims, 0, seed=seed + 7)
    bs = [stag.spinor_pack(np.ascontiguousarray(slab.scatter_spinor(b, dims, r, nranks)), slabs[r].dims, 0) for r in range(nranks)]
    xs, sts = slab.cg_solve_in_process(slabs, bs, 0.2, 1e-10, 5000, stag.CG_RELIABLE, recon12=True)
    x = slab.gather_spinor([stag.spinor_unpack(xs[r], slabs[r].dims, 0) for r in range(nranks)], dims)
    assert all(st["status"] == stag.OK for st in sts)
    res = np.linalg.norm((b - oracle.apply_A(x, W, dims, 0.2)).ravel()) / np.linalg.norm(b.ravel())
    assert res <= 1e-10 * (1 + 1e-3)
