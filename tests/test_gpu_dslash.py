"""GPU parity of the Dslash hop and of A against the CPU oracle, element by element, through
the C ABI (include/stag.h).  Tolerances are BASELINE.json's: relative L2 error <= 1e-13 in
fp64 and <= 2e-6 in fp32 (the same bars for the 12-real variants)."""
import numpy as np
import pytest

import fieldgen
import oracle
import paper_1111_0125_b200 as stag

pytestmark = pytest.mark.gpu

TOL = {stag.PREC_F64: 1e-13, stag.PREC_F64_R12: 1e-13, stag.PREC_F32: 2e-6, stag.PREC_F32_R12: 2e-6}
ALL_PREC = [stag.PREC_F64, stag.PREC_F32, stag.PREC_F64_R12, stag.PREC_F32_R12]


from tests.parity import rel_err as rel_l2  # L2 AND worst-site bound (tests/parity.py)


# several tiles + ragged tails (Vh not a multiple of 32 or of the 128-thread block), extents of
# 2 (forward and backward neighbour coincide), and the small BASELINE configs
DIMS = [(4, 4, 4, 4), (2, 2, 2, 2), (6, 4, 2, 10), (2, 6, 6, 4), (8, 8, 8, 8), (10, 6, 4, 6), (4, 2, 2, 2)]


@pytest.mark.parametrize("dims", DIMS)
@pytest.mark.parametrize("prec", ALL_PREC)
@pytest.mark.parametrize("parity", [0, 1])
def test_dslash_matches_oracle(dims, prec, parity):
    W = fieldgen.links(dims, "random", seed=11)
    chi = fieldgen.spinor_gaussian(dims, 1 - parity, seed=12)
    ref = oracle.dslash(chi, W, dims, parity)
    L = stag.Links(dims, W)
    out = stag.spinor_unpack(stag.dslash(stag.spinor_pack(chi, dims, prec), L, parity, prec), dims, prec)
    assert rel_l2(out, ref) <= TOL[prec]


@pytest.mark.parametrize("prec", ALL_PREC)
def test_dslash_periodic_time_boundary(prec):
    """antiperiodic_t = 0: the 12-real sign rebuild must not assume a boundary sign."""
    dims = (4, 4, 2, 6)
    W = fieldgen.links(dims, "random", seed=5, antiperiodic_t=False)
    chi = fieldgen.spinor_gaussian(dims, 0, seed=6)
    L = stag.Links(dims, W, antiperiodic_t=False)
    out = stag.spinor_unpack(stag.dslash(stag.spinor_pack(chi, dims, prec), L, 1, prec), dims, prec)
    assert rel_l2(out, oracle.dslash(chi, W, dims, 1)) <= TOL[prec]


def test_pack_unpack_roundtrip_and_pad_is_zero():
    dims = (6, 4, 2, 10)          # Vh = 240, Vh_pad = 256
    chi = fieldgen.spinor_gaussian(dims, 0, seed=3)
    v = stag.spinor_pack(chi, dims, stag.PREC_F64)
    assert v.numel() == 6 * 256
    planes = v.view(3, 256, 2)
    assert float(planes[:, 240:, :].abs().max()) == 0.0
    assert np.array_equal(stag.spinor_unpack(v, dims, stag.PREC_F64), chi)
    v32 = stag.spinor_pack(chi, dims, stag.PREC_F32)
    assert np.array_equal(stag.spinor_unpack(v32, dims, stag.PREC_F32), chi.astype(np.complex64).astype(np.complex128))


def test_dslash_keeps_pad_lanes_zero():
    dims = (6, 4, 2, 10)
    W = fieldgen.links(dims, "random", seed=1)
    chi = fieldgen.spinor_gaussian(dims, 0, seed=2)
    L = stag.Links(dims, W)
    for prec in ALL_PREC:
        out = stag.empty_spinor(dims, prec)
        out.fill_(float("nan"))
        stag.dslash(stag.spinor_pack(chi, dims, prec), L, 1, prec, out=out)
        assert float(out.view(3, 256, 2)[:, 240:, :].abs().max()) == 0.0


def test_twelve_real_links_refused_when_not_special_unitary():
    dims = (4, 4, 4, 4)
    rng = np.random.default_rng(0)
    W = rng.normal(size=(4, 2, 128, 3, 3)) + 1j * rng.normal(size=(4, 2, 128, 3, 3))
    chi = fieldgen.spinor_gaussian(dims, 0, seed=2)
    L = stag.Links(dims, W)
    assert L.recon_error() > 1e-3
    out = stag.spinor_unpack(stag.dslash(stag.spinor_pack(chi, dims, stag.PREC_F64), L, 1, stag.PREC_F64), dims, stag.PREC_F64)
    assert rel_l2(out, oracle.dslash(chi, W, dims, 1)) <= 1e-13   # 18-real works for any W
    with pytest.raises(stag.StagError) as e:
        stag.dslash(stag.spinor_pack(chi, dims, stag.PREC_F32_R12), L, 1, stag.PREC_F32_R12)
    assert e.value.status == stag.EINVAL


def test_recon_error_is_rounding_for_folded_su3_links():
    dims = (4, 6, 4, 8)
    for kind, eps in (("random", 0.0), ("smooth", 0.5), ("unit", 0.0)):
        L = stag.Links(dims, fieldgen.links(dims, kind, seed=9, eps=eps))
        assert L.recon_error() < 1e-14


def test_links_from_device_memory_match_links_from_host():
    import torch
    dims = (4, 4, 6, 4)
    W = fieldgen.links(dims, "random", seed=21)
    chi = fieldgen.spinor_gaussian(dims, 0, seed=22)
    Wd = torch.from_numpy(W.view(np.float64).reshape(-1)).cuda()
    a = stag.dslash(stag.spinor_pack(chi, dims, stag.PREC_F64), stag.Links(dims, W), 1, stag.PREC_F64)
    b = stag.dslash(stag.spinor_pack(chi, dims, stag.PREC_F64), stag.Links(dims, Wd), 1, stag.PREC_F64)
    assert torch.equal(a, b)


def test_argument_errors_on_device():
    dims = (4, 4, 4, 4)
    L = stag.Links(dims, fieldgen.links(dims, "random", seed=1))
    v = stag.spinor_pack(fieldgen.spinor_gaussian(dims, 0, seed=2), dims, stag.PREC_F64)
    with pytest.raises(stag.StagError):
        stag.dslash(v, L, 1, stag.PREC_F64, out=v)            # out aliases in
    with pytest.raises(stag.StagError):
        stag.dslash(v, L, 2, stag.PREC_F64)                   # bad parity
    with pytest.raises(stag.StagError):
        stag.dslash(v, L, 1, 9, out=stag.empty_spinor(dims, 0))  # bad precision
    L2 = stag.Links((4, 4, 4, 6), fieldgen.links((4, 4, 4, 6), "random", seed=1))
    import ctypes
    out = stag.empty_spinor(dims, stag.PREC_F64)
    rc = stag.lib().stag_dslash(ctypes.c_void_p(out.data_ptr()), ctypes.c_void_p(v.data_ptr()),
                                L2.handle, 1, (ctypes.c_int * 4)(*dims), 0)
    assert rc == stag.EINVAL                                  # dims != the handle's


@pytest.mark.parametrize("name", ["c1_4^4", "c2_8^4_free", "c2_8^4", "c3_16^3x32"])
@pytest.mark.parametrize("prec", ALL_PREC)
def test_apply_A_matches_oracle_on_baseline_configs(name, prec):
    cfg = fieldgen.CONFIGS[name]
    W, b = cfg.links(), cfg.source()
    ref = oracle.apply_A(b, W, cfg.dims, cfg.mass)
    L = stag.Links(cfg.dims, W)
    out = stag.spinor_unpack(stag.apply_A(stag.spinor_pack(b, cfg.dims, prec), L, cfg.mass, prec), cfg.dims, prec)
    assert rel_l2(out, ref) <= TOL[prec]


def test_free_field_plane_wave_eigenvalue_on_gpu():
    """BASELINE configs[1]: A chi = (m^2 + 4 sum sin^2 p_mu) chi for plane waves on U = 1."""
    dims, m = (8, 8, 8, 8), 0.05
    W = fieldgen.links(dims, "unit")
    L = stag.Links(dims, W)
    for n in [(0, 0, 0, 0), (1, 2, 3, 0), (3, 1, 0, 5)]:
        chi = fieldgen.spinor_planewave(dims, n)
        p = [2 * np.pi * (n[mu] + (0.5 if mu == 3 else 0.0)) / dims[mu] for mu in range(4)]
        lam = m * m + 4 * sum(np.sin(pm) ** 2 for pm in p)
        out = stag.spinor_unpack(stag.apply_A(stag.spinor_pack(chi, dims, 0), L, m, 0), dims, 0)
        assert rel_l2(out, lam * chi) <= 1e-13


@pytest.mark.slow
@pytest.mark.parametrize("name", ["c4_28^3x96", "c5_48^3x96"])
def test_dslash_full_size_matches_oracle(name):
    """The bench configuration (and the largest one): all four precisions, both hops, every
    output site compared with the oracle's hop on the same seeded field."""
    cfg = fieldgen.CONFIGS[name]
    W = cfg.links()
    chi = cfg.source()
    L = stag.Links(cfg.dims, W)
    ref1 = oracle.dslash(chi, W, cfg.dims, 1)
    ref0 = oracle.dslash(ref1, W, cfg.dims, 0)
    del W
    for prec in ALL_PREC:
        o1 = stag.spinor_unpack(stag.dslash(stag.spinor_pack(chi, cfg.dims, prec), L, 1, prec), cfg.dims, prec)
        assert rel_l2(o1, ref1) <= TOL[prec]
        o0 = stag.spinor_unpack(stag.dslash(stag.spinor_pack(ref1, cfg.dims, prec), L, 0, prec), cfg.dims, prec)
        assert rel_l2(o0, ref0) <= TOL[prec]
    L.close()


@pytest.mark.parametrize("antiperiodic", [True, False])
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (6, 4, 2, 10), (2, 2, 2, 2)])
def test_device_side_phase_folding_is_bit_identical_to_the_generator(dims, antiperiodic):
    """stag_links_create_unfolded folds eta*bc on the device; +-1 is exact, so both hops
    in all four precisions give the bits of the handle built from the pre-folded field, and the
    fp64 result still matches the oracle (which only ever sees the folded field)."""
    import torch
    U = fieldgen.links(dims, "random", seed=77, fold=False, antiperiodic_t=antiperiodic)
    W = fieldgen.links(dims, "random", seed=77, fold=True, antiperiodic_t=antiperiodic)
    La = stag.Links(dims, W, antiperiodic_t=antiperiodic)
    Lb = stag.Links(dims, U, antiperiodic_t=antiperiodic, folded=False)
    assert Lb.recon_error() < 1e-14
    for parity in (0, 1):
        chi = fieldgen.spinor_gaussian(dims, 1 - parity, seed=78)
        for prec in ALL_PREC:
            v = stag.spinor_pack(chi, dims, prec)
            assert torch.equal(stag.dslash(v, La, parity, prec), stag.dslash(v, Lb, parity, prec))
        out = stag.spinor_unpack(stag.dslash(stag.spinor_pack(chi, dims, 0), Lb, parity, 0), dims, 0)
        assert rel_l2(out, oracle.dslash(chi, W, dims, parity)) <= 1e-13


# ---- the 8-parameter link form ---------------------------------
# Tolerances: fp64 keeps 1e-11 (the rebuild divides by N = |a2|^2+|a3|^2, which amplifies the
# 1e-16 rounding of the stored slots by 1/N; measured <= 8e-14 down to eps = 0.05 smooth links);
# fp32 gets 5e-6, NOT the 2e-6 of the other fp32 forms: measured 4.7e-7 (random SU(3)) to 1.9e-6
# (smooth eps = 0.3), single rebuilt entries off by up to 4e-4 -- the round-off the paper rejects
# the form for.
TOL8 = {stag.PREC_F64_R8: 1e-11, stag.PREC_F32_R8: 5e-6}


def check8(out, ref, chi, L, prec):
    """Relative L2 error within TOL8, and the worst component within the bound the form's own
    measured accuracy implies: a rebuilt entry is off by at most E = stag_links_recon8_error
    (largest entry error, measured at setup in the hop's arithmetic), an output component sums
    8 directions x 3 columns of (entry x chi), so |out - ref| <= 24 E max|chi| on top of the
    rounding bar every other form meets (tests/parity.py with c = 1)."""
    from tests.parity import max_site, rel_l2 as l2
    assert l2(out, ref) <= TOL8[prec]
    rounding = 1e-13 if prec == stag.PREC_F64_R8 else 2e-6
    assert np.abs(out - ref).max() <= rounding * np.abs(ref).max() + 24 * L.recon8_error(prec) * np.abs(chi).max()


@pytest.mark.parametrize("kind,eps", [("random", 0.0), ("smooth", 0.5), ("smooth", 0.3)])
@pytest.mark.parametrize("prec", [stag.PREC_F64_R8, stag.PREC_F32_R8])
@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (6, 4, 2, 10)])
def test_eight_parameter_hop_matches_oracle(dims, prec, kind, eps):
    W = fieldgen.links(dims, kind, seed=5, eps=eps)
    L = stag.Links(dims, W)
    for parity in (0, 1):
        chi = fieldgen.spinor_gaussian(dims, 1 - parity, seed=6 + parity)
        out = stag.spinor_unpack(stag.dslash(stag.spinor_pack(chi, dims, prec), L, parity, prec), dims, prec)
        check8(out, oracle.dslash(chi, W, dims, parity), chi, L, prec)
    assert L.recon8_error(prec) <= (1e-9 if prec == stag.PREC_F64_R8 else 1e-3)


def test_eight_parameter_periodic_boundary_and_apply_A():
    dims = (4, 4, 2, 6)
    W = fieldgen.links(dims, "random", seed=5, antiperiodic_t=False)
    L = stag.Links(dims, W, antiperiodic_t=False)
    chi = fieldgen.spinor_gaussian(dims, 0, seed=6)
    for prec in (stag.PREC_F64_R8, stag.PREC_F32_R8):
        out = stag.spinor_unpack(stag.apply_A(stag.spinor_pack(chi, dims, prec), L, 0.1, prec), dims, prec)
        # two hops: the first hop's error passes through the second (|M| <= 1 per entry, 24 terms)
        from tests.parity import rel_l2 as l2
        ref = oracle.apply_A(chi, W, dims, 0.1)
        assert l2(out, ref) <= TOL8[prec]
        bound = 24 * L.recon8_error(prec) * (np.abs(chi).max() + np.abs(oracle.dslash(chi, W, dims, 1)).max())
        assert np.abs(out - ref).max() <= (1e-13 if prec == stag.PREC_F64_R8 else 2e-6) * np.abs(ref).max() + 25 * bound


def test_eight_parameter_form_refused_where_it_does_not_exist():
    """Unit links have first row (1,0,0): N = 0, no 8-parameter form; nearly-unit links lose all
    fp32 accuracy.  Both must be refused with STAG_EINVAL, never silently wrong."""
    dims = (4, 4, 4, 4)
    chi = fieldgen.spinor_gaussian(dims, 0, seed=2)
    L = stag.Links(dims, fieldgen.links(dims, "unit"))
    for prec in (stag.PREC_F64_R8, stag.PREC_F32_R8):
        with pytest.raises(stag.StagError) as e:
            stag.dslash(stag.spinor_pack(chi, dims, prec), L, 1, prec)
        assert e.value.status == stag.EINVAL
    L2 = stag.Links(dims, fieldgen.links(dims, "smooth", seed=3, eps=0.003))
    with pytest.raises(stag.StagError):
        stag.dslash(stag.spinor_pack(chi, dims, stag.PREC_F32_R8), L2, 1, stag.PREC_F32_R8)
    rng = np.random.default_rng(0)
    L3 = stag.Links(dims, rng.normal(size=(4, 2, 128, 3, 3)) + 1j * rng.normal(size=(4, 2, 128, 3, 3)))
    with pytest.raises(stag.StagError):
        stag.dslash(stag.spinor_pack(chi, dims, stag.PREC_F64_R8), L3, 1, stag.PREC_F64_R8)


def _random_cases(n, seed):
    rng = np.random.default_rng(seed)
    cases = []
    while len(cases) < n:
        dims = tuple(int(v) for v in rng.choice([2, 4, 6, 8, 10, 12], size=4))
        if np.prod(dims) <= 6000:
            cases.append((dims, int(rng.integers(0, 2)), bool(rng.integers(0, 2)), int(rng.integers(1, 10**6))))
    return cases


@pytest.mark.parametrize("dims,parity,antiperiodic,seed", _random_cases(24, 20111125))
def test_hop_on_randomly_drawn_small_lattices(dims, parity, antiperiodic, seed):
    """Two dozen lattices drawn from even extents 2..12 (fixed seed): every mixture of extents of 2
    (coinciding neighbours), ragged volumes and boundary conditions, all storage forms, single and
    batch entry, against the oracle."""
    W = fieldgen.links(dims, "random", seed=seed, antiperiodic_t=antiperiodic)
    L = stag.Links(dims, W, antiperiodic_t=antiperiodic)
    chis = [fieldgen.spinor_gaussian(dims, 1 - parity, seed=seed + 1 + k) for k in range(3)]
    refs = [oracle.dslash(c, W, dims, parity) for c in chis]
    for prec in ALL_PREC + [stag.PREC_F64_R8, stag.PREC_F32_R8]:
        tol = TOL.get(prec) or TOL8[prec]
        out = stag.spinor_unpack(stag.dslash(stag.spinor_pack(chis[0], dims, prec), L, parity, prec), dims, prec)
        assert rel_l2(out, refs[0]) <= tol, (prec, dims)
        if prec in ALL_PREC:
            outs = stag.dslash_mrhs(stag.spinor_pack_mrhs(chis, dims, prec), L, parity, prec)
            for k, o in enumerate(stag.spinor_unpack_mrhs(outs, dims, prec)):
                assert rel_l2(o, refs[k]) <= tol, (prec, dims, k)
