"""Pins for the oracle's Dslash and A (no GPU): every check here is fixed by the
paper or by mathematics, none by the oracle itself."""
import numpy as np
import pytest

import fieldgen
import oracle
from tests import lattice_ref as L
from tests.golden.load import paper_values


def _vdot(a, b):
    return np.vdot(a.ravel(), b.ravel())


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 4, 6, 4), (6, 2, 2, 8)])
def test_anti_hermiticity(dims):
    """D^dag = -D by construction of eq. 2.4: phi_o^dag (D_oe chi_e) = -(D_eo phi_o)^dag chi_e."""
    W = fieldgen.links(dims, "random", seed=1)
    chi_e = fieldgen.spinor_gaussian(dims, 0, seed=2)
    phi_o = fieldgen.spinor_gaussian(dims, 1, seed=3)
    lhs = _vdot(phi_o, oracle.dslash(chi_e, W, dims, 1))
    rhs = -_vdot(oracle.dslash(phi_o, W, dims, 0), chi_e)
    assert abs(lhs - rhs) <= 1e-13 * abs(lhs)


def test_anti_hermiticity_holds_for_arbitrary_links():
    """Every link is shared by the forward hop from x and the backward hop from x+mu,
    so D^dag = -D for ANY W, unitary or not."""
    dims = (4, 4, 2, 4)
    rng = np.random.default_rng(0)
    vh = L.volume(dims) // 2
    W = rng.normal(size=(4, 2, vh, 3, 3)) + 1j * rng.normal(size=(4, 2, vh, 3, 3))
    chi_e = fieldgen.spinor_gaussian(dims, 0, seed=2)
    phi_o = fieldgen.spinor_gaussian(dims, 1, seed=3)
    lhs = _vdot(phi_o, oracle.dslash(chi_e, W, dims, 1))
    rhs = -_vdot(oracle.dslash(phi_o, W, dims, 0), chi_e)
    assert abs(lhs - rhs) <= 1e-13 * abs(lhs)


def test_positivity_identity():
    """chi^dag A chi = m^2 |chi|^2 + |D_oe chi|^2, real: A is Hermitian positive definite."""
    dims, m = (4, 4, 4, 6), 0.1
    W = fieldgen.links(dims, "random", seed=4)
    chi = fieldgen.spinor_gaussian(dims, 0, seed=5)
    q = _vdot(chi, oracle.apply_A(chi, W, dims, m))
    ref = m * m * _vdot(chi, chi).real + _vdot(*(2 * [oracle.dslash(chi, W, dims, 1)])).real
    assert abs(q.imag) <= 1e-13 * abs(q)
    assert abs(q.real - ref) <= 1e-13 * ref


def test_A_is_hermitian():
    dims, m = (4, 2, 4, 4), 0.3
    W = fieldgen.links(dims, "smooth", seed=4, eps=0.4)
    a = fieldgen.spinor_gaussian(dims, 0, seed=5)
    b = fieldgen.spinor_gaussian(dims, 0, seed=6)
    lhs = _vdot(a, oracle.apply_A(b, W, dims, m))
    rhs = _vdot(oracle.apply_A(a, W, dims, m), b)
    assert abs(lhs - rhs) <= 1e-13 * abs(lhs)


FREE_CASES = [
    ((8, 8, 8, 8), 0.05, (0, 0, 0, 0)),
    ((8, 8, 8, 8), 0.05, (1, 2, 3, 0)),
    ((8, 8, 8, 8), 0.05, (3, 1, 0, 5)),
    ((4, 6, 4, 8), 0.2, (1, 5, 2, 3)),
    ((2, 2, 2, 2), 0.1, (1, 0, 1, 0)),
]


@pytest.mark.parametrize("dims,m,n", FREE_CASES)
def test_free_field_plane_waves_are_eigenvectors(dims, m, n):
    """U = 1 with eta and the antiperiodic time boundary folded in: plane waves on the even
    sites are eigenvectors of A with eigenvalue m^2 + 4 sum_mu sin^2 p_mu (BASELINE.json
    north_star; needs eq. 2.5 WITHOUT a factor 1/2 and the right eta convention)."""
    W = fieldgen.links(dims, "unit", fold=True, antiperiodic_t=True)
    chi = fieldgen.spinor_planewave(dims, n, parity=0, antiperiodic_t=True)
    p = [2 * np.pi * (n[mu] + (0.5 if mu == 3 else 0.0)) / dims[mu] for mu in range(4)]
    lam = m * m + 4 * sum(np.sin(pm) ** 2 for pm in p)
    out = oracle.apply_A(chi, W, dims, m)
    assert np.abs(out - lam * chi).max() <= 1e-13 * lam


def test_free_field_eigenvalue_literals():
    """The two closed-form values quoted in SURVEY.md 8c pin 3 for 8^4, m = 0.05."""
    assert abs(0.05 ** 2 + 4 * np.sin(np.pi / 8) ** 2 - 0.5882864376269049) < 1e-15
    lam = 0.05 ** 2 + 4 * (np.sin(2 * np.pi / 8) ** 2 + np.sin(4 * np.pi / 8) ** 2
                           + np.sin(6 * np.pi / 8) ** 2 + np.sin(np.pi / 8) ** 2)
    assert abs(lam - 8.588286437626904) < 1e-14
    dims = (8, 8, 8, 8)
    W = fieldgen.links(dims, "unit")
    chi = fieldgen.spinor_planewave(dims, (1, 2, 3, 0))
    out = oracle.apply_A(chi, W, dims, 0.05)
    assert np.abs(out - 8.588286437626904 * chi).max() < 1e-12


def test_free_field_wrong_eta_would_fail():
    """Without eta the cross terms of D^2 survive: the pin above really pins eta."""
    dims, m, n = (8, 8, 8, 8), 0.05, (1, 2, 3, 0)
    W = fieldgen.links(dims, "unit", fold=False)
    chi = fieldgen.spinor_planewave(dims, n, parity=0, antiperiodic_t=False)
    p = [2 * np.pi * n[mu] / dims[mu] for mu in range(4)]
    lam = m * m + 4 * sum(np.sin(pm) ** 2 for pm in p)
    out = oracle.apply_A(chi, W, dims, m)
    assert np.abs(out - lam * chi).max() > 0.1


@pytest.mark.parametrize("kind,eps", [("random", 0.0), ("smooth", 0.5)])
def test_gauge_covariance(kind, eps):
    """W' = G(x) W G(x+mu)^dag, chi' = G chi  =>  D' chi' = G (D chi) and A' chi' = G (A chi)."""
    dims, m = (4, 4, 2, 6), 0.07
    W = fieldgen.links(dims, kind, seed=7, eps=eps)
    G = fieldgen.gauge_transform(dims, seed=777)
    Wp = L.gauge_transform_links(W, G, dims)
    chi = fieldgen.spinor_gaussian(dims, 0, seed=8)
    chip = L.gauge_transform_spinor(chi, G, 0)
    d = oracle.dslash(chi, W, dims, 1)
    dp = oracle.dslash(chip, Wp, dims, 1)
    assert np.abs(dp - L.gauge_transform_spinor(d, G, 1)).max() < 1e-13
    a = oracle.apply_A(chi, W, dims, m)
    ap = oracle.apply_A(chip, Wp, dims, m)
    assert np.abs(ap - L.gauge_transform_spinor(a, G, 0)).max() < 1e-12


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (2, 4, 2, 6), (4, 2, 4, 2)])
def test_dense_brute_force(dims):
    """Dense D built column by column from eq. 2.4 by independent numpy code."""
    vh = L.volume(dims) // 2
    W = fieldgen.links(dims, "random", seed=11)
    D = L.dense_D(W, dims)
    n = 3 * vh
    assert np.abs(D + D.conj().T).max() < 1e-14              # anti-Hermitian
    assert np.abs(D[:n, :n]).max() == 0 and np.abs(D[n:, n:]).max() == 0   # no e-e, o-o blocks
    chi_e = fieldgen.spinor_gaussian(dims, 0, seed=12)
    chi_o = fieldgen.spinor_gaussian(dims, 1, seed=13)
    ref_o = (D[n:, :n] @ chi_e.ravel()).reshape(vh, 3)
    ref_e = (D[:n, n:] @ chi_o.ravel()).reshape(vh, 3)
    assert np.abs(oracle.dslash(chi_e, W, dims, 1) - ref_o).max() < 1e-13
    assert np.abs(oracle.dslash(chi_o, W, dims, 0) - ref_e).max() < 1e-13
    m = 0.1
    A = m * m * np.eye(n) - D[:n, n:] @ D[n:, :n]
    ref_A = (A @ chi_e.ravel()).reshape(vh, 3)
    assert np.abs(oracle.apply_A(chi_e, W, dims, m) - ref_A).max() < 1e-12
    ev = np.linalg.eigvalsh(A)
    assert ev.min() >= m * m - 1e-12


def test_flop_and_byte_counters_match_the_paper():
    """576 flop and 1584 bytes per site; 28^3 x 96 totals 0.6 Gflop / 1.6 GB."""
    pv = paper_values()
    dims = (4, 4, 4, 4)
    vh = L.volume(dims) // 2
    W = fieldgen.links(dims, "random", seed=1)
    chi = fieldgen.spinor_gaussian(dims, 0, seed=2)
    out, flops, nbytes = oracle.dslash_counted(chi, W, dims, 1)
    assert flops == int(pv["flops_per_site"]) * vh
    assert nbytes == int(pv["bytes_per_site"]) * vh
    assert np.array_equal(out, oracle.dslash(chi, W, dims, 1))
    vh_fine = int(pv["lattice_X"]) ** 3 * int(pv["lattice_T"]) // 2
    assert vh_fine == fieldgen.CONFIGS["c4_28^3x96"].vh
    assert round(pv["flops_per_site"] * vh_fine / 1e9, 1) == pv["dslash_flops_28c96"] / 1e9
    assert abs(pv["bytes_per_site"] * vh_fine / 1e9 - pv["dslash_bytes_28c96"] / 1e9) < 0.1


def test_paper_table1_and_smem_arithmetic():
    pv = paper_values()
    assert abs(sum(pv["table1_dp_rows_ms"]) - pv["table1_dp_total_ms"]) < 0.05
    assert abs(sum(pv["table1_sp_rows_ms"]) - pv["table1_sp_total_ms"]) < 0.05
    assert pv["smem_threads"] * 2 * 4 * 4 == pv["smem_bytes"]


def test_zero_links_give_mass_term_only():
    dims, m = (4, 4, 4, 4), 0.3
    W = np.zeros((4, 2, 128, 3, 3), dtype=np.complex128)
    chi = fieldgen.spinor_gaussian(dims, 0, seed=2)
    assert np.array_equal(oracle.apply_A(chi, W, dims, m), (m * m) * chi)


def test_bad_arguments_raise():
    W = fieldgen.links((4, 4, 4, 4), "unit")
    chi = fieldgen.spinor_gaussian((4, 4, 4, 4), 0, seed=2)
    with pytest.raises(ValueError):
        oracle.dslash(chi, W, (4, 4, 4, 4), 2)
    with pytest.raises(ValueError):
        oracle.dslash(chi[:-1], W, (4, 4, 4, 4), 0)
