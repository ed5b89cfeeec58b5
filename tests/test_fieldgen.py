"""The seeded input generator: SU(3)-ness, folded phases, reproducibility."""
import numpy as np
import pytest
import scipy.linalg

import fieldgen
from tests import lattice_ref as L


def _unitarity(W):
    I = np.eye(3)
    return np.abs(np.einsum("...ij,...kj->...ik", W, W.conj()) - I).max()


def test_random_links_are_su3():
    dims = (4, 6, 2, 4)
    U = fieldgen.links(dims, "random", seed=5, fold=False)
    assert _unitarity(U) < 1e-14
    assert np.abs(np.linalg.det(U) - 1.0).max() < 1e-14


def test_smooth_links_are_su3_and_near_identity():
    dims = (4, 4, 4, 4)
    U1 = fieldgen.links(dims, "smooth", seed=5, eps=0.3, fold=False)
    assert _unitarity(U1) < 1e-14
    assert np.abs(np.linalg.det(U1) - 1.0).max() < 1e-14
    U0 = fieldgen.links(dims, "smooth", seed=5, eps=1e-3, fold=False)
    assert np.abs(U0 - np.eye(3)).max() < 1e-2
    assert np.abs(U1 - np.eye(3)).max() > 0.05


def test_smooth_link_is_exp_of_the_drawn_generator():
    """U = exp(i eps H), H = (G+G^dag)/2 - tr/3 from the same counter-based draws."""
    dims = (4, 4, 4, 4)
    eps, seed = 0.5, 31
    U = fieldgen.links(dims, "smooth", seed=seed, eps=eps, fold=False)
    for x, mu in [((1, 2, 3, 0), 2), ((0, 0, 0, 0), 0), ((3, 3, 3, 3), 3)]:
        idx = L.lex(dims, x)
        g = np.array([fieldgen.normal_at(seed, 0x4C494E4B, idx * 4 + mu, k) for k in range(18)])
        G = (g[0::2] + 1j * g[1::2]).reshape(3, 3)
        H = 0.5 * (G + G.conj().T)
        H -= np.trace(H) / 3 * np.eye(3)
        ref = scipy.linalg.expm(1j * eps * H)
        assert np.abs(U[mu, L.parity(x), L.cb(dims, x)] - ref).max() < 1e-13


def test_folded_phases_match_eta_and_time_boundary():
    dims = (4, 2, 6, 4)
    U = fieldgen.links(dims, "random", seed=9, fold=False)
    W = fieldgen.links(dims, "random", seed=9, fold=True, antiperiodic_t=True)
    Wp = fieldgen.links(dims, "random", seed=9, fold=True, antiperiodic_t=False)
    for x in L.sites(dims):
        p, c = L.parity(x), L.cb(dims, x)
        for mu in range(4):
            s = L.eta(x, mu)
            assert np.array_equal(Wp[mu, p, c], s * U[mu, p, c])
            if mu == 3 and x[3] == dims[3] - 1:
                s = -s
            assert np.array_equal(W[mu, p, c], s * U[mu, p, c])


def test_unit_links_folded_are_pure_signs():
    dims = (4, 4, 4, 4)
    W = fieldgen.links(dims, "unit", fold=True)
    assert np.array_equal(np.abs(W), np.broadcast_to(np.eye(3), W.shape))


def test_reproducible_and_seed_sensitive():
    dims = (4, 4, 4, 4)
    a = fieldgen.links(dims, "random", seed=1)
    b = fieldgen.links(dims, "random", seed=1)
    c = fieldgen.links(dims, "random", seed=2)
    assert np.array_equal(a, b) and not np.array_equal(a, c)
    s1 = fieldgen.spinor_gaussian(dims, 0, seed=3)
    s2 = fieldgen.spinor_gaussian(dims, 0, seed=3)
    assert np.array_equal(s1, s2)
    assert not np.array_equal(s1, fieldgen.spinor_gaussian(dims, 1, seed=3))


def test_gaussian_source_statistics():
    chi = fieldgen.spinor_gaussian((8, 8, 8, 8), 0, seed=4)
    v = np.concatenate([chi.real.ravel(), chi.imag.ravel()])
    assert abs(v.mean()) < 0.03 and abs(v.var() - 1.0) < 0.05
    assert abs(np.mean(v ** 4) - 3.0) < 0.3


def test_planewave_values():
    dims = (4, 4, 6, 8)
    n = (1, 0, 2, 3)
    v = np.array([1.0, 0.5 - 0.25j, -0.3 + 0.8j])
    chi = fieldgen.spinor_planewave(dims, n, v, parity=0, antiperiodic_t=True)
    for x in [(0, 0, 0, 0), (1, 2, 3, 2), (3, 3, 5, 7)]:
        assert L.parity(x) == 0
        ph = 2 * np.pi * (n[0] * x[0] / 4 + n[1] * x[1] / 4 + n[2] * x[2] / 6 + (n[3] + 0.5) * x[3] / 8)
        assert np.abs(chi[L.cb(dims, x)] - np.exp(1j * ph) * v).max() < 1e-13


def test_config_table_matches_baseline_json():
    c = fieldgen.CONFIGS
    assert c["c4_28^3x96"].vh == 1053696 and c["c5_48^3x96"].vh == 5308416
    assert c["c1_4^4"].mass == 0.1 and c["c2_8^4"].mass == 0.05
    assert c["c3_16^3x32"].eps == 0.3 and c["c5_48^3x96"].eps == 0.5
    assert c["c4_28^3x96"].mass == 0.0124 and c["c5_48^3x96"].mass == 0.005


@pytest.mark.parametrize("kind,eps", [("random", 0.0), ("smooth", 0.3), ("unit", 0.0)])
def test_time_slices_generated_alone_equal_the_whole_field(kind, eps):
    """fg_links_slices: what a rank of a T-slab decomposition generates for itself is bit-identical to
    the same slices of the whole field, including a range that wraps around the time extent (the
    slice before a slab that starts at t = 0)."""
    dims = (4, 2, 6, 8)
    s3 = dims[0] * dims[1] * dims[2] // 2
    W = fieldgen.links(dims, kind, seed=17, eps=eps)
    for t0, nt in ((0, 8), (2, 4), (6, 2), (7, 1), (-1, 1)):
        part = fieldgen.links_slices(dims, t0, nt, kind, seed=17, eps=eps)
        want = np.concatenate([W[:, :, ((t0 + j) % 8) * s3:((t0 + j) % 8 + 1) * s3] for j in range(nt)], axis=2)
        assert part.shape == want.shape and np.array_equal(part, want)
