"""Pins for the oracle's full-lattice operator M = D + m and its solve (Q23), no GPU.

M is not written in the paper; it is the operator whose normal equations are the paper's
A = -D^2 + m^2 (eq. 2.3) once D^dag = -D (eq. 2.4).  The pins below fix
every piece against something other than the oracle itself: an independent dense numpy
construction (tests/lattice_ref.py), the already-pinned A, LAPACK, and closed forms."""
import numpy as np
import pytest

import fieldgen
import oracle
from tests import lattice_ref as L


def _rel(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


def _full_gaussian(dims, seed):
    return np.ascontiguousarray(np.stack([fieldgen.spinor_gaussian(dims, 0, seed),
                                          fieldgen.spinor_gaussian(dims, 1, seed + 1)]))


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 2, 4)])
def test_apply_M_matches_dense_D_plus_m(dims):
    """Brute force: dense D from eq. 2.4 (even block first, then odd) plus m on the diagonal."""
    m = 0.37
    W = fieldgen.links(dims, "random", seed=5)
    psi = _full_gaussian(dims, 50)
    M = L.dense_D(W, dims) + m * np.eye(3 * L.volume(dims))
    ref = (M @ psi.ravel()).reshape(psi.shape)
    assert _rel(oracle.apply_M(psi, W, dims, m), ref) < 1e-14


def test_normal_equations_are_A_on_even_sites():
    """(D+m)^dag (D+m) = A and it does not mix parities: for psi supported on even sites,
    M^dag M psi = (A psi_e, 0), with M^dag phi = 2 m phi - M phi."""
    dims, m = (4, 4, 4, 4), 0.2
    W = fieldgen.links(dims, "random", seed=6)
    psi = _full_gaussian(dims, 60)
    psi[1] = 0
    Mpsi = oracle.apply_M(psi, W, dims, m)
    MdM = 2 * m * Mpsi - oracle.apply_M(Mpsi, W, dims, m)
    A = oracle.apply_A(np.ascontiguousarray(psi[0]), W, dims, m)
    assert _rel(MdM[0], A) < 1e-13
    assert np.linalg.norm(MdM[1]) < 1e-13 * np.linalg.norm(A)


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (2, 4, 2, 4)])
def test_solve_M_matches_dense_lapack(dims):
    m = 0.1
    W = fieldgen.links(dims, "random", seed=7)
    h = _full_gaussian(dims, 70)
    M = L.dense_D(W, dims) + m * np.eye(3 * L.volume(dims))
    ref = np.linalg.solve(M, h.ravel()).reshape(h.shape)
    psi, it, rho, rc = oracle.solve_M(h, W, dims, m, 1e-13, 4000)
    assert rc == 0 and rho < 1e-11
    assert _rel(psi, ref) < 1e-11


def test_solve_M_residual_on_4444():
    """|h - (D+m) psi| / |h| recomputed here with apply_M; bounded by tol |b_e| / (m |h|)."""
    dims, m, tol = (4, 4, 4, 4), 0.1, 1e-10
    W = fieldgen.links(dims, "random", seed=8)
    h = _full_gaussian(dims, 80)
    psi, it, rho, rc = oracle.solve_M(h, W, dims, m, tol, 4000)
    assert rc == 0 and it > 10
    res = _rel(oracle.apply_M(psi, W, dims, m), h)
    assert abs(res - rho) < 1e-13
    # residual of M psi = h lives on the even sites only: M^dag r = (b_e - A psi_e, 0) and the odd rows
    # hold exactly, so |r| <= |b_e - A psi_e| / m  (sigma_min(M) = sqrt(lambda_min(A)) >= m)
    b_e = m * h[0] - oracle.dslash(np.ascontiguousarray(h[1]), W, dims, 0)
    assert res <= tol * np.linalg.norm(b_e) / (m * np.linalg.norm(h)) * (1 + 1e-6)


def test_solve_M_zero_links_is_division_by_m():
    dims, m = (4, 4, 4, 4), 0.5
    W = np.zeros((4, 2, 128, 3, 3), dtype=np.complex128)
    h = _full_gaussian(dims, 90)
    psi, it, rho, rc = oracle.solve_M(h, W, dims, m, 1e-12, 10)
    assert rc == 0 and it == 1
    assert _rel(psi, h / m) < 1e-14


def test_solve_M_is_gauge_covariant():
    """W' = G W G^dag(x+mu), h' = G h  =>  psi' = G psi."""
    dims, m = (4, 4, 4, 4), 0.15
    W = fieldgen.links(dims, "random", seed=9)
    G = fieldgen.gauge_transform(dims)
    Wp = L.gauge_transform_links(W, G, dims)
    h = _full_gaussian(dims, 100)
    hp = np.ascontiguousarray(np.stack([L.gauge_transform_spinor(h[p], G, p) for p in (0, 1)]))
    psi, _, _, rc = oracle.solve_M(h, W, dims, m, 1e-12, 4000)
    psip, _, _, rcp = oracle.solve_M(hp, Wp, dims, m, 1e-12, 4000)
    assert rc == 0 and rcp == 0
    ref = np.stack([L.gauge_transform_spinor(psi[p], G, p) for p in (0, 1)])
    assert _rel(psip, ref) < 1e-10


def test_free_field_point_source_propagator_is_translation_invariant():
    """U = 1 (eta, bc folded): the propagator from a point source at x and at x + 2 e_0 are
    translates of each other (eta is invariant under shifts by 2)."""
    dims, m = (4, 4, 4, 4), 0.3
    W = fieldgen.links(dims, "unit")
    vh = 128
    h1 = np.zeros((2, vh, 3), dtype=np.complex128)
    h2 = np.zeros((2, vh, 3), dtype=np.complex128)
    x1, x2 = (0, 1, 2, 1), (2, 1, 2, 1)
    h1[L.parity(x1), L.cb(dims, x1), 1] = 1.0
    h2[L.parity(x2), L.cb(dims, x2), 1] = 1.0
    p1, _, _, _ = oracle.solve_M(h1, W, dims, m, 1e-13, 1000)
    p2, _, _, _ = oracle.solve_M(h2, W, dims, m, 1e-13, 1000)
    for x in L.sites(dims):
        xs = ((x[0] + 2) % dims[0], x[1], x[2], x[3])
        a = p1[L.parity(x), L.cb(dims, x)]
        b = p2[L.parity(xs), L.cb(dims, xs)]
        assert np.allclose(a, b, atol=1e-11)
