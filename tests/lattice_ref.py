"""Test-only numpy helpers written from the definitions, independent of both
the C oracle and the CUDA path: site indexing, a dense D built column by
column from eq. 2.4, and gauge transformations."""
import itertools

import numpy as np


def volume(dims):
    return int(np.prod(dims))


def sites(dims):
    """All coordinates (x0,x1,x2,x3), x0 fastest."""
    X0, X1, X2, X3 = dims
    for x3 in range(X3):
        for x2 in range(X2):
            for x1 in range(X1):
                for x0 in range(X0):
                    yield (x0, x1, x2, x3)


def lex(dims, x):
    return x[0] + dims[0] * (x[1] + dims[1] * (x[2] + dims[2] * x[3]))


def parity(x):
    return sum(x) & 1


def cb(dims, x):
    return lex(dims, x) >> 1


def full_index(dims, x):
    """Row of the dense full-lattice operator: even block first, then odd."""
    vh = volume(dims) // 2
    return (parity(x) * vh + cb(dims, x)) * 3


def dense_D(W, dims):
    """Dense 3V x 3V matrix of eq. 2.4: D_{x,y} = W_mu(x) d_{y,x+mu} - W_mu(x-mu)^dag d_{y,x-mu}.
    Contributions are ADDED, so coinciding neighbours (X_mu = 2) both count."""
    n = 3 * volume(dims)
    D = np.zeros((n, n), dtype=np.complex128)
    for x in sites(dims):
        r = full_index(dims, x)
        for mu in range(4):
            xf = list(x); xf[mu] = (x[mu] + 1) % dims[mu]
            xb = list(x); xb[mu] = (x[mu] - 1) % dims[mu]
            cf, cbk = full_index(dims, xf), full_index(dims, xb)
            D[r:r + 3, cf:cf + 3] += W[mu, parity(x), cb(dims, x)]
            D[r:r + 3, cbk:cbk + 3] -= W[mu, parity(xb), cb(dims, xb)].conj().T
    return D


def gauge_transform_links(W, G, dims):
    """W'_mu(x) = G(x) W_mu(x) G(x+mu)^dag."""
    Wp = np.empty_like(W)
    for x in sites(dims):
        p, c = parity(x), cb(dims, x)
        for mu in range(4):
            xf = list(x); xf[mu] = (x[mu] + 1) % dims[mu]
            Wp[mu, p, c] = G[p, c] @ W[mu, p, c] @ G[parity(xf), cb(dims, xf)].conj().T
    return Wp


def gauge_transform_spinor(chi, G, par):
    """chi'(x) = G(x) chi(x) on one parity."""
    return np.einsum("sij,sj->si", G[par], chi)


def eta(x, mu):
    return -1.0 if (sum(x[:mu]) & 1) else 1.0
