"""How every GPU-vs-oracle comparison in tests/ is scored.

rel_err(out, ref, c) = max( |out - ref|_2 / |ref|_2 ,  max_x |out(x) - ref(x)| / (c * max_x |ref(x)|) )

The first term is north_star's metric (relative L2 error over the whole field).  On its own it lets
one wrong site hide: on 10^6 sites a single fp32 component off by 1e-3 relative moves the L2 error
by 1e-6.  The second term applies the same tolerance to the WORST component, normalised by the
largest reference component; c = 1 unless a test states otherwise with its reason.  A test asserts
rel_err(...) <= tol, i.e. both bounds at once.
"""
import numpy as np


def rel_l2(out, ref) -> float:
    return float(np.linalg.norm((out - ref).ravel()) / np.linalg.norm(ref.ravel()))


def max_site(out, ref) -> float:
    """Largest component error over the field, relative to the largest reference component."""
    return float(np.abs(out - ref).max() / np.abs(ref).max())


def rel_err(out, ref, c: float = 1.0) -> float:
    out, ref = np.asarray(out), np.asarray(ref)
    assert out.shape == ref.shape, (out.shape, ref.shape)
    if not np.all(np.isfinite(out.view(np.float64) if np.iscomplexobj(out) else out)):
        return float("inf")
    return max(rel_l2(out, ref), max_site(out, ref) / c)
