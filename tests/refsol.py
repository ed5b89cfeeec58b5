"""Scoring a full-size solution against a compact oracle record (tests/golden/refsol_*.npz, written
by tests/golden/make_reference_solutions.py from oracle/ alone).  The records hold x_ref at seeded
sample sites plus the projections <z_k, x_ref> on seeded Gaussian vectors; for any error field e
E |<z, e>|^2 = 2 |e|^2 (re, im of z ~ N(0,1)), so the projections estimate |x - x_ref|_2 over the
WHOLE field without the 51-255 MB vector.  No arithmetic of the method lives here."""
import os

import numpy as np

import fieldgen

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def load(name):
    path = os.path.join(GOLDEN, "refsol_%s.npz" % name.replace("^", "").replace("/", "_"))
    rec = dict(np.load(path))
    cfg = fieldgen.CONFIGS[name]
    assert str(rec["config"]) == name and tuple(int(v) for v in rec["dims"]) == tuple(cfg.dims)
    assert int(rec["link_seed"]) == fieldgen.LINK_SEED + cfg.index
    assert int(rec["source_seed"]) == fieldgen.SOURCE_SEED + cfg.index
    assert float(rec["mass"]) == cfg.mass and float(rec["true_resid"]) <= float(rec["ref_tol"]) * (1 + 1e-6)
    return rec


def score(x, rec, cfg):
    """x: canonical complex128 [Vh][3].  Returns a dict of errors relative to the reference:
    l2_sketch   estimate of |x - x_ref|_2 / |x_ref|_2 over every site, from the projections
    l2_sites    |x - x_ref|_2 / |x_ref|_2 over the sampled sites
    max_site    max over sampled sites and colours of |x - x_ref| / max |x_ref| (whole field)
    norm        | |x|_2 - |x_ref|_2 | / |x_ref|_2"""
    sites = rec["sites"]
    d = x[sites] - rec["x_sites"]
    proj = rec["proj"]
    seed0 = int(rec["sketch_seed0"])
    dp = np.array([np.vdot(fieldgen.spinor_gaussian(cfg.dims, 0, seed0 + k), x) for k in range(len(proj))]) - proj
    xn = float(rec["x_norm"])
    return {"l2_sketch": float(np.sqrt(np.mean(np.abs(dp) ** 2) / 2.0)) / xn,
            "l2_sites": float(np.linalg.norm(d.ravel()) / np.linalg.norm(rec["x_sites"].ravel())),
            "max_site": float(np.abs(d).max() / float(rec["x_absmax"])),
            "norm": abs(float(np.linalg.norm(x.ravel())) - xn) / xn}
