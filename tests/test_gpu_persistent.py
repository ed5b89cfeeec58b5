"""The CG iteration as one persistent cooperative kernel per chunk of passes (stag_persist.cuh,
params.persistent = 1): grid barriers instead of four kernel boundaries per pass, replicated
scalars.  Same bars as the kernel-per-step path: the solution against the oracle's solve (1e-8),
the true residual recomputed with the oracle's A, iteration counts within a few per cent (Q17: the
summation order differs, the iterates are not compared)."""
import numpy as np
import pytest

import fieldgen
import oracle
import paper_1111_0125_b200 as stag
from tests.parity import rel_err

pytestmark = pytest.mark.gpu

# ragged volumes (pads), an extent of 2 (both neighbours the same site), more tiles than warps
LATTICES = [((4, 4, 4, 4), 0.1), ((6, 4, 2, 10), 0.1), ((2, 2, 2, 4), 0.2), ((8, 8, 8, 8), 0.05), ((16, 8, 8, 12), 0.05)]


def _true_resid(x, b, W, dims, mass):
    return float(np.linalg.norm((b - oracle.apply_A(x, W, dims, mass)).ravel()) / np.linalg.norm(b.ravel()))


@pytest.mark.parametrize("dims,mass", LATTICES)
@pytest.mark.parametrize("mode,recon12", [(stag.CG_F64, False), (stag.CG_F64, True), (stag.CG_RELIABLE, False),
                                          (stag.CG_RELIABLE, True), (stag.CG_DEFECT, True)])
def test_persistent_iteration_matches_oracle(dims, mass, mode, recon12):
    tol = 1e-10
    W = fieldgen.links(dims, "random", seed=81)
    b = fieldgen.spinor_gaussian(dims, 0, seed=82)
    x_ref, it_ref, _, _, rc = oracle.cg(b, W, dims, mass, 1e-12, 50000)
    assert rc == 0
    L = stag.Links(dims, W)
    bd = stag.spinor_pack(b, dims, 0)
    x, st = stag.cg_solve(bd, L, mass, tol, 20000, mode, recon12=recon12, persistent=True, persist_chunk=37)
    assert st["status"] == stag.OK and st["true_resid"] <= tol, st
    xs = stag.spinor_unpack(x, dims, 0)
    assert rel_err(xs, x_ref) <= 1e-8
    assert _true_resid(xs, b, W, dims, mass) <= tol * (1 + 1e-3)
    # pads of the solution stay zero
    vh = int(np.prod(dims)) // 2
    planes = x.view(3, -1, 2)
    if planes.shape[1] > vh:
        assert float(planes[:, vh:, :].abs().max()) == 0.0
    # against the kernel-per-step path: same algorithm, other summation order
    x2, st2 = stag.cg_solve(bd, L, mass, tol, 20000, mode, recon12=recon12, persistent=False)
    assert abs(st["iters"] - st2["iters"]) <= max(3, 0.05 * st2["iters"]), (st["iters"], st2["iters"])
    assert rel_err(xs, stag.spinor_unpack(x2, dims, 0)) <= 1e-8
    L.close()


def test_persistent_degenerate_cases():
    dims, mass = (4, 4, 4, 4), 0.1
    W = fieldgen.links(dims, "random", seed=83)
    L = stag.Links(dims, W)
    b = fieldgen.spinor_gaussian(dims, 0, seed=84)
    bd = stag.spinor_pack(b, dims, 0)
    import torch
    # b = 0 -> x = 0, no iteration
    x, st = stag.cg_solve(torch.zeros_like(bd), L, mass, 1e-10, 100, stag.CG_RELIABLE, persistent=True)
    assert st["status"] == stag.OK and st["iters"] == 0 and float(x.abs().max()) == 0.0
    # maxiter reached: reported, x and the true residual still written; chunk larger and smaller than maxiter
    for chunk in (4, 1000):
        x, st = stag.cg_solve(bd, L, mass, 1e-10, 10, stag.CG_RELIABLE, persistent=True, persist_chunk=chunk)
        assert st["status"] == stag.ENOCONV and st["iters"] == 10 and st["true_resid"] > 1e-10
        xs = stag.spinor_unpack(x, dims, 0)
        assert abs(_true_resid(xs, b, W, dims, mass) - st["true_resid"]) <= 1e-6 * st["true_resid"]
    # maxiter = 0
    x, st = stag.cg_solve(bd, L, mass, 1e-10, 0, stag.CG_F64, persistent=True)
    assert st["iters"] == 0 and st["status"] == stag.ENOCONV
    # a plane-wave source on the free field converges in exactly one pass (closed form, SURVEY pin 3)
    dims8 = (8, 8, 8, 8)
    Wf = fieldgen.links(dims8, "unit")
    Lf = stag.Links(dims8, Wf)
    pw = fieldgen.spinor_planewave(dims8, (1, 2, 3, 0))
    x, st = stag.cg_solve(stag.spinor_pack(pw, dims8, 0), Lf, 0.05, 1e-10, 100, stag.CG_F64, persistent=True)
    lam = 0.05 ** 2 + 4 * (np.sin(2 * np.pi * 1 / 8) ** 2 + np.sin(2 * np.pi * 2 / 8) ** 2 + np.sin(2 * np.pi * 3 / 8) ** 2
                           + np.sin(2 * np.pi * 0.5 / 8) ** 2)
    assert st["iters"] == 1 and rel_err(stag.spinor_unpack(x, dims8, 0), pw / lam) <= 1e-12
    L.close()
    Lf.close()


def test_persistent_is_bit_reproducible_and_independent_of_the_chunk():
    dims, mass = (8, 8, 8, 8), 0.05
    W = fieldgen.links(dims, "random", seed=85)
    L = stag.Links(dims, W)
    bd = stag.spinor_pack(fieldgen.spinor_gaussian(dims, 0, seed=86), dims, 0)
    runs = [stag.cg_solve(bd, L, mass, 1e-10, 20000, stag.CG_RELIABLE, recon12=True, persistent=True, persist_chunk=c)
            for c in (1024, 1024, 5)]
    for x, st in runs[1:]:
        assert st["iters"] == runs[0][1]["iters"] and bool((x == runs[0][0]).all())
    L.close()


def test_mixed_solve_is_one_launch_with_the_reliable_updates_inside_the_kernel():
    """Mode 3, fp64 corrections on 18-real links: the trigger of P:L97 is served inside the persistent
    kernel (x += y, r = b - A x in fp64, beta from the corrected residual), so after the initial
    residual the whole solve is ONE launch -- counted -- and still meets every bar."""
    dims, mass, tol = (8, 8, 8, 8), 0.05, 1e-10
    W = fieldgen.links(dims, "random", seed=87)
    b = fieldgen.spinor_gaussian(dims, 0, seed=88)
    x_ref, _, _, _, rc = oracle.cg(b, W, dims, mass, 1e-12, 50000)
    assert rc == 0
    L = stag.Links(dims, W)
    bd = stag.spinor_pack(b, dims, 0)
    stag.cg_solve(bd, L, mass, tol, 20000, stag.CG_RELIABLE, recon12=True, persistent=True)     # derive the link forms
    stag.reset_launch_count()
    x, st = stag.cg_solve(bd, L, mass, tol, 20000, stag.CG_RELIABLE, recon12=True, persistent=True, persist_chunk=100000)
    launches = stag.launch_count()
    assert st["status"] == stag.OK and st["true_resid"] <= tol
    assert st["n_updates"] >= 3 and st["applies_f64"] == st["n_updates"] + 1      # the initial residual + one per update
    assert launches <= 6, launches        # |b|^2, two hops and the residual of r0, the persistent kernel: no launch per update
    xs = stag.spinor_unpack(x, dims, 0)
    assert rel_err(xs, x_ref) <= 1e-8
    assert _true_resid(xs, b, W, dims, mass) <= tol * (1 + 1e-3)
    # Fig. 2's outer steps (mode 2) run inside the kernel the same way
    stag.reset_launch_count()
    xd, std = stag.cg_solve(bd, L, mass, tol, 20000, stag.CG_DEFECT, recon12=True, persistent=True, persist_chunk=100000)
    assert stag.launch_count() <= 6 and std["status"] == stag.OK and std["n_updates"] >= 2
    assert std["applies_f64"] == std["n_updates"] + 1
    assert rel_err(stag.spinor_unpack(xd, dims, 0), x_ref) <= 1e-8
    # with 12-real fp64 corrections the update stays on the host: more launches, same solution within the bars
    stag.reset_launch_count()
    x2, st2 = stag.cg_solve(bd, L, mass, tol, 20000, stag.CG_RELIABLE, recon12=True, recon12_f64=True, persistent=True)
    assert stag.launch_count() > launches and st2["status"] == stag.OK
    assert rel_err(stag.spinor_unpack(x2, dims, 0), x_ref) <= 1e-8
    L.close()
