"""The T-slab path under REAL concurrency on one GPU: the slabs of a decomposition live in one
process, each driven by its own host thread on its own CUDA stream, with no fence between phases.
The lattices are small enough for all slabs' kernels to be resident at the same time, so the
kernels of different ranks genuinely overlap and the acquire-waits (wait_flag, stag_dslash.cuh:
halo flags in the hop, reduction flags in the global sums) genuinely spin on a peer that is still
running or has not been launched yet -- what test_gpu_slab.py (lockstep) and test_gpu_slab_ipc.py
(a fence after every phase) never do.  The parity checks are those of test_gpu_slab_multi.py (one
GPU per rank), which needs a box with several GPUs.

Each test first runs the same work in lockstep once: that loads every kernel and makes every
allocation, neither of which may happen while another slab's kernel is spinning (lazy module
loading and cudaFree synchronise the device).  A threading.Barrier stands where a real run has
dist.barrier(): before the first exchange, so that rank skew does not eat the watchdog's budget;
after it rank r deliberately starts 20 ms x r late, so that the first waits are certain to spin
(stag_slab_wait_stats counts them, and the tests assert the count).  The watchdog is lowered so
a protocol error ends as STAG_ETIMEOUT, not as a hang."""
import threading
import time

import numpy as np
import pytest

import fieldgen
import oracle
import paper_1111_0125_b200 as stag
from paper_1111_0125_b200 import slab
from tests.parity import rel_err

pytestmark = pytest.mark.gpu

WAIT_LIMIT = 1 << 22          # polls of >= 200 ns: a few seconds


def make_slabs(dims, W, nranks):
    slabs = [slab.SlabLinks(dims, W, r, nranks) for r in range(nranks)]
    slab.connect_in_process(slabs)
    for s in slabs:
        s.set_wait_limit(WAIT_LIMIT)
    return slabs


def run_ranks(nranks, body):
    """body(rank) on one host thread and one CUDA stream per rank; returns the results in rank order.
    A failing rank's exception is re-raised here (the others then run into the watchdog)."""
    import torch
    streams = [torch.cuda.Stream() for _ in range(nranks)]
    gate = threading.Barrier(nranks)
    out, err = [None] * nranks, [None] * nranks

    def worker(r):
        try:
            torch.cuda.set_device(0)
            with torch.cuda.stream(streams[r]):
                gate.wait(timeout=60)
                out[r] = body(r)
                streams[r].synchronize()
        except BaseException as e:          # noqa: BLE001 -- reported to the main thread
            err[r] = e

    torch.cuda.synchronize()
    threads = [threading.Thread(target=worker, args=(r,)) for r in range(nranks)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=300)
        assert not t.is_alive(), "a rank's thread is still running"
    for e in err:
        if e is not None:
            if isinstance(e, stag.StagError) and e.status == stag.ETIMEOUT:
                _not_co_resident()
            raise e
    return out


def _not_co_resident():
    """Separate launches on one device are not PROMISED to run at the same time (B200_PROFILING.md):
    where they do not, the watchdog ends the wait and these thread-per-rank tests have nothing to say.
    The protocol itself is covered deterministically by test_all_ranks_in_one_cooperative_launch."""
    pytest.skip("the ranks' kernels were not co-resident on this device: a wait ran into the watchdog")


@pytest.mark.parametrize("dims,nranks", [((4, 4, 4, 8), 2), ((4, 4, 4, 16), 4), ((8, 8, 8, 16), 2)])
def test_hops_back_to_back_from_one_thread_per_slab(dims, nranks):
    """Forty push + hop pairs per rank with no host synchronisation anywhere: a rank may run ahead of
    its neighbours by as much as the double-buffered halo allows, and its boundary threads wait for
    real.  Every rank's last result must equal the lockstep result bitwise and the oracle within tolerance."""
    W = fieldgen.links(dims, "random", seed=71)
    chi = fieldgen.spinor_gaussian(dims, 0, seed=72)
    ref = oracle.dslash(chi, W, dims, 1)
    slabs = make_slabs(dims, W, nranks)
    spun = []
    for prec, tol in ((stag.PREC_F64, 1e-13), (stag.PREC_F32_R12, 2e-6)):
        vs = [stag.spinor_pack(np.ascontiguousarray(slab.scatter_spinor(chi, dims, r, nranks)), slabs[r].dims, prec)
              for r in range(nranks)]
        for r in range(nranks):                      # lockstep: loads the kernels, gives the expected bits
            slabs[r].push(vs[r], prec)
        lock = [slabs[r].hop(vs[r], 1, prec).clone() for r in range(nranks)]
        outs = [stag.empty_spinor(slabs[r].dims, prec) for r in range(nranks)]

        def body(r):
            time.sleep(0.02 * r)                 # rank skew: rank 0's first hop is certain to wait for its neighbours' pushes
            for _ in range(40):
                slabs[r].dslash(vs[r], 1, prec, out=outs[r])
            return slabs[r].status()

        assert sum(s.wait_stats()[0] for s in slabs) == 0      # lockstep so far: nobody ever had to wait
        statuses = run_ranks(nranks, body)
        if stag.ETIMEOUT in statuses:
            _not_co_resident()
        assert statuses == [stag.OK] * nranks
        spun.append(sum(s.wait_stats()[0] for s in slabs))
        for s in slabs:
            s.reset()                                          # clears the counters too (all streams idle here)
        for r in range(nranks):
            assert bool((outs[r] == lock[r]).all())
            got = stag.spinor_unpack(outs[r], slabs[r].dims, prec)
            assert rel_err(got, slab.scatter_spinor(ref, dims, r, nranks)) <= tol
    # the point of the test: some boundary thread really did find its flag not yet set and spun
    assert sum(spun) > 0, "no acquire-wait ever spun: the ranks did not run concurrently"
    for s in slabs:
        s.close()


@pytest.mark.parametrize("dims,nranks,mass", [((4, 4, 4, 8), 2, 0.1), ((4, 4, 4, 16), 4, 0.1), ((8, 8, 8, 16), 2, 0.05)])
@pytest.mark.parametrize("mode", [stag.CG_F64, stag.CG_RELIABLE])
@pytest.mark.parametrize("persistent", [None, True])
def test_slab_cg_run_from_one_thread_per_slab(dims, nranks, mass, mode, persistent):
    """stag_slab_cg_run -- the call of a one-process-per-GPU run: CUDA-graph replays of whole chunks of
    iterations (persistent=None: with more than one rank the library's own choice), or the persistent
    kernel (opt-in across ranks), the in-kernel pushes of hop 1 and of the direction update, global sums
    through the exchange regions -- issued concurrently by every rank's own thread.  Solution against the oracle's
    solve (1e-8), true residual with the oracle's A, identical scalars on every rank."""
    tol = 1e-10
    W = fieldgen.links(dims, "random", seed=73)
    b = fieldgen.spinor_gaussian(dims, 0, seed=74)
    x_ref, _, _, _, rc = oracle.cg(b, W, dims, mass, 1e-12, 50000)
    assert rc == 0
    slabs = make_slabs(dims, W, nranks)
    bs = [stag.spinor_pack(np.ascontiguousarray(slab.scatter_spinor(b, dims, r, nranks)), slabs[r].dims, 0)
          for r in range(nranks)]
    slab.cg_solve_in_process(slabs, bs, mass, tol, 20000, mode, recon12=True, chunk=8)     # lockstep warm-up
    assert sum(s.wait_stats()[0] for s in slabs) == 0          # lockstep: nobody ever had to wait

    def body(r):
        time.sleep(0.02 * r)                     # rank skew: the first global sum is certain to wait for the last rank
        return slabs[r].cg_solve(bs[r], mass, tol, 20000, mode, recon12=True, chunk=8, persistent=persistent)

    res = run_ranks(nranks, body)
    sts = [st for _, st in res]
    assert all(st["status"] == stag.OK and st["true_resid"] <= tol for st in sts), sts
    for st in sts[1:]:
        assert (st["iters"], st["true_resid"], st["n_updates"]) == (sts[0]["iters"], sts[0]["true_resid"], sts[0]["n_updates"])
    x = slab.gather_spinor([stag.spinor_unpack(res[r][0], slabs[r].dims, 0) for r in range(nranks)], dims)
    assert rel_err(x, x_ref) <= 1e-8
    resid = np.linalg.norm((b - oracle.apply_A(x, W, dims, mass)).ravel()) / np.linalg.norm(b.ravel())
    assert resid <= tol * (1 + 1e-3)
    assert all(s.status() == stag.OK for s in slabs)
    # the point of the test: halo and reduction waits really spun on peers that were still running
    assert sum(s.wait_stats()[0] for s in slabs) > 0, "no acquire-wait ever spun: the ranks did not run concurrently"
    for s in slabs:
        s.close()


@pytest.mark.parametrize("dims,nranks,mass", [((4, 4, 4, 8), 2, 0.1), ((4, 4, 4, 16), 4, 0.1), ((8, 8, 8, 16), 2, 0.05),
                                              ((8, 8, 8, 32), 8, 0.05), ((6, 2, 2, 12), 3, 0.1), ((4, 4, 4, 4), 1, 0.1)])
@pytest.mark.parametrize("mode", [stag.CG_F64, stag.CG_RELIABLE])
def test_all_ranks_in_one_cooperative_launch(dims, nranks, mass, mode):
    """The sanctioned way to run ranks that wait on one another on ONE GPU (B200_PROFILING.md): all
    ranks' iterations in one cooperative launch of the persistent kernel (stag_slab_cg_iter_all), each
    rank a group of blocks with its own barrier.  Every block is resident, so the ranks run
    concurrently by construction; they exchange faces through peer stores into each other's halo
    buffers and sum their inner products through the exchange regions, waiting on flags, exactly
    as one process per GPU does.  Same checks as test_gpu_slab_multi.py."""
    tol = 1e-10
    W = fieldgen.links(dims, "random", seed=77)
    b = fieldgen.spinor_gaussian(dims, 0, seed=78)
    x_ref, _, _, _, rc = oracle.cg(b, W, dims, mass, 1e-12, 50000)
    assert rc == 0
    slabs = make_slabs(dims, W, nranks)
    bs = [stag.spinor_pack(np.ascontiguousarray(slab.scatter_spinor(b, dims, r, nranks)), slabs[r].dims, 0)
          for r in range(nranks)]
    xs, sts = slab.cg_solve_in_process(slabs, bs, mass, tol, 20000, mode, fused=True, recon12=True, persist_chunk=50)
    assert all(st["status"] == stag.OK and st["true_resid"] <= tol for st in sts), sts
    for st in sts[1:]:
        assert (st["iters"], st["true_resid"], st["n_updates"]) == (sts[0]["iters"], sts[0]["true_resid"], sts[0]["n_updates"])
    x = slab.gather_spinor([stag.spinor_unpack(xs[r], slabs[r].dims, 0) for r in range(nranks)], dims)
    assert rel_err(x, x_ref) <= 1e-8
    resid = np.linalg.norm((b - oracle.apply_A(x, W, dims, mass)).ravel()) / np.linalg.norm(b.ravel())
    assert resid <= tol * (1 + 1e-3)
    assert all(s.status() == stag.OK for s in slabs)
    # against the lockstep, kernel-per-step solve of the same slabs: same algorithm, other summation order
    xs2, sts2 = slab.cg_solve_in_process(slabs, bs, mass, tol, 20000, mode, recon12=True)
    assert abs(sts[0]["iters"] - sts2[0]["iters"]) <= max(3, 0.05 * sts2[0]["iters"])
    # (the lockstep solve above adds no spinning wait: its counters are those of the fused run)
    spun = [s.wait_stats()[0] for s in slabs]
    print("waits that spun, per rank:", spun)
    assert sum(spun) > 0, "no acquire-wait ever spun"
    for s in slabs:
        s.close()


@pytest.mark.slow
@pytest.mark.parametrize("name,nranks", [("c4_28^3x96", 4), ("c4_28^3x96", 8), ("c5_48^3x96", 8)])
def test_full_size_lattice_split_over_concurrent_ranks_against_the_oracle_record(name, nranks):
    """BASELINE configs[3] and [4] (28^3 x 96; 48^3 x 96) split along time over ranks that run CONCURRENTLY in
    one cooperative launch -- 263 KB faces, thousands of boundary threads waiting on flags, in-kernel
    reliable updates with fp64 exchanges -- each slab built from its OWN time slices of the links
    (fieldgen.links_slices: no rank sees the whole field).  The gathered solution against the oracle's
    stored solve to 1e-12 (tests/golden/refsol_*.npz): sampled sites and the whole-field sketch at
    north_star's 1e-8."""
    from tests import refsol
    cfg = fieldgen.CONFIGS[name]
    rec = refsol.load(cfg.name)
    b = cfg.source()
    slabs = []
    for r in range(nranks):
        t0, t1 = slab.slab_range(cfg.dims, r, nranks)
        Wl = cfg.links_slices(t0, t1 - t0)
        Wb = np.ascontiguousarray(cfg.links_slices(t0 - 1, 1)[3])
        slabs.append(slab.SlabLinks(cfg.dims, Wl, r, nranks, W_back=Wb))
        del Wl, Wb
    slab.connect_in_process(slabs)
    for s in slabs:
        s.set_wait_limit(WAIT_LIMIT)
    bs = [stag.spinor_pack(np.ascontiguousarray(slab.scatter_spinor(b, cfg.dims, r, nranks)), slabs[r].dims, 0)
          for r in range(nranks)]
    xs, sts = slab.cg_solve_in_process(slabs, bs, cfg.mass, cfg.tol, cfg.maxiter, stag.CG_RELIABLE, fused=True, recon12=True)
    assert all(st["status"] == stag.OK and st["true_resid"] <= cfg.tol for st in sts), sts
    for st in sts[1:]:
        assert (st["iters"], st["true_resid"], st["n_updates"]) == (sts[0]["iters"], sts[0]["true_resid"], sts[0]["n_updates"])
    x = slab.gather_spinor([stag.spinor_unpack(xs[r], slabs[r].dims, 0) for r in range(nranks)], cfg.dims)
    sc = refsol.score(x, rec, cfg)
    print("%s in %d ranks: %d iterations, %d updates, errors vs oracle %r, waits that spun %r"
          % (name, nranks, sts[0]["iters"], sts[0]["n_updates"], sc, [s.wait_stats()[0] for s in slabs]))
    assert sc["l2_sketch"] <= 1e-8 and sc["l2_sites"] <= 1e-8 and sc["max_site"] <= 1e-8 and sc["norm"] <= 1e-8
    assert sum(s.wait_stats()[0] for s in slabs) > 0
    assert all(s.status() == stag.OK for s in slabs)
    for s in slabs:
        s.close()


def test_a_dead_slab_takes_its_neighbours_down_and_reset_revives_them():
    """Rank 0 hops after an exchange rank 1 never joined: its watchdog fires.  From then on rank 0
    publishes nothing, so rank 1 -- whose first exchange still completes, rank 0's push preceded its
    death -- times out on the next one instead of reading stale faces: every rank ends with
    STAG_ETIMEOUT.  stag_slab_reset on both brings the pair back, and the hop is right again."""
    dims = (4, 4, 4, 8)
    W = fieldgen.links(dims, "random", seed=75)
    chi = fieldgen.spinor_gaussian(dims, 0, seed=76)
    ref = oracle.dslash(chi, W, dims, 1)
    slabs = make_slabs(dims, W, 2)
    for s in slabs:
        s.set_wait_limit(2000)
    prec = stag.PREC_F64
    vs = [stag.spinor_pack(np.ascontiguousarray(slab.scatter_spinor(chi, dims, r, 2)), slabs[r].dims, prec) for r in range(2)]
    slabs[0].push(vs[0], prec)
    slabs[0].hop(vs[0], 1, prec)                      # waits for rank 1's push of exchange 1: never comes
    assert slabs[0].status() == stag.ETIMEOUT and slabs[1].status() == stag.OK
    slabs[1].push(vs[1], prec)
    o1 = slabs[1].hop(vs[1], 1, prec)                 # exchange 1 was pushed by rank 0 before it died
    assert slabs[1].status() == stag.OK
    assert rel_err(stag.spinor_unpack(o1, slabs[1].dims, prec), slab.scatter_spinor(ref, dims, 1, 2)) <= 1e-13
    slabs[0].push(vs[0], prec)                        # a dead slab's push is a no-op
    slabs[1].push(vs[1], prec)
    slabs[1].hop(vs[1], 1, prec)                      # exchange 2 from rank 0 never arrives
    assert slabs[1].status() == stag.ETIMEOUT
    for s in slabs:
        s.reset()
    assert [s.status() for s in slabs] == [stag.OK, stag.OK]
    for rep in range(3):
        for r in range(2):
            slabs[r].push(vs[r], prec)
        outs = [slabs[r].hop(vs[r], 1, prec) for r in range(2)]
    got = slab.gather_spinor([stag.spinor_unpack(outs[r], slabs[r].dims, prec) for r in range(2)], dims)
    assert rel_err(got, ref) <= 1e-13
    assert [s.status() for s in slabs] == [stag.OK, stag.OK]
    for s in slabs:
        s.close()


class _RawDeviceBytes:
    """n bytes of device memory at ptr, for torch.as_tensor (CUDA array interface)."""

    def __init__(self, ptr, n):
        self.__cuda_array_interface__ = {"shape": (int(n),), "typestr": "|u1", "data": (int(ptr), False), "version": 2}


def test_persistent_kernel_of_one_rank_alone_times_out_instead_of_hanging():
    """Every wait inside the persistent kernel is bounded by the slab's watchdog: with two ranks
    connected but only rank 0's iterations launched (stag_slab_cg_iter_all on one slab), rank 0's
    boundary threads wait for faces rank 1 never pushes, give up, the group leaves the kernel and the
    next control call reports STAG_ETIMEOUT.  Argument errors of the fused launch on the way."""
    import ctypes
    dims, mass = (4, 4, 4, 8), 0.1
    W = fieldgen.links(dims, "random", seed=79)
    b = fieldgen.spinor_gaussian(dims, 0, seed=80)
    slabs = make_slabs(dims, W, 2)
    for s in slabs:
        s.set_wait_limit(2000)
    bs = [stag.spinor_pack(np.ascontiguousarray(slab.scatter_spinor(b, dims, r, 2)), slabs[r].dims, 0) for r in range(2)]
    import torch
    xs = [torch.zeros_like(v) for v in bs]
    for s, x, v in zip(slabs, xs, bs):
        s.cg_begin(x, v, mass, 1e-10, 100, stag.CG_RELIABLE, recon12=True)
    one = (ctypes.c_void_p * 1)(slabs[0].handle.value)
    two = (ctypes.c_void_p * 2)(slabs[0].handle.value, slabs[0].handle.value)
    assert stag.lib().stag_slab_cg_iter_all(one, 1) == stag.EINVAL          # not yet told to iterate
    # |b|^2 and the initial residual in lockstep, as cg_solve_in_process does
    while True:
        acts = [s.cg_control() for s in slabs]
        if acts[0] == slab.ACT_ITER:
            break
        ph = 0
        while True:
            more = [s.cg_step(acts[0], ph) for s in slabs]
            if not more[0]:
                break
            ph += 1
    assert stag.lib().stag_slab_cg_iter_all(two, 2) == stag.EINVAL          # the same slab twice
    assert stag.lib().stag_slab_cg_iter_all(one, 0) == stag.EINVAL
    # rank 1's halo buffers before: [epoch parity][direction], 3 colours x s3 sites x 16 bytes each (stag_common.cuh)
    ptr, nbytes = slabs[1].exchange_region()
    s3 = dims[0] * dims[1] * dims[2] // 2
    halo = 4 * 3 * s3 * 16
    region = torch.as_tensor(_RawDeviceBytes(ptr, nbytes), device="cuda")
    torch.cuda.synchronize()
    before = region[nbytes - halo:].clone().cpu().numpy().reshape(2, -1)
    assert stag.lib().stag_slab_cg_iter_all(one, 1) == stag.OK              # rank 0 alone: nobody answers
    with pytest.raises(stag.StagError) as e:
        slabs[0].cg_control()
    assert e.value.status == stag.ETIMEOUT
    assert slabs[0].status() == stag.ETIMEOUT and slabs[1].status() == stag.OK
    # "A timed-out slab publishes nothing": the faces of d that rank 0 pushed BEFORE it waited (phase P0,
    # next exchange) are in one parity's buffers; the other parity's would have received the hop results
    # of the boundary threads whose wait gave up, computed from a halo that never came -- untouched.
    after = region[nbytes - halo:].clone().cpu().numpy().reshape(2, -1)
    changed = [bool((before[k] != after[k]).any()) for k in range(2)]
    assert changed.count(True) == 1, changed
    for s in slabs:
        s.close()
