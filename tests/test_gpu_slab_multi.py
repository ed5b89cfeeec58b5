"""The T-slab path with ONE GPU PER RANK and no fences between phases: kernels of different ranks
really run at the same time and wait for each other through the exchange regions.  Needs at
least two visible GPUs; skipped otherwise (this round's boxes have one -- everything up to real
concurrency is covered by test_gpu_slab.py and test_gpu_slab_ipc.py)."""
import os
import socket

import numpy as np
import pytest
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu

DIMS, MASS, TOL = (8, 8, 8, 16), 0.05, 1e-10


def _ngpus():
    try:
        import torch
        return torch.cuda.device_count() if torch.cuda.is_available() else 0
    except Exception:
        return 0


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    try:
        import torch
        import torch.distributed as dist
        import fieldgen
        import oracle
        import paper_1111_0125_b200 as stag
        from paper_1111_0125_b200 import slab
        os.environ.update({"MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
        torch.cuda.set_device(rank)
        dist.init_process_group("nccl", rank=rank, world_size=world)
        W = fieldgen.links(DIMS, "random", seed=11)                # for the oracle; the slab sees only its own slices
        b = fieldgen.spinor_gaussian(DIMS, 0, seed=12)
        t0, t1 = slab.slab_range(DIMS, rank, world)
        S = slab.SlabLinks(DIMS, fieldgen.links_slices(DIMS, t0, t1 - t0, "random", seed=11), rank, world,
                           W_back=np.ascontiguousarray(fieldgen.links_slices(DIMS, t0 - 1, 1, "random", seed=11)[3]))
        S.connect_distributed()
        S.set_wait_limit(1 << 22)

        from tests.parity import rel_err as rel      # L2 AND worst-site bound (tests/parity.py)

        # all the CPU work first (the oracle's solve takes a different time on every rank), then a barrier
        # before every first exchange: rank skew counts against the slab watchdog (include/stag.h)
        ref = slab.scatter_spinor(oracle.dslash(b, W, DIMS, 1), DIMS, rank, world)
        x_ref, _, _, _, _ = oracle.cg(b, W, DIMS, MASS, 1e-12, 50000)
        for prec, tol in ((0, 1e-13), (3, 2e-6)):
            v = stag.spinor_pack(np.ascontiguousarray(slab.scatter_spinor(b, DIMS, rank, world)), S.dims, prec)
            torch.cuda.synchronize()
            dist.barrier()
            for rep in range(20):                      # back to back, no host synchronisation
                o = S.dslash(v, 1, prec)
            assert rel(stag.spinor_unpack(o, S.dims, prec), ref) <= tol
        out = {}
        for mode, persistent in ((stag.CG_F64, False), (stag.CG_RELIABLE, False), (stag.CG_F64, True), (stag.CG_RELIABLE, True)):
            bd = stag.spinor_pack(np.ascontiguousarray(slab.scatter_spinor(b, DIMS, rank, world)), S.dims, 0)
            torch.cuda.synchronize()
            dist.barrier()
            # stag_slab_cg_run: graph replays of the kernel-per-step pass, or the persistent kernel with the
            # reliable updates inside; real waits on the other GPUs either way
            x, st = S.cg_solve(bd, MASS, TOL, 20000, mode, persistent=persistent)
            assert st["status"] == stag.OK and st["true_resid"] <= TOL, st
            assert rel(stag.spinor_unpack(x, S.dims, 0), slab.scatter_spinor(x_ref, DIMS, rank, world)) <= 1e-8
            out[(mode, persistent)] = (st["iters"], st["true_resid"], st["n_updates"])
        assert S.status() == stag.OK
        torch.cuda.synchronize()
        dist.barrier()
        S.close()
        dist.destroy_process_group()
        q.put((rank, "ok", out))
    except Exception:
        import traceback
        q.put((rank, "fail", traceback.format_exc()))
        raise


@pytest.mark.skipif(_ngpus() < 2, reason="needs two GPUs (one per rank)")
@pytest.mark.parametrize("world", [2, 4, 8])
def test_slab_hop_and_cg_with_one_gpu_per_rank(world):
    if _ngpus() < world:
        pytest.skip("needs %d GPUs" % world)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = {}
    for _ in procs:
        rank, status, payload = q.get(timeout=900)
        assert status == "ok", payload
        got[rank] = payload
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    for r in range(1, world):
        assert got[r] == got[0]            # identical scalars on every rank
