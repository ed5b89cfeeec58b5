"""Two PROCESSES, each one rank of a two-slab decomposition, wired through CUDA IPC handles
exchanged over gloo -- the multi-GPU wiring, on the one GPU this box has.  Because both ranks share
the device, every phase is followed by a stream synchronise and a barrier, so no kernel ever waits
for a kernel of the other process that has not run (with one GPU per rank that barrier is not
there).  What this adds to test_gpu_slab.py: cudaIpcGetMemHandle / OpenMemHandle, stores into
another process's allocation, and the flags' visibility across processes."""
import os
import socket

import numpy as np
import pytest
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu

DIMS, NRANKS, MASS, TOL = (4, 4, 4, 8), 2, 0.1, 1e-10


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, port, q):
    try:
        import torch
        import torch.distributed as dist
        import fieldgen
        import oracle
        import paper_1111_0125_b200 as stag
        from paper_1111_0125_b200 import slab
        os.environ.update({"MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
        dist.init_process_group("gloo", rank=rank, world_size=NRANKS)
        torch.cuda.set_device(0)
        W = fieldgen.links(DIMS, "random", seed=11)
        chi = fieldgen.spinor_gaussian(DIMS, 0, seed=12)
        S = slab.SlabLinks(DIMS, W, rank, NRANKS)
        S.connect_distributed()

        def fence():
            torch.cuda.synchronize()
            dist.barrier()

        from tests.parity import rel_err as rel      # L2 AND worst-site bound (tests/parity.py)

        out = {}
        # the hop, all four precisions, twice each (both halo buffers)
        ref = slab.scatter_spinor(oracle.dslash(chi, W, DIMS, 1), DIMS, rank, NRANKS)
        for prec, tol in ((0, 1e-13), (1, 2e-6), (2, 1e-13), (3, 2e-6)):
            v = stag.spinor_pack(np.ascontiguousarray(slab.scatter_spinor(chi, DIMS, rank, NRANKS)), S.dims, prec)
            for rep in range(2):
                S.push(v, prec)
                fence()
                o = S.hop(v, 1, prec)
                fence()
            err = rel(stag.spinor_unpack(o, S.dims, prec), ref)
            assert err <= tol, (prec, err)
            out["hop%d" % prec] = err
        # the solve, both modes
        b = chi
        x_ref, _, _, _, rc = oracle.cg(b, W, DIMS, MASS, 1e-12, 20000)
        for mode in (stag.CG_F64, stag.CG_RELIABLE):
            bd = stag.spinor_pack(np.ascontiguousarray(slab.scatter_spinor(b, DIMS, rank, NRANKS)), S.dims, 0)
            x, st = S.cg_solve(bd, MASS, TOL, 5000, mode, after_phase=fence, chunk=8)
            assert st["status"] == stag.OK and st["true_resid"] <= TOL, st
            err = rel(stag.spinor_unpack(x, S.dims, 0), slab.scatter_spinor(x_ref, DIMS, rank, NRANKS))
            assert err <= 1e-8, err
            out["cg%d" % mode] = (st["iters"], st["true_resid"], st["n_updates"])
        fence()
        S.close()
        dist.destroy_process_group()
        q.put((rank, "ok", out))
    except Exception as e:      # report instead of hanging the parent
        import traceback
        q.put((rank, "fail", traceback.format_exc()))
        raise


def test_two_processes_share_a_lattice_through_cuda_ipc():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, port, q)) for r in range(NRANKS)]
    for p in procs:
        p.start()
    got = {}
    for _ in procs:
        rank, status, payload = q.get(timeout=600)
        assert status == "ok", payload
        got[rank] = payload
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    # both ranks formed the same global scalars
    for mode in (0, 3):
        assert got[0]["cg%d" % mode] == got[1]["cg%d" % mode]
