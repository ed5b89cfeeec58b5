"""The N > 1 path of bench.py is 'replicas only': the host-side
aggregation is exercised here with two gloo ranks on CPU."""
import os
import socket

import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update({"RANK": str(rank), "LOCAL_RANK": str(rank), "WORLD_SIZE": str(world),
                       "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    from paper_1111_0125_b200 import replicas
    r, l, w = replicas.init("gloo")
    assert (r, l, w) == (rank, rank, world)
    replicas.barrier()
    # rank r processed (r+1)*100 units in (r+1) seconds
    agg = replicas.aggregate_throughput(100.0 * (rank + 1), 1.0 * (rank + 1))
    seeds = replicas.replica_seed(7, rank)
    q.put((rank, agg, seeds, replicas.max_over_ranks(rank), replicas.sum_over_ranks(1.0)))
    replicas.finalize()


def test_two_rank_aggregation_over_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, agg, seed, mx, sm in out:
        assert agg["units"] == 300.0 and agg["seconds"] == 2.0 and agg["throughput"] == 150.0
        assert mx == 1.0 and sm == 2.0
    assert out[0][2] != out[1][2]          # each replica gets its own right-hand side


def test_single_process_defaults():
    from paper_1111_0125_b200 import replicas
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        os.environ.pop(k, None)
    assert replicas.env_world() == (0, 0, 1)
    assert replicas.aggregate_throughput(10.0, 2.0)["throughput"] == 5.0
    assert replicas.max_over_ranks(3.5) == 3.5
