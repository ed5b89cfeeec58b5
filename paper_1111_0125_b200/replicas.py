"""Multi-GPU plumbing for bench.py: REPLICAS ONLY.

The single-GPU hot path has no exchange step (north_star: no halo exchange, no collectives),
so N GPUs run N independent solves (one process per GPU, different right-hand sides) and the
only communication is the barrier around the timed region and the max/sum of a few scalars.
The same code runs under `gloo` on CPU in tests/test_replicas_gloo.py.
"""
from __future__ import annotations

import os


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when absent."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str):
    """Join the process group when launched with WORLD_SIZE > 1.  Returns (rank, local, world)."""
    rank, local, world = env_world()
    if world > 1:
        import torch.distributed as dist
        if not dist.is_initialized():
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29511")
            dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local, world


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def _reduce(value: float, op_name: str, device: str) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=getattr(dist.ReduceOp, op_name))
    return float(t.item())


def max_over_ranks(value: float, device: str = "cpu") -> float:
    return _reduce(value, "MAX", device)


def sum_over_ranks(value: float, device: str = "cpu") -> float:
    return _reduce(value, "SUM", device)


def replica_seed(base_seed: int, rank: int) -> int:
    """Each replica solves for its own right-hand side."""
    return int(base_seed) + 1000003 * int(rank)


def aggregate_throughput(units_this_rank: float, seconds_this_rank: float, device: str = "cpu") -> dict:
    """Whole-job throughput: the units all ranks processed divided by the slowest rank's time."""
    total = sum_over_ranks(units_this_rank, device)
    tmax = max_over_ranks(seconds_this_rank, device)
    return {"units": total, "seconds": tmax, "throughput": total / tmax if tmax > 0 else 0.0}


def finalize():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()
