"""Host-side logic of the T-slab decomposition (paper_1111_0125_b200/slab.py), no GPU: which
slices a rank owns, its neighbours, scatter / gather of canonical spinors, and the exchange of
the IPC handles between two processes over gloo.  A decomposed hop assembled from the ORACLE
applied slab by slab (each slab fed its two neighbour slices) must equal the oracle's hop on the
whole lattice: that pins the halo convention the CUDA path implements."""
import os
import socket

import numpy as np
import pytest
import torch.multiprocessing as mp

import fieldgen
import oracle
from paper_1111_0125_b200 import slab


def test_ranges_neighbours_and_errors():
    dims = (4, 4, 4, 12)
    assert slab.slab_extent(dims, 3) == 4 and slab.local_dims(dims, 3) == (4, 4, 4, 4)
    assert [slab.slab_range(dims, r, 3) for r in range(3)] == [(0, 4), (4, 8), (8, 12)]
    assert slab.neighbours(0, 3) == (2, 1) and slab.neighbours(2, 3) == (1, 0)
    assert slab.neighbours(0, 1) == (0, 0) and slab.neighbours(1, 2) == (0, 0)
    assert slab.slice_sites(dims) == 32
    for bad in (5, 4, 0):                       # 12/5 not integer; 12/4 = 3 odd; 0 ranks
        with pytest.raises(ValueError):
            slab.slab_extent(dims, bad)
    with pytest.raises(ValueError):
        slab.slab_extent((4, 4, 4, 4), 4)       # one slice per rank
    with pytest.raises(ValueError):
        slab.slab_range(dims, 3, 3)


def test_scatter_gather_round_trip_is_by_time_slice():
    dims = (4, 2, 6, 8)
    chi = fieldgen.spinor_gaussian(dims, 1, seed=3)
    parts = [slab.scatter_spinor(chi, dims, r, 2) for r in range(2)]
    assert np.array_equal(slab.gather_spinor(parts, dims), chi)
    # every site of part r really has t0 <= x3 < t1: checkerboard index -> lexicographic -> x3
    s3 = slab.slice_sites(dims)
    for r, part in enumerate(parts):
        t0, t1 = slab.slab_range(dims, r, 2)
        cb = np.arange(t0 * s3, t1 * s3)
        x3 = (2 * cb) // (dims[0] * dims[1] * dims[2])
        assert part.shape[0] == len(cb) and x3.min() == t0 and x3.max() == t1 - 1
    with pytest.raises(ValueError):
        slab.gather_spinor(parts[:1], dims)


def test_only_the_two_boundary_slices_of_a_slab_need_the_neighbours():
    """The halo convention, stated with the oracle alone: zeroing the input outside
    [t0-1, t1] (periodically) leaves the hop on slab [t0, t1) unchanged, and zeroing either
    neighbour slice changes only the adjacent boundary slice."""
    dims, nranks = (4, 4, 2, 8), 2
    W = fieldgen.links(dims, "random", seed=4)
    chi = fieldgen.spinor_gaussian(dims, 0, seed=5)
    ref = oracle.dslash(chi, W, dims, 1)
    s3 = slab.slice_sites(dims)
    for r in range(nranks):
        t0, t1 = slab.slab_range(dims, r, nranks)
        keep = np.zeros(dims[3], dtype=bool)
        for t in range(t0 - 1, t1 + 1):
            keep[t % dims[3]] = True
        masked = chi.copy().reshape(dims[3], s3, 3)
        masked[~keep] = 0
        out = oracle.dslash(np.ascontiguousarray(masked.reshape(-1, 3)), W, dims, 1)
        assert np.array_equal(slab.scatter_spinor(out, dims, r, nranks), slab.scatter_spinor(ref, dims, r, nranks))
        masked[(t0 - 1) % dims[3]] = 0                           # drop the backward neighbour slice
        out2 = oracle.dslash(np.ascontiguousarray(masked.reshape(-1, 3)), W, dims, 1).reshape(dims[3], s3, 3)
        refr = ref.reshape(dims[3], s3, 3)
        assert not np.array_equal(out2[t0], refr[t0])
        assert np.array_equal(out2[t0 + 1:t1], refr[t0 + 1:t1])


def test_a_slab_needs_only_its_own_links_and_the_t_links_of_the_slice_before_it():
    """What stag_slab_create_local is given (slab.scatter_links), stated with the oracle alone: take a
    DIFFERENT gauge field, overwrite the slab's own time slices and the t-links leaving slice t0-1
    with those of W, and the hop on the slab's sites is the hop with W -- for both parities.
    Without the t-links of slice t0-1 the slab's first slice (and only it) changes."""
    dims, nranks = (4, 2, 4, 12), 3
    W = fieldgen.links(dims, "random", seed=6)
    s3 = slab.slice_sites(dims)
    for parity in (0, 1):
        chi = fieldgen.spinor_gaussian(dims, 1 - parity, seed=7 + parity)
        ref = oracle.dslash(chi, W, dims, parity).reshape(dims[3], s3, 3)
        for r in range(nranks):
            t0, t1 = slab.slab_range(dims, r, nranks)
            Wl, Wb = slab.scatter_links(W, dims, r, nranks)
            assert Wl.shape == (4, 2, (t1 - t0) * s3, 3, 3) and Wb.shape == (2, s3, 3, 3)
            other = fieldgen.links(dims, "random", seed=99)
            other[:, :, t0 * s3:t1 * s3] = Wl
            no_back = other.copy()
            tb = (t0 - 1) % dims[3]
            other[3, :, tb * s3:(tb + 1) * s3] = Wb
            out = oracle.dslash(chi, other, dims, parity).reshape(dims[3], s3, 3)
            assert np.array_equal(out[t0:t1], ref[t0:t1])
            out2 = oracle.dslash(chi, no_back, dims, parity).reshape(dims[3], s3, 3)
            assert not np.array_equal(out2[t0], ref[t0]) and np.array_equal(out2[t0 + 1:t1], ref[t0 + 1:t1])


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ.update({"MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = bytes([rank + 1]) * slab.IPC_HANDLE_BYTES            # a stand-in for the 64-byte handle
    hb, hf = slab.exchange_handles(mine, rank, world)
    q.put((rank, hb[0], hf[0], len(hb), len(hf)))
    bad = None
    try:
        slab.exchange_handles(b"short", rank, world)
    except ValueError as e:
        bad = str(e)
    q.put((rank, "bad", bad is not None, 0, 0))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_ipc_handles_reach_the_right_neighbours_over_gloo(world):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = [q.get(timeout=180) for _ in range(2 * world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, hb, hf, nb, nf in got:
        if hb == "bad":
            assert hf is True
            continue
        b, f = slab.neighbours(rank, world)
        assert (hb, hf) == (b + 1, f + 1) and nb == nf == slab.IPC_HANDLE_BYTES
