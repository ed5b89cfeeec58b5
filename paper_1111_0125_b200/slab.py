"""T-slab decomposition of the hop over several GPUs (include/stag.h "T-slabs"; DESIGN.md
section 14): host-side plumbing only.  Every number is computed by the kernels behind
stag_slab_push / stag_slab_hop; this module

  * says which time slices a rank owns and who its neighbours are (pure host logic, tested with a
    world-size-2 gloo group on CPU),
  * scatters / gathers canonical spinors between the whole lattice and the slabs (time slices are
    contiguous in the checkerboard index, so a slab's part of a one-parity spinor is one slice
    [t0*s3, (t0+Tl)*s3) of it),
  * wires the exchange regions: between processes by exchanging the 64-byte CUDA IPC handles through
    torch.distributed (one process per GPU), inside one process by handing the raw pointers over.

The paper's pipeline for the same step is boundary collect -> memcpy to host -> MPI -> memcpy to
device (Table 1); here the faces are stored straight into the neighbour GPU's memory.
"""
from __future__ import annotations

import ctypes

import paper_1111_0125_b200 as stag

IPC_HANDLE_BYTES = 64
ACT_DONE, ACT_NORM, ACT_INIT, ACT_ITER, ACT_UPDATE, ACT_VERIFY, ACT_FINAL = range(7)


# ---- pure host logic ---------------------------------------------------------------------
def slab_extent(global_dims, nranks: int) -> int:
    """Local time extent; raises unless X3 splits into nranks even slabs of >= 2 slices."""
    x3 = int(global_dims[3])
    if nranks < 1 or x3 % nranks:
        raise ValueError("X3 = %d does not split into %d slabs" % (x3, nranks))
    tl = x3 // nranks
    if tl < 2 or tl % 2:
        raise ValueError("local time extent %d must be even and >= 2" % tl)
    return tl


def slab_range(global_dims, rank: int, nranks: int):
    """(t0, t1): rank owns time slices t0 <= x3 < t1."""
    tl = slab_extent(global_dims, nranks)
    if not 0 <= rank < nranks:
        raise ValueError("rank %d outside 0..%d" % (rank, nranks - 1))
    return rank * tl, (rank + 1) * tl


def local_dims(global_dims, nranks: int):
    return (int(global_dims[0]), int(global_dims[1]), int(global_dims[2]), slab_extent(global_dims, nranks))


def neighbours(rank: int, nranks: int):
    """(backward, forward) ranks along time, periodic."""
    return (rank - 1) % nranks, (rank + 1) % nranks


def stag_vh(dims) -> int:
    """Sites of one parity."""
    v = 1
    for d in dims:
        v *= int(d)
    return v // 2


def slice_sites(global_dims) -> int:
    """s3: sites of one parity in one time slice."""
    return int(global_dims[0]) * int(global_dims[1]) * int(global_dims[2]) // 2


def scatter_spinor(chi_global, global_dims, rank: int, nranks: int):
    """The slab's part of a canonical one-parity spinor chi[cb][3] of the whole lattice."""
    t0, t1 = slab_range(global_dims, rank, nranks)
    s3 = slice_sites(global_dims)
    return chi_global[t0 * s3:t1 * s3]


def scatter_links(W_global, global_dims, rank: int, nranks: int):
    """(W_local, W_back) for stag_slab_create_local: the rank's own time slices of the canonical
    links W[mu][p][cb][3][3] and the t-links leaving the slice before the slab (slicing only)."""
    t0, t1 = slab_range(global_dims, rank, nranks)
    s3 = slice_sites(global_dims)
    tb = (t0 - 1) % int(global_dims[3])
    return W_global[:, :, t0 * s3:t1 * s3], W_global[3, :, tb * s3:(tb + 1) * s3]


def gather_spinor(parts, global_dims):
    """Inverse of scatter_spinor: parts[r] from rank r, in rank order."""
    import numpy as np
    out = np.concatenate(list(parts), axis=0)
    vh = slice_sites(global_dims) * int(global_dims[3])
    if out.shape[0] != vh:
        raise ValueError("parts hold %d sites, the lattice has %d per parity" % (out.shape[0], vh))
    return out


def all_handles(my_handle: bytes, nranks: int, group=None):
    """Every rank's IPC handle, in rank order, through torch.distributed (any backend)."""
    import torch.distributed as dist
    if len(my_handle) != IPC_HANDLE_BYTES:
        raise ValueError("an IPC handle is %d bytes" % IPC_HANDLE_BYTES)
    world = dist.get_world_size(group)
    if world != nranks:
        raise ValueError("group has %d ranks, the decomposition %d" % (world, nranks))
    allh = [None] * world
    dist.all_gather_object(allh, bytes(my_handle), group=group)
    return allh


def exchange_handles(my_handle: bytes, rank: int, nranks: int, group=None):
    """The (backward, forward) neighbours' handles."""
    allh = all_handles(my_handle, nranks, group)
    b, f = neighbours(rank, nranks)
    return allh[b], allh[f]


# ---- the handle --------------------------------------------------------------------------
class SlabLinks:
    """One rank's slab.  W: canonical complex128 links of the WHOLE lattice (stag_slab_create; only
    the rank's part goes to the device), or, with W_back given, of the rank's OWN time slices
    (stag_slab_create_local, see scatter_links): no rank then needs the whole field."""

    def __init__(self, global_dims, W, rank: int, nranks: int, antiperiodic_t: bool = True, W_back=None):
        import numpy as np
        torch = stag._require_cuda()
        stag.use_current_stream()
        self.global_dims = tuple(int(v) for v in global_dims)
        self.dims = local_dims(global_dims, nranks)
        self.rank, self.nranks = int(rank), int(nranks)
        self._h = ctypes.c_void_p()
        self._opened = []
        W = np.ascontiguousarray(W, dtype=np.complex128)
        if W_back is None:
            if W.shape[2] != stag_vh(self.global_dims):
                raise ValueError("W must cover the whole lattice when W_back is not given")
            stag._check(stag.lib().stag_slab_create(ctypes.byref(self._h), stag._cdims(self.global_dims),
                                                    int(bool(antiperiodic_t)), ctypes.c_void_p(W.ctypes.data), 0,
                                                    self.rank, self.nranks))
        else:
            Wb = np.ascontiguousarray(W_back, dtype=np.complex128)
            if W.shape[:3] != (4, 2, stag_vh(self.dims)) or Wb.shape[:2] != (2, slice_sites(self.global_dims)):
                raise ValueError("W_local / W_back have the wrong shape for this slab")
            stag._check(stag.lib().stag_slab_create_local(ctypes.byref(self._h), stag._cdims(self.global_dims),
                                                          int(bool(antiperiodic_t)), ctypes.c_void_p(W.ctypes.data),
                                                          ctypes.c_void_p(Wb.ctypes.data), 0, self.rank, self.nranks))
        torch.cuda.current_stream().synchronize()

    @property
    def handle(self):
        return self._h

    def exchange_region(self):
        """(device pointer, bytes) of this slab's exchange region."""
        p, n = ctypes.c_void_p(), ctypes.c_size_t()
        stag._check(stag.lib().stag_slab_info(self._h, None, None, None, ctypes.byref(p), ctypes.byref(n)))
        return p.value, n.value

    def ipc_handle(self) -> bytes:
        buf = ctypes.create_string_buffer(IPC_HANDLE_BYTES)
        stag._check(stag.lib().stag_slab_ipc_handle(self._h, buf))
        return buf.raw

    def connect_pointers(self, bwd_ptr: int, fwd_ptr: int):
        stag._check(stag.lib().stag_slab_connect(self._h, ctypes.c_void_p(bwd_ptr), ctypes.c_void_p(fwd_ptr)))

    def connect_all_pointers(self, ptrs):
        """ptrs[r]: device-accessible address of rank r's exchange region (own included)."""
        arr = (ctypes.c_void_p * self.nranks)(*[ctypes.c_void_p(p) for p in ptrs])
        stag._check(stag.lib().stag_slab_connect_all(self._h, arr))

    def connect_distributed(self, group=None):
        """One process per GPU: exchange IPC handles over torch.distributed and map every other
        rank's exchange region into this process (the hop needs the two neighbours, the CG's
        global sums every rank)."""
        if self.nranks == 1:
            return
        allh = all_handles(self.ipc_handle(), self.nranks, group)
        ptrs = []
        for r, h in enumerate(allh):
            if r == self.rank:
                ptrs.append(self.exchange_region()[0])
                continue
            p = ctypes.c_void_p()
            stag._check(stag.lib().stag_slab_ipc_open(ctypes.c_char_p(h), ctypes.byref(p)))
            ptrs.append(p.value)
            self._opened.append(p.value)
        self.connect_all_pointers(ptrs)

    # -- CG over the slabs: control flow only, every decision is taken in the library --------
    def cg_begin(self, x, b, mass, tol, maxiter, mode, eps_in=None, recon12=False, chunk=None, recon12_f64=False,
                 persistent=None, persist_chunk=None):
        stag.use_current_stream()
        p = stag._params(eps_in, recon12, chunk, recon12_f64, False, persistent, persist_chunk)
        stag._check(stag.lib().stag_slab_cg_begin(self._h, ctypes.c_void_p(x.data_ptr()), ctypes.c_void_p(b.data_ptr()),
                                                  float(mass), float(tol), int(maxiter), int(mode), ctypes.byref(p)))

    def cg_control(self) -> int:
        stag.use_current_stream()
        a = ctypes.c_int()
        stag._check(stag.lib().stag_slab_cg_control(self._h, ctypes.byref(a)))
        return a.value

    def cg_step(self, action: int, phase: int) -> bool:
        more = ctypes.c_int()
        stag._check(stag.lib().stag_slab_cg_step(self._h, int(action), int(phase), ctypes.byref(more)))
        return bool(more.value)

    def cg_finish(self):
        st = stag._Stats()
        rc = stag.lib().stag_slab_cg_finish(self._h, ctypes.byref(st))
        stag._check(rc, allow=(stag.OK, stag.ENOCONV, stag.EBREAKDOWN))
        return stag._stats_dict(st, rc)

    def cg_solve(self, b, mass, tol, maxiter, mode=stag.CG_RELIABLE, x0=None, after_phase=None, **kw):
        """This rank's part of the solve in a real multi-GPU run (one process per GPU, all ranks
        call it together).  b, x0: fp64 device spinors of the local dims.  Returns (x, stats).
        after_phase: called after every enqueued phase; ranks that SHARE a device pass a
        "synchronise + barrier" here so that no kernel ever waits for a kernel of another
        process that has not run yet (tests; never needed with one GPU per rank)."""
        torch = stag._require_cuda()
        x = torch.zeros_like(b) if x0 is None else x0.clone()
        if after_phase is None:                 # the whole loop in the library: stag_slab_cg_run
            stag.use_current_stream()
            st = stag._Stats()
            p = stag._params(kw.get("eps_in"), kw.get("recon12", False), kw.get("chunk"), kw.get("recon12_f64", False),
                             False, kw.get("persistent"), kw.get("persist_chunk"))
            rc = stag.lib().stag_slab_cg_run(self._h, ctypes.c_void_p(x.data_ptr()), ctypes.c_void_p(b.data_ptr()),
                                             float(mass), float(tol), int(maxiter), int(mode), ctypes.byref(p),
                                             ctypes.byref(st))
            stag._check(rc, allow=(stag.OK, stag.ENOCONV, stag.EBREAKDOWN))
            return x, stag._stats_dict(st, rc)
        self.cg_begin(x, b, mass, tol, maxiter, mode, **kw)
        while True:
            act = self.cg_control()
            if act == ACT_DONE:
                break
            ph = 0
            while True:
                more = self.cg_step(act, ph)
                if after_phase is not None:
                    after_phase()
                if not more:
                    break
                ph += 1
        return x, self.cg_finish()

    def set_wait_limit(self, polls: int):
        """Watchdog of the acquire-waits (stag_slab_set_wait_limit); 0 = the default (~10 s)."""
        stag.use_current_stream()
        stag._check(stag.lib().stag_slab_set_wait_limit(self._h, int(polls)))

    def reset(self):
        """Revive a slab whose watchdog fired (stag_slab_reset): collective, see include/stag.h."""
        stag.use_current_stream()
        stag._check(stag.lib().stag_slab_reset(self._h))

    def wait_stats(self):
        """(waits that had to spin, polls they spent) since creation / reset (stag_slab_wait_stats)."""
        stag.use_current_stream()
        a, b = ctypes.c_ulonglong(), ctypes.c_ulonglong()
        stag._check(stag.lib().stag_slab_wait_stats(self._h, ctypes.byref(a), ctypes.byref(b)))
        return a.value, b.value

    def status(self) -> int:
        """stag.OK, or stag.ETIMEOUT once a kernel of this slab gave up waiting for a peer."""
        stag.use_current_stream()
        return int(stag.lib().stag_slab_status(self._h))

    # -- the operator; spinors are device spinors of the LOCAL dims -------------------------
    def push(self, v, prec):
        stag.use_current_stream()
        stag._check(stag.lib().stag_slab_push(ctypes.c_void_p(v.data_ptr()), self._h, int(prec)))

    def hop(self, v, parity: int, prec, out=None, a: float = 0.0, own=None):
        stag.use_current_stream()
        if out is None:
            out = stag.empty_spinor(self.dims, prec)
        stag._check(stag.lib().stag_slab_hop(ctypes.c_void_p(out.data_ptr()), ctypes.c_void_p(v.data_ptr()),
                                             self._h, int(parity), int(prec), float(a),
                                             ctypes.c_void_p(own.data_ptr()) if own is not None else None))
        return out

    def dslash(self, v, parity: int, prec, out=None):
        """push + hop: what each rank of a real multi-GPU run calls (all ranks in step)."""
        self.push(v, prec)
        return self.hop(v, parity, prec, out=out)

    def apply_A(self, v_even, mass: float, prec):
        """m^2 v - D_eo D_oe v on the slab's even sites (eq. 2.3): two exchanges, two hops."""
        tmp = self.dslash(v_even, 1, prec)
        self.push(tmp, prec)
        return self.hop(tmp, 0, prec, a=mass * mass, own=v_even)

    def close(self):
        for p in self._opened:
            stag.lib().stag_slab_ipc_close(ctypes.c_void_p(p))
        self._opened = []
        if self._h:
            stag.lib().stag_links_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def connect_in_process(slabs):
    """Slabs that live in one process (one GPU holding several, or tests): hand each every
    rank's exchange region as raw device pointers."""
    n = len(slabs)
    ptrs = [s.exchange_region()[0] for s in slabs]
    for r, s in enumerate(slabs):
        if s.rank != r or s.nranks != n:
            raise ValueError("slabs must be given in rank order, all of them")
        s.connect_all_pointers(ptrs)


def cg_solve_in_process(slabs, bs, mass, tol, maxiter, mode=stag.CG_RELIABLE, fused=False, **kw):
    """The multi-GPU solve with all slabs in THIS process on one device.  bs[r]: rank r's fp64 device
    spinor.  Returns (xs, [stats]).
    fused = False: every phase is enqueued for rank 0, 1, ... before the next phase, so a kernel
    that waits for its peers always finds their kernels already finished (lockstep).
    fused = True: the iterations of ALL ranks run in one cooperative launch of the persistent kernel
    (stag_slab_cg_iter_all), each rank a group of blocks: the ranks execute concurrently and their
    acquire-waits really spin on peers that are still running, as on separate GPUs.  The rare fp64
    steps (initial residual, reliable updates, verification) stay stepped."""
    torch = stag._require_cuda()
    xs = [torch.zeros_like(b) for b in bs]
    for s, x, b in zip(slabs, xs, bs):
        s.cg_begin(x, b, mass, tol, maxiter, mode, **kw)
    while True:
        acts = [s.cg_control() for s in slabs]
        if any(a != acts[0] for a in acts):
            raise RuntimeError("ranks disagree on the next action: %r" % (acts,))
        if acts[0] == ACT_DONE:
            break
        if fused and acts[0] == ACT_ITER:
            stag.use_current_stream()
            arr = (ctypes.c_void_p * len(slabs))(*[s.handle.value for s in slabs])
            stag._check(stag.lib().stag_slab_cg_iter_all(arr, len(slabs)))
            continue
        ph = 0
        while True:
            more = [s.cg_step(acts[0], ph) for s in slabs]
            if not more[0]:
                break
            ph += 1
    return xs, [s.cg_finish() for s in slabs]
