"""paper_1111_0125_b200 -- Python binding of libstag (include/stag.h).

Argument marshalling only: every step of the hot path (Dslash, A, the CG vector
algebra, the mixed-precision drivers) runs in the CUDA kernels behind the C ABI.
PyTorch supplies device memory and streams; nothing here computes.

The names mirror the C entry points:

    links = Links(dims, W)                      # stag_links_create  (step S0)
    v     = spinor_pack(chi, dims, prec)        # stag_spinor_pack
    out   = dslash(v, links, parity, prec)      # stag_dslash        (eq. 2.5)
    out   = apply_A(v, links, mass, prec)       # stag_apply_A       (eq. 2.3)
    x, st = cg_solve(b, links, mass, tol, maxiter, mode)   # stag_cg_solve_ex

Several right-hand sides sharing each pass over the links (a batch is a 2-D tensor
[nrhs][6*Vh_pad], one device spinor per row):

    outs    = dslash_mrhs(vs, links, parity, prec)          # stag_dslash_mrhs
    outs    = apply_A_mrhs(vs, links, mass, prec)           # stag_apply_A_mrhs
    xs, sts = cg_solve_mrhs(bs, links, mass, tol, maxiter)  # stag_cg_solve_mrhs
    pe, po, sts = solve_M(he, ho, links, mass, tol, maxiter)   # stag_solve_M: (D+m) psi = h

There is no CPU fallback: importing works anywhere the shared library loads, but
every compute entry raises unless a CUDA device is present.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_LIB = os.path.join(_HERE, "libstag.so")
_HEADER = os.path.join(os.path.dirname(_HERE), "include", "stag.h")

PREC_F64, PREC_F32, PREC_F64_R12, PREC_F32_R12, PREC_F64_R8, PREC_F32_R8 = 0, 1, 2, 3, 4, 5
CG_F64, CG_F32, CG_DEFECT, CG_RELIABLE = 0, 1, 2, 3
OK, EINVAL, ECUDA, ENOMEM, ETIMEOUT, ENOCONV, EBREAKDOWN = 0, -1, -2, -3, -4, 1, 2

MAX_RHS = 12
BATCH_BLOCKED, BATCH_PAIRED = 0, 1

PREC_NAMES = {PREC_F64: "fp64/18", PREC_F32: "fp32/18", PREC_F64_R12: "fp64/12", PREC_F32_R12: "fp32/12",
              PREC_F64_R8: "fp64/8", PREC_F32_R8: "fp32/8"}


class StagError(RuntimeError):
    def __init__(self, status, text):
        super().__init__("libstag status %d: %s" % (status, text))
        self.status = status


def _sources():
    out = [_HEADER]
    for f in sorted(os.listdir(_CSRC)):
        if f.endswith((".cu", ".cuh", ".h")):
            out.append(os.path.join(_CSRC, f))
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/*.cu into libstag.so (in-tree) for sm_100a with nvcc."""
    newest = max(os.path.getmtime(p) for p in _sources())
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        tmp = _LIB + ".tmp.%d" % os.getpid()
        cus = [p for p in _sources() if p.endswith(".cu")]
        cmd = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3",
               "-std=c++17", "-Xcompiler", "-fPIC", "-shared", "-o", tmp] + cus
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        subprocess.check_call(cmd)
        os.replace(tmp, _LIB)
    return _LIB


class _Params(ctypes.Structure):
    _fields_ = [("eps_in", ctypes.c_double), ("recon12", ctypes.c_int),
                ("graph_chunk", ctypes.c_int), ("recon12_f64", ctypes.c_int), ("recon8", ctypes.c_int),
                ("persistent", ctypes.c_int), ("persist_chunk", ctypes.c_int)]


class _Stats(ctypes.Structure):
    _fields_ = [("iters", ctypes.c_int), ("n_updates", ctypes.c_int), ("n_restarts", ctypes.c_int),
                ("iters_f32", ctypes.c_int), ("applies_f64", ctypes.c_int),
                ("true_resid", ctypes.c_double), ("iter_resid", ctypes.c_double),
                ("seconds", ctypes.c_double)]


_lib = None

# name -> (restype, argtypes); the ABI test checks this table against include/stag.h
_vp, _ip, _dp = ctypes.c_void_p, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_double)
SIGNATURES = {
    "stag_set_stream": (ctypes.c_int, [_vp]),
    "stag_strerror": (ctypes.c_char_p, [ctypes.c_int]),
    "stag_cg_workspace_bytes": (ctypes.c_size_t, [_ip, ctypes.c_int, ctypes.c_int]),
    "stag_set_workspace": (ctypes.c_int, [_vp, ctypes.c_size_t]),
    "stag_launch_count": (ctypes.c_ulonglong, []),
    "stag_reset_launch_count": (None, []),
    "stag_links_create": (ctypes.c_int, [ctypes.POINTER(_vp), _ip, ctypes.c_int, _vp, ctypes.c_int]),
    "stag_links_create_unfolded": (ctypes.c_int, [ctypes.POINTER(_vp), _ip, ctypes.c_int, _vp, ctypes.c_int]),
    "stag_links_destroy": (None, [_vp]),
    "stag_links_recon_error": (ctypes.c_int, [_vp, _dp]),
    "stag_links_recon8_error": (ctypes.c_int, [_vp, ctypes.c_int, _dp]),
    "stag_spinor_bytes": (ctypes.c_size_t, [_ip, ctypes.c_int]),
    "stag_spinor_pack": (ctypes.c_int, [_vp, _vp, _ip, ctypes.c_int]),
    "stag_spinor_unpack": (ctypes.c_int, [_vp, _vp, _ip, ctypes.c_int]),
    "stag_dslash": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_int, _ip, ctypes.c_int]),
    "stag_apply_A": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_double, ctypes.c_int]),
    "stag_apply_A_noalloc": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_double, ctypes.c_int]),
    "stag_cg_solve": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_double, ctypes.c_double, ctypes.c_int,
                                     ctypes.c_int, _ip, _dp]),
    "stag_cg_solve_ex": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_double, ctypes.c_double, ctypes.c_int,
                                        ctypes.c_int, ctypes.POINTER(_Params), ctypes.POINTER(_Stats)]),
    "stag_dslash_mrhs": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_int, _ip, ctypes.c_int, ctypes.c_int]),
    "stag_apply_A_mrhs": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_double, ctypes.c_int, ctypes.c_int]),
    "stag_batch_convert": (ctypes.c_int, [_vp, _vp, _ip, ctypes.c_int, ctypes.c_int, ctypes.c_int]),
    "stag_dslash_batch": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_int, _ip, ctypes.c_int, ctypes.c_int, ctypes.c_int]),
    "stag_apply_A_batch": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_double, ctypes.c_int, ctypes.c_int, ctypes.c_int]),
    "stag_cg_solve_mrhs": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_double, ctypes.c_double, ctypes.c_int,
                                          ctypes.c_int, ctypes.c_int, ctypes.POINTER(_Params),
                                          ctypes.POINTER(_Stats)]),
    "stag_solve_M": (ctypes.c_int, [_vp, _vp, _vp, _vp, _vp, ctypes.c_double, ctypes.c_double,
                                    ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.POINTER(_Params),
                                    ctypes.POINTER(_Stats)]),
    "stag_slab_create": (ctypes.c_int, [ctypes.POINTER(_vp), _ip, ctypes.c_int, _vp, ctypes.c_int,
                                        ctypes.c_int, ctypes.c_int]),
    "stag_slab_create_local": (ctypes.c_int, [ctypes.POINTER(_vp), _ip, ctypes.c_int, _vp, _vp, ctypes.c_int,
                                              ctypes.c_int, ctypes.c_int]),
    "stag_slab_info": (ctypes.c_int, [_vp, _ip, _ip, _ip, ctypes.POINTER(_vp), ctypes.POINTER(ctypes.c_size_t)]),
    "stag_slab_ipc_handle": (ctypes.c_int, [_vp, ctypes.c_char_p]),
    "stag_slab_ipc_open": (ctypes.c_int, [ctypes.c_char_p, ctypes.POINTER(_vp)]),
    "stag_slab_ipc_close": (ctypes.c_int, [_vp]),
    "stag_slab_connect": (ctypes.c_int, [_vp, _vp, _vp]),
    "stag_slab_push": (ctypes.c_int, [_vp, _vp, ctypes.c_int]),
    "stag_slab_hop": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_int, ctypes.c_int, ctypes.c_double, _vp]),
    "stag_slab_dslash": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_int, ctypes.c_int]),
    "stag_slab_set_wait_limit": (ctypes.c_int, [_vp, ctypes.c_ulonglong]),
    "stag_slab_status": (ctypes.c_int, [_vp]),
    "stag_slab_reset": (ctypes.c_int, [_vp]),
    "stag_slab_wait_stats": (ctypes.c_int, [_vp, ctypes.POINTER(ctypes.c_ulonglong), ctypes.POINTER(ctypes.c_ulonglong)]),
    "stag_slab_connect_all": (ctypes.c_int, [_vp, ctypes.POINTER(_vp)]),
    "stag_slab_cg_begin": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_double, ctypes.c_double, ctypes.c_int,
                                          ctypes.c_int, ctypes.POINTER(_Params)]),
    "stag_slab_cg_control": (ctypes.c_int, [_vp, _ip]),
    "stag_slab_cg_step": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int, _ip]),
    "stag_slab_cg_finish": (ctypes.c_int, [_vp, ctypes.POINTER(_Stats)]),
    "stag_slab_cg_iter_all": (ctypes.c_int, [ctypes.POINTER(_vp), ctypes.c_int]),
    "stag_slab_cg_run": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_double, ctypes.c_double, ctypes.c_int,
                                        ctypes.c_int, ctypes.POINTER(_Params), ctypes.POINTER(_Stats)]),
    "stag_cg_solve_host": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_double, ctypes.c_double,
                                          ctypes.c_int, ctypes.c_int, ctypes.POINTER(_Params),
                                          ctypes.POINTER(_Stats)]),
}


def lib():
    """The loaded shared library (built on first use if missing or stale)."""
    global _lib
    if _lib is None:
        path = build()
        h = ctypes.CDLL(path)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(h, name)          # AttributeError = the .so does not export the symbol
            fn.restype = res
            fn.argtypes = args
        _lib = h
    return _lib


def loaded_library_path() -> str:
    lib()
    return _LIB


def _check(status: int, allow=(OK,)):
    if status not in allow:
        raise StagError(status, lib().stag_strerror(status).decode())
    return status


def _require_cuda():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("libstag needs a CUDA device (sm_100a); there is no CPU fallback")
    return torch


def _cdims(dims):
    d = [int(v) for v in dims]
    if len(d) != 4:
        raise ValueError("dims must have four extents")
    return (ctypes.c_int * 4)(*d)


def use_current_stream():
    """Point the library at torch's current CUDA stream."""
    torch = _require_cuda()
    _check(lib().stag_set_stream(ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)))


def cg_workspace_bytes(dims, mode: int, nrhs: int = 1) -> int:
    """stag_cg_workspace_bytes: pure arithmetic, works without a device."""
    return int(lib().stag_cg_workspace_bytes(_cdims(dims), int(mode), int(nrhs)))


def set_workspace(ws=None):
    """stag_set_workspace for the calling host thread.  ws: a CUDA uint8 tensor the caller keeps
    alive (e.g. torch.empty(cg_workspace_bytes(...), dtype=torch.uint8, device="cuda")), or None
    to return to the handle-owned default."""
    if ws is None:
        _check(lib().stag_set_workspace(None, 0))
        return
    _require_cuda()
    if not ws.is_cuda or not ws.is_contiguous():
        raise ValueError("the workspace must be a contiguous CUDA tensor")
    _check(lib().stag_set_workspace(ctypes.c_void_p(ws.data_ptr()), ws.numel() * ws.element_size()))


def launch_count() -> int:
    return int(lib().stag_launch_count())


def reset_launch_count():
    lib().stag_reset_launch_count()


def spinor_bytes(dims, prec) -> int:
    return int(lib().stag_spinor_bytes(_cdims(dims), int(prec)))


def _is_f32(prec):
    return prec in (PREC_F32, PREC_F32_R12, PREC_F32_R8)


def empty_spinor(dims, prec):
    """Uninitialised device spinor (torch tensor of reals, 6*Vh_pad long)."""
    torch = _require_cuda()
    nbytes = spinor_bytes(dims, prec)
    if nbytes == 0:
        raise ValueError("bad dims %r" % (dims,))
    dt = torch.float32 if _is_f32(prec) else torch.float64
    return torch.empty(nbytes // (4 if _is_f32(prec) else 8), dtype=dt, device="cuda")


class Links:
    """Owner of a stag_links_t handle.  W: canonical complex128 [4][2][Vh][3][3] (numpy, host)
    or a CUDA float64 tensor holding the same 4*2*Vh*18 doubles."""

    def __init__(self, dims, W, antiperiodic_t: bool = True, folded: bool = True):
        """folded=False: W is the bare U; eta and the time boundary sign are folded in on the
        device (stag_links_create_unfolded)."""
        torch = _require_cuda()
        use_current_stream()
        self.dims = tuple(int(v) for v in dims)
        self._h = ctypes.c_void_p()
        vh = 1
        for v in self.dims:
            vh *= v
        vh //= 2
        if hasattr(W, "is_cuda"):
            if not W.is_cuda or W.dtype != torch.float64 or W.numel() != 4 * 2 * vh * 18:
                raise ValueError("device W must be a CUDA float64 tensor of 4*2*Vh*18 elements")
            W = W.contiguous()
            ptr, on_dev = ctypes.c_void_p(W.data_ptr()), 1
        else:
            import numpy as np
            W = np.ascontiguousarray(W, dtype=np.complex128)
            if W.shape != (4, 2, vh, 3, 3):
                raise ValueError("host W must have shape (4,2,Vh,3,3)")
            ptr, on_dev = ctypes.c_void_p(W.ctypes.data), 0
        self._keep = W
        create = lib().stag_links_create if folded else lib().stag_links_create_unfolded
        _check(create(ctypes.byref(self._h), _cdims(self.dims), int(bool(antiperiodic_t)), ptr, on_dev))
        torch.cuda.current_stream().synchronize()
        self._keep = None

    @property
    def handle(self):
        return self._h

    def recon8_error(self, prec) -> float:
        """Largest rebuilt-entry error of the 8-parameter form (builds it); raises if refused."""
        e = ctypes.c_double()
        _check(lib().stag_links_recon8_error(self._h, int(prec), ctypes.byref(e)))
        return e.value

    def recon_error(self) -> float:
        e = ctypes.c_double()
        _check(lib().stag_links_recon_error(self._h, ctypes.byref(e)))
        return e.value

    def close(self):
        if self._h:
            lib().stag_links_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def spinor_pack(chi, dims, prec):
    """canonical complex128 [Vh][3] (numpy) or CUDA float64 tensor of Vh*6 -> device spinor."""
    torch = _require_cuda()
    use_current_stream()
    if not hasattr(chi, "is_cuda"):
        import numpy as np
        chi = torch.from_numpy(np.ascontiguousarray(chi, dtype=np.complex128).view(np.float64).reshape(-1)).cuda()
    out = empty_spinor(dims, prec)
    _check(lib().stag_spinor_pack(ctypes.c_void_p(out.data_ptr()), ctypes.c_void_p(chi.data_ptr()),
                                  _cdims(dims), int(prec)))
    return out


def spinor_unpack(v, dims, prec, to_numpy: bool = True):
    """device spinor -> canonical fp64 (numpy complex128 [Vh][3] or CUDA float64 tensor)."""
    torch = _require_cuda()
    use_current_stream()
    vh = 1
    for d in dims:
        vh *= int(d)
    vh //= 2
    out = torch.empty(vh * 6, dtype=torch.float64, device="cuda")
    _check(lib().stag_spinor_unpack(ctypes.c_void_p(out.data_ptr()), ctypes.c_void_p(v.data_ptr()),
                                    _cdims(dims), int(prec)))
    if not to_numpy:
        return out
    import numpy as np
    return out.cpu().numpy().view(np.complex128).reshape(vh, 3)


def dslash(v, links: Links, parity: int, prec, out=None):
    """out (sites of `parity`) = D v (other parity): one hop of eq. 2.5."""
    use_current_stream()
    if out is None:
        out = empty_spinor(links.dims, prec)
    _check(lib().stag_dslash(ctypes.c_void_p(out.data_ptr()), ctypes.c_void_p(v.data_ptr()),
                             links.handle, int(parity), _cdims(links.dims), int(prec)))
    return out


def apply_A(v_even, links: Links, mass: float, prec, out=None):
    """out_even = mass^2 v_even - D_eo D_oe v_even (eq. 2.3 on even sites)."""
    use_current_stream()
    if out is None:
        out = empty_spinor(links.dims, prec)
    _check(lib().stag_apply_A(ctypes.c_void_p(out.data_ptr()), ctypes.c_void_p(v_even.data_ptr()),
                              links.handle, float(mass), int(prec)))
    return out


NOALLOC_SCRATCH_BYTES = 8 << 20


def apply_A_noalloc(v_even, out, links: Links, mass: float, prec):
    """stag_apply_A_noalloc: out = mass^2 v_even - D_eo D_oe v_even written into the spinor `out`
    YOU pass (this wrapper creates no tensor), with the odd-site intermediate in the library's
    built-in 8 MiB device array instead of a workspace.  For callers that may not allocate device
    memory (all of it belongs to their own pool, or cudaMalloc is banned where they run).
    Raises StagError(EINVAL) when the lattice is too large for the array or the links of `prec`
    have not been built by an earlier ordinary call.  Calls on different streams must not overlap:
    they share the one array."""
    use_current_stream()
    _check(lib().stag_apply_A_noalloc(ctypes.c_void_p(out.data_ptr()), ctypes.c_void_p(v_even.data_ptr()),
                                      links.handle, float(mass), int(prec)))
    return out


def _params(eps_in, recon12, graph_chunk, recon12_f64, recon8=False, persistent=None, persist_chunk=None):
    p = _Params()
    p.recon8 = int(bool(recon8))
    p.persistent = 0 if persistent is None else (1 if persistent else -1)
    p.persist_chunk = int(persist_chunk or 0)
    p.eps_in = float(eps_in or 0.0)
    p.recon12 = int(bool(recon12))
    p.graph_chunk = int(graph_chunk or 0)
    p.recon12_f64 = int(bool(recon12_f64))
    return p


def _stats_dict(st: _Stats, status: int):
    d = {name: getattr(st, name) for name, _ in _Stats._fields_}
    d["status"] = status
    return d


def cg_solve(b, links: Links, mass: float, tol: float, maxiter: int, mode: int = CG_RELIABLE,
             x0=None, eps_in=None, recon12=False, graph_chunk=None, recon12_f64=False, recon8=False,
             persistent=None, persist_chunk=None):
    """Solve A x = b on the even sites.  b, x0: fp64 device spinors.  Returns (x, stats dict);
    stats["status"] is 0, ENOCONV or EBREAKDOWN.  Errors (< 0) raise StagError.
    persistent: True / False forces the persistent-kernel iteration on / off, None = by volume."""
    torch = _require_cuda()
    use_current_stream()
    x = torch.zeros_like(b) if x0 is None else x0.clone()
    st = _Stats()
    p = _params(eps_in, recon12, graph_chunk, recon12_f64, recon8, persistent, persist_chunk)
    rc = lib().stag_cg_solve_ex(ctypes.c_void_p(x.data_ptr()), ctypes.c_void_p(b.data_ptr()),
                                links.handle, float(mass), float(tol), int(maxiter), int(mode),
                                ctypes.byref(p), ctypes.byref(st))
    _check(rc, allow=(OK, ENOCONV, EBREAKDOWN))
    return x, _stats_dict(st, rc)


def cg_solve_basic(b, links: Links, mass: float, tol: float, maxiter: int, mode: int):
    """The plain north-star entry stag_cg_solve: returns (x, iters, true_resid, status)."""
    torch = _require_cuda()
    use_current_stream()
    x = torch.zeros_like(b)
    it, rr = ctypes.c_int(0), ctypes.c_double(0.0)
    rc = lib().stag_cg_solve(ctypes.c_void_p(x.data_ptr()), ctypes.c_void_p(b.data_ptr()),
                             links.handle, float(mass), float(tol), int(maxiter), int(mode),
                             ctypes.byref(it), ctypes.byref(rr))
    _check(rc, allow=(OK, ENOCONV, EBREAKDOWN))
    return x, it.value, rr.value, rc


def cg_solve_host(b_host, links: Links, mass: float, tol: float, maxiter: int,
                  mode: int = CG_RELIABLE, x_host=None, eps_in=None, recon12=False,
                  graph_chunk=None, recon12_f64=False):
    """End-to-end solve from/to HOST canonical fp64 arrays (torch CPU float64 tensors of Vh*6,
    ideally pinned).  x_host is the initial guess on entry (zeros if None) and is overwritten."""
    torch = _require_cuda()
    use_current_stream()
    if x_host is None:
        x_host = torch.zeros_like(b_host)
    st = _Stats()
    p = _params(eps_in, recon12, graph_chunk, recon12_f64)
    rc = lib().stag_cg_solve_host(ctypes.c_void_p(x_host.data_ptr()), ctypes.c_void_p(b_host.data_ptr()),
                                  links.handle, float(mass), float(tol), int(maxiter), int(mode),
                                  ctypes.byref(p), ctypes.byref(st))
    _check(rc, allow=(OK, ENOCONV, EBREAKDOWN))
    return x_host, _stats_dict(st, rc)


# ---- several right-hand sides (include/stag.h "several right-hand sides") -------------------

def spinor_pack_mrhs(chis, dims, prec):
    """list of canonical spinors -> batch tensor [nrhs][6*Vh_pad] (one device spinor per row)."""
    torch = _require_cuda()
    return torch.stack([spinor_pack(c, dims, prec) for c in chis]).contiguous()


def spinor_unpack_mrhs(vs, dims, prec):
    return [spinor_unpack(vs[k], dims, prec) for k in range(vs.shape[0])]


def _batch(vs):
    if vs.dim() != 2 or not vs.is_contiguous():
        raise ValueError("a batch is a contiguous 2-D tensor [nrhs][6*Vh_pad]")
    return int(vs.shape[0])


def batch_convert(vs, dims, prec, to_layout: int, out=None):
    """stag_batch_convert: the batch in the other layout (BATCH_BLOCKED <-> BATCH_PAIRED)."""
    torch = _require_cuda()
    use_current_stream()
    n = _batch(vs)
    if out is None:
        out = torch.empty_like(vs)
    _check(lib().stag_batch_convert(ctypes.c_void_p(out.data_ptr()), ctypes.c_void_p(vs.data_ptr()),
                                    _cdims(dims), int(prec), n, int(to_layout)))
    return out


def dslash_mrhs(vs, links: Links, parity: int, prec, out=None, layout: int = BATCH_BLOCKED):
    """One hop of eq. 2.5 applied to every spinor of the batch, links read once per chunk
    (stag_dslash_batch; layout BATCH_BLOCKED is stag_dslash_mrhs)."""
    torch = _require_cuda()
    use_current_stream()
    n = _batch(vs)
    if out is None:
        out = torch.empty_like(vs)
    _check(lib().stag_dslash_batch(ctypes.c_void_p(out.data_ptr()), ctypes.c_void_p(vs.data_ptr()),
                                   links.handle, int(parity), _cdims(links.dims), int(prec), n, int(layout)))
    return out


def apply_A_mrhs(vs_even, links: Links, mass: float, prec, out=None, layout: int = BATCH_BLOCKED):
    torch = _require_cuda()
    use_current_stream()
    n = _batch(vs_even)
    if out is None:
        out = torch.empty_like(vs_even)
    _check(lib().stag_apply_A_batch(ctypes.c_void_p(out.data_ptr()), ctypes.c_void_p(vs_even.data_ptr()),
                                    links.handle, float(mass), int(prec), n, int(layout)))
    return out


def cg_solve_mrhs(bs, links: Links, mass: float, tol: float, maxiter: int, mode: int = CG_RELIABLE,
                  x0=None, eps_in=None, recon12=False, graph_chunk=None, recon12_f64=False):
    """nrhs systems A x_k = b_k in lockstep.  bs, x0: fp64 batches.  Returns (xs, [stats])."""
    torch = _require_cuda()
    use_current_stream()
    n = _batch(bs)
    xs = torch.zeros_like(bs) if x0 is None else x0.clone()
    sts = (_Stats * n)()
    p = _params(eps_in, recon12, graph_chunk, recon12_f64)
    rc = lib().stag_cg_solve_mrhs(ctypes.c_void_p(xs.data_ptr()), ctypes.c_void_p(bs.data_ptr()),
                                  links.handle, float(mass), float(tol), int(maxiter), int(mode), n,
                                  ctypes.byref(p), sts)
    _check(rc, allow=(OK, ENOCONV, EBREAKDOWN))
    return xs, [_stats_dict(sts[k], rc) for k in range(n)]


def solve_M(h_even, h_odd, links: Links, mass: float, tol: float, maxiter: int,
            mode: int = CG_RELIABLE, eps_in=None, recon12=False, graph_chunk=None, recon12_f64=False):
    """(D + m) psi = h on the whole lattice for a batch of sources (fp64 batches, one parity
    each).  Returns (psi_even, psi_odd, [stats of the even-site solve])."""
    torch = _require_cuda()
    use_current_stream()
    n = _batch(h_even)
    if _batch(h_odd) != n:
        raise ValueError("h_even and h_odd must hold the same number of sources")
    pe, po = torch.zeros_like(h_even), torch.empty_like(h_odd)
    sts = (_Stats * n)()
    p = _params(eps_in, recon12, graph_chunk, recon12_f64)
    rc = lib().stag_solve_M(ctypes.c_void_p(pe.data_ptr()), ctypes.c_void_p(po.data_ptr()),
                            ctypes.c_void_p(h_even.data_ptr()), ctypes.c_void_p(h_odd.data_ptr()),
                            links.handle, float(mass), float(tol), int(maxiter), int(mode), n,
                            ctypes.byref(p), sts)
    _check(rc, allow=(OK, ENOCONV, EBREAKDOWN))
    return pe, po, [_stats_dict(sts[k], rc) for k in range(n)]
