"""CPU ORACLE (test infrastructure, not the product) -- see stag_oracle.c.

Thin ctypes wrapper over liboracle.so: plain fp64 staggered Dslash (eq. 2.5,
PAPER.md L42), A = -D^2 + m^2 on even sites (eq. 2.3; L62) and the CG of
Fig. 1 (L45-56).  Arrays are the canonical complex128 layouts of
``fieldgen`` (W[mu][p][cb][3][3], chi[cb][3]).

Only tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline /
``--impl reference`` leg may import this package.  It imports nothing from the
CUDA package and the CUDA package imports nothing from here.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "stag_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


CFLAGS = ["-O2", "-fopenmp"]                       # the checker: portable code, it travels between machines
CFLAGS_NATIVE = ["-O3", "-march=native", "-fopenmp"]   # the timed CPU baseline, built where it runs
_flags_in_use = list(CFLAGS)


def build(force: bool = False) -> str:
    """Compile the oracle as it stands (plain -O2 + OpenMP; never tuned)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(
            ["gcc"] + CFLAGS + ["-fPIC", "-shared", "-std=c11", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


def use_native_build() -> list:
    """For the timed CPU baseline only (bench.py): rebuild the SAME source with -O3 -march=native
    on the machine it will run on (a .so built for another CPU could not be carried there) into a
    private temporary file, and use it from now on in this process.  Falls back to the portable
    build if the compiler refuses.  Returns the flags in use."""
    global _lib, _flags_in_use
    import tempfile
    out = os.path.join(tempfile.mkdtemp(prefix="oracle_native_"), "liboracle_native.so")
    try:
        subprocess.check_call(["gcc"] + CFLAGS_NATIVE + ["-fPIC", "-shared", "-std=c11", "-o", out, _SRC, "-lm"],
                              stderr=subprocess.DEVNULL)
    except (OSError, subprocess.CalledProcessError):
        return list(_flags_in_use)
    _lib = None
    _load(out)
    _flags_in_use = list(CFLAGS_NATIVE)
    return list(_flags_in_use)


def compile_flags() -> list:
    return list(_flags_in_use)


def max_threads() -> int:
    """omp_get_max_threads() of the loaded oracle."""
    return int(_load().so_max_threads())


def _load(path=None):
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(path or build())
        lib.so_max_threads.argtypes = []
        lib.so_max_threads.restype = ctypes.c_int
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        u64p = ctypes.POINTER(ctypes.c_uint64)
        lib.so_dslash.argtypes = [dp, dp, dp, ip, ctypes.c_int]
        lib.so_dslash.restype = ctypes.c_int
        lib.so_dslash_counted.argtypes = [dp, dp, dp, ip, ctypes.c_int, u64p, u64p]
        lib.so_dslash_counted.restype = ctypes.c_int
        lib.so_apply_A.argtypes = [dp, dp, dp, ip, ctypes.c_double, dp]
        lib.so_apply_A.restype = ctypes.c_int
        lib.so_cg.argtypes = [dp, dp, dp, ip, ctypes.c_double, ctypes.c_double, ctypes.c_int,
                              ip, dp, ip]
        lib.so_cg.restype = ctypes.c_int
        lib.so_apply_M.argtypes = [dp, dp, dp, ip, ctypes.c_double]
        lib.so_apply_M.restype = ctypes.c_int
        lib.so_solve_M.argtypes = [dp, dp, dp, ip, ctypes.c_double, ctypes.c_double, ctypes.c_int,
                                   ip, dp]
        lib.so_solve_M.restype = ctypes.c_int
        lib.so_redot.argtypes = [dp, dp, ctypes.c_long]
        lib.so_redot.restype = ctypes.c_double
        _lib = lib
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _cdims(dims):
    return (ctypes.c_int * 4)(*[int(v) for v in dims])


def _vh(dims):
    v = 1
    for d in dims:
        v *= int(d)
    return v // 2


def _check(W, dims, *vecs):
    vh = _vh(dims)
    if W.dtype != np.complex128 or W.shape != (4, 2, vh, 3, 3) or not W.flags.c_contiguous:
        raise ValueError("W must be C-contiguous complex128 [4][2][Vh][3][3]")
    for v in vecs:
        if v.dtype != np.complex128 or v.shape != (vh, 3) or not v.flags.c_contiguous:
            raise ValueError("spinor must be C-contiguous complex128 [Vh][3]")


def dslash(chi, W, dims, parity_out: int):
    """One parity hop of eq. 2.5: returns D chi on the ``parity_out`` sites."""
    _check(W, dims, chi)
    out = np.empty_like(chi)
    if _load().so_dslash(_dp(out), _dp(chi), _dp(W), _cdims(dims), int(parity_out)):
        raise ValueError("so_dslash: bad argument")
    return out


def dslash_counted(chi, W, dims, parity_out: int):
    """Same hop with the flop and byte tallies of P:L62: (out, flops, bytes)."""
    _check(W, dims, chi)
    out = np.empty_like(chi)
    fl, by = ctypes.c_uint64(0), ctypes.c_uint64(0)
    if _load().so_dslash_counted(_dp(out), _dp(chi), _dp(W), _cdims(dims), int(parity_out),
                                 ctypes.byref(fl), ctypes.byref(by)):
        raise ValueError("so_dslash_counted: bad argument")
    return out, fl.value, by.value


def apply_A(chi_e, W, dims, mass: float):
    """A chi_e = m^2 chi_e - D_eo D_oe chi_e (eq. 2.3 on even sites)."""
    _check(W, dims, chi_e)
    out = np.empty_like(chi_e)
    tmp = np.empty_like(chi_e)
    if _load().so_apply_A(_dp(out), _dp(chi_e), _dp(W), _cdims(dims), float(mass), _dp(tmp)):
        raise ValueError("so_apply_A: bad argument")
    return out


def cg(b, W, dims, mass: float, tol: float, maxiter: int, x0=None):
    """Fig. 1 CG in fp64.  Returns (x, iters, true_resid, restarts, rc)."""
    _check(W, dims, b)
    x = np.zeros_like(b) if x0 is None else np.ascontiguousarray(x0, dtype=np.complex128).copy()
    it, rs = ctypes.c_int(0), ctypes.c_int(0)
    rho = ctypes.c_double(0.0)
    rc = _load().so_cg(_dp(x), _dp(b), _dp(W), _cdims(dims), float(mass), float(tol),
                       int(maxiter), ctypes.byref(it), ctypes.byref(rho), ctypes.byref(rs))
    if rc < 0:
        raise ValueError("so_cg: bad argument")
    return x, it.value, rho.value, rs.value, rc


def redot(a, b) -> float:
    """Re <a, b> with the oracle's fixed-block summation."""
    a = np.ascontiguousarray(a, dtype=np.complex128)
    b = np.ascontiguousarray(b, dtype=np.complex128)
    return _load().so_redot(_dp(a), _dp(b), a.size * 2)


def _check_full(W, dims, *vecs):
    vh = _vh(dims)
    _check(W, dims)
    for v in vecs:
        if v.dtype != np.complex128 or v.shape != (2, vh, 3) or not v.flags.c_contiguous:
            raise ValueError("full-lattice spinor must be C-contiguous complex128 [2][Vh][3]")


def apply_M(psi, W, dims, mass: float):
    """(D + m) psi on the whole lattice; psi[parity][cb][3] (Q23)."""
    _check_full(W, dims, psi)
    out = np.empty_like(psi)
    if _load().so_apply_M(_dp(out), _dp(psi), _dp(W), _cdims(dims), float(mass)):
        raise ValueError("so_apply_M: bad argument")
    return out


def solve_M(h, W, dims, mass: float, tol: float, maxiter: int):
    """(D + m) psi = h through the even-site solve of A.  Returns (psi, iters, resid, rc)."""
    _check_full(W, dims, h)
    psi = np.zeros_like(h)
    it = ctypes.c_int(0)
    rho = ctypes.c_double(0.0)
    rc = _load().so_solve_M(_dp(psi), _dp(h), _dp(W), _cdims(dims), float(mass), float(tol),
                            int(maxiter), ctypes.byref(it), ctypes.byref(rho))
    if rc < 0:
        raise ValueError("so_solve_M: bad argument")
    return psi, it.value, rho.value, rc
