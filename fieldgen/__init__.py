"""Seeded synthetic lattice inputs (see fieldgen.c for the recipe and layouts).

Input generation only: no Dslash, no A, no CG lives here.  Both the oracle's
tests and the CUDA path's tests / bench draw their inputs from this module.

Per-config recipes follow BASELINE.json ``configs``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fieldgen.c")
_LIB = os.path.join(_HERE, "libfieldgen.so")

_lib = None


def build(force: bool = False) -> str:
    """Compile fieldgen.c into libfieldgen.so (in-tree) with gcc."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        lib.fg_links.argtypes = [dp, ip, ctypes.c_int, ctypes.c_uint64, ctypes.c_double,
                                 ctypes.c_int, ctypes.c_int]
        lib.fg_links.restype = ctypes.c_int
        lib.fg_links_slices.argtypes = [dp, ip, ctypes.c_int, ctypes.c_uint64, ctypes.c_double,
                                        ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int]
        lib.fg_links_slices.restype = ctypes.c_int
        lib.fg_spinor_gaussian.argtypes = [dp, ip, ctypes.c_int, ctypes.c_uint64]
        lib.fg_spinor_gaussian.restype = ctypes.c_int
        lib.fg_spinor_planewave.argtypes = [dp, ip, ctypes.c_int, ip, dp, ctypes.c_int]
        lib.fg_spinor_planewave.restype = ctypes.c_int
        lib.fg_gauge.argtypes = [dp, ip, ctypes.c_uint64]
        lib.fg_gauge.restype = ctypes.c_int
        lib.fg_normal_at.argtypes = [ctypes.c_uint64] * 4
        lib.fg_normal_at.restype = ctypes.c_double
        _lib = lib
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _dims(dims):
    d = [int(v) for v in dims]
    if len(d) != 4 or any(v < 2 or v % 2 for v in d):
        raise ValueError("dims must be four even extents >= 2, got %r" % (dims,))
    return (ctypes.c_int * 4)(*d), d


def volume(dims) -> int:
    v = 1
    for d in dims:
        v *= int(d)
    return v


KIND = {"unit": 0, "random": 1, "smooth": 2}


def links(dims, kind: str = "random", seed: int = 0, eps: float = 0.0,
          fold: bool = True, antiperiodic_t: bool = True) -> np.ndarray:
    """W[mu][p][cb][3][3] complex128 (eta*bc folded in when ``fold``)."""
    cd, d = _dims(dims)
    vh = volume(d) // 2
    w = np.empty((4, 2, vh, 3, 3), dtype=np.complex128)
    rc = _load().fg_links(_dp(w), cd, KIND[kind], seed, float(eps), int(fold), int(antiperiodic_t))
    if rc:
        raise RuntimeError("fg_links failed")
    return w


def links_slices(dims, t0: int, nt: int, kind: str = "random", seed: int = 0, eps: float = 0.0,
                 fold: bool = True, antiperiodic_t: bool = True) -> np.ndarray:
    """Time slices t0 .. t0+nt-1 (mod X3) of links(dims, ...) without generating the rest:
    W[mu][p][nt*s3][3][3], equal to links(...)[:, :, t0*s3:(t0+nt)*s3] when the range does not wrap."""
    cd, d = _dims(dims)
    s3 = d[0] * d[1] * d[2] // 2
    w = np.empty((4, 2, int(nt) * s3, 3, 3), dtype=np.complex128)
    rc = _load().fg_links_slices(_dp(w), cd, KIND[kind], seed, float(eps), int(fold), int(antiperiodic_t), int(t0), int(nt))
    if rc:
        raise RuntimeError("fg_links_slices failed")
    return w


def spinor_gaussian(dims, parity: int = 0, seed: int = 0) -> np.ndarray:
    """chi[cb][3] complex128 on one parity, re/im ~ N(0,1)."""
    cd, d = _dims(dims)
    chi = np.empty((volume(d) // 2, 3), dtype=np.complex128)
    if _load().fg_spinor_gaussian(_dp(chi), cd, int(parity), seed):
        raise RuntimeError("fg_spinor_gaussian failed")
    return chi


def spinor_planewave(dims, n, v=(1.0, 0.5 - 0.25j, -0.3 + 0.8j), parity: int = 0,
                     antiperiodic_t: bool = True) -> np.ndarray:
    """chi(x) = exp(i p.x) v on one parity; p_3 carries the +1/2 when antiperiodic."""
    cd, d = _dims(dims)
    chi = np.empty((volume(d) // 2, 3), dtype=np.complex128)
    nn = (ctypes.c_int * 4)(*[int(k) for k in n])
    vv = np.ascontiguousarray(np.asarray(v, dtype=np.complex128))
    if _load().fg_spinor_planewave(_dp(chi), cd, int(parity), nn, _dp(vv), int(antiperiodic_t)):
        raise RuntimeError("fg_spinor_planewave failed")
    return chi


def gauge_transform(dims, seed: int = 777) -> np.ndarray:
    """G[p][cb][3][3] complex128, random SU(3) per site."""
    cd, d = _dims(dims)
    g = np.empty((2, volume(d) // 2, 3, 3), dtype=np.complex128)
    if _load().fg_gauge(_dp(g), cd, seed):
        raise RuntimeError("fg_gauge failed")
    return g


def normal_at(seed: int, tag: int, idx: int, k: int) -> float:
    return _load().fg_normal_at(seed, tag, idx, k)


# ---------------------------------------------------------------------------
# The five BASELINE.json configs as seeded recipes.
# ---------------------------------------------------------------------------

LINK_SEED = 11110125
SOURCE_SEED = 20110710


@dataclass(frozen=True)
class Config:
    name: str
    dims: tuple
    kind: str
    eps: float
    mass: float
    tol: float
    maxiter: int
    index: int

    @property
    def vh(self) -> int:
        return volume(self.dims) // 2

    def links(self) -> np.ndarray:
        return links(self.dims, self.kind, LINK_SEED + self.index, self.eps, True, True)

    def links_slices(self, t0: int, nt: int) -> np.ndarray:
        return links_slices(self.dims, t0, nt, self.kind, LINK_SEED + self.index, self.eps, True, True)

    def source(self) -> np.ndarray:
        return spinor_gaussian(self.dims, 0, SOURCE_SEED + self.index)


CONFIGS = {
    "c1_4^4": Config("c1_4^4", (4, 4, 4, 4), "random", 0.0, 0.1, 1e-10, 1000, 1),
    "c2_8^4_free": Config("c2_8^4_free", (8, 8, 8, 8), "unit", 0.0, 0.05, 1e-10, 5000, 2),
    "c2_8^4": Config("c2_8^4", (8, 8, 8, 8), "random", 0.0, 0.05, 1e-10, 5000, 2),
    "c3_16^3x32": Config("c3_16^3x32", (16, 16, 16, 32), "smooth", 0.3, 0.02, 1e-10, 20000, 3),
    "c4_28^3x96": Config("c4_28^3x96", (28, 28, 28, 96), "random", 0.0, 0.0124, 1e-10, 20000, 4),
    "c5_48^3x96": Config("c5_48^3x96", (48, 48, 48, 96), "smooth", 0.5, 0.005, 1e-10, 100000, 5),
}
