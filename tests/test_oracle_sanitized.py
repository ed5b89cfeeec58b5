"""The oracle and the generator rebuilt with -fsanitize=undefined -fno-sanitize-recover (gcc's UBSan:
signed overflow, out-of-bounds on known-size arrays, misaligned or null pointer use, bad shifts abort
the process) and run on the small configurations: they must finish and return the bits of the
regular build.  (compute-sanitizer is not available for the CUDA side on this pool; its stand-in is
tests/test_gpu_guards.py.)"""
import ctypes
import os
import subprocess
import sys
import textwrap

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SCRIPT = textwrap.dedent("""
    import ctypes, sys
    import numpy as np
    sys.path.insert(0, %(root)r)
    import fieldgen, oracle
    # regular build first
    dims = (4, 2, 6, 4)
    W = fieldgen.links(dims, "smooth", seed=3, eps=0.4)
    b = fieldgen.spinor_gaussian(dims, 0, seed=4)
    ref_hop = oracle.dslash(b, W, dims, 1)
    ref_x, ref_it, ref_rho, _, _ = oracle.cg(b, W, dims, 0.1, 1e-10, 500)
    h = np.ascontiguousarray(np.stack([b, fieldgen.spinor_gaussian(dims, 1, seed=5)]))
    ref_psi, _, _, _ = oracle.solve_M(h, W, dims, 0.1, 1e-10, 500)
    # swap in the sanitized libraries and repeat
    fieldgen._lib = None; fieldgen._LIB = %(fg)r; fieldgen.build = lambda *a, **k: fieldgen._LIB
    oracle._lib = None; oracle._LIB = %(orc)r; oracle.build = lambda *a, **k: oracle._LIB
    W2 = fieldgen.links(dims, "smooth", seed=3, eps=0.4)
    b2 = fieldgen.spinor_gaussian(dims, 0, seed=4)
    assert np.array_equal(W, W2) and np.array_equal(b, b2)
    assert np.array_equal(oracle.dslash(b2, W2, dims, 1), ref_hop)
    x, it, rho, _, _ = oracle.cg(b2, W2, dims, 0.1, 1e-10, 500)
    assert it == ref_it and np.array_equal(x, ref_x)
    psi, _, _, _ = oracle.solve_M(h, W2, dims, 0.1, 1e-10, 500)
    assert np.array_equal(psi, ref_psi)
    out, fl, by = oracle.dslash_counted(b2, W2, dims, 1)
    assert fl == 576 * len(b2) and by == 1584 * len(b2)
    print("sanitized ok")
""")


def test_oracle_and_generator_run_clean_under_ubsan(tmp_path):
    flags = ["-O1", "-g", "-fsanitize=undefined", "-fno-sanitize-recover=undefined", "-fopenmp", "-fPIC", "-shared", "-std=c11"]
    orc = str(tmp_path / "liboracle_ubsan.so")
    fg = str(tmp_path / "libfieldgen_ubsan.so")
    subprocess.check_call(["gcc"] + flags + ["-o", orc, os.path.join(ROOT, "oracle", "stag_oracle.c"), "-lm"])
    subprocess.check_call(["gcc"] + flags + ["-o", fg, os.path.join(ROOT, "fieldgen", "fieldgen.c"), "-lm"])
    r = subprocess.run([sys.executable, "-c", SCRIPT % {"root": ROOT, "fg": fg, "orc": orc}],
                       capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and "sanitized ok" in r.stdout, r.stdout + r.stderr
    assert "runtime error" not in r.stderr
