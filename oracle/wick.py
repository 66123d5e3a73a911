"""ctypes wrapper of oracle/wick_cpu.c: the multi-threaded CPU restatement of the Wick's-theorem algorithm W1-W10
(the like-for-like CPU baseline).  TEST / BENCH INFRASTRUCTURE (see oracle/__init__.py); checked
against tier O2 in tests/test_oracle_pins.py."""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libwick_cpu.so")
_lib = None


def build(force: bool = False) -> str:
    src = os.path.join(_HERE, "wick_cpu.c")
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-march=native", "-fopenmp", "-fcx-limited-range", "-std=c99", "-shared",
                               "-fPIC", "-o", _SO, src, "-lm"])
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        c = ctypes
        lib.msd_wick_cpu.restype = c.c_int
        lib.msd_wick_cpu.argtypes = [c.c_int, c.c_int, c.c_int, c.c_int, c.c_int64, c.c_int, c.c_void_p, c.c_void_p,
                                     c.c_double] + [c.c_void_p] * 11 + [c.c_int] + [c.c_void_p] * 3 + [c.c_int]
        lib.msd_wick_cpu_threads.restype = c.c_int
        _lib = lib
    return _lib


def threads() -> int:
    return int(_load().msd_wick_cpu_threads())


def run(inp, walkers=None, want=("ovlp", "fb", "energy"), nthreads=0):
    """Returns dict(ovlp[nw], fb[nw,ng], E[nw,3]) for the walkers (all by default) of an msd_inputs.MSDInputs."""
    lib = _load()
    pa, pb = inp.phi_a, inp.phi_b
    if walkers is not None:
        pa, pb = pa[walkers], pb[walkers]
    pa = np.ascontiguousarray(pa, dtype=np.complex128)
    pb = np.ascontiguousarray(pb, dtype=np.complex128)
    f64 = lambda a: np.ascontiguousarray(a, dtype=np.float64)
    i32 = lambda a: np.ascontiguousarray(a, dtype=np.int32)
    i64 = lambda a: np.ascontiguousarray(a, dtype=np.int64)
    h1, L, ci = f64(inp.h1), f64(inp.L), f64(inp.ci)
    arrs = [i32(inp.occ_ref_a), i32(inp.occ_ref_b), i64(inp.exc_off_a), i32(inp.holes_a), i32(inp.parts_a),
            i64(inp.exc_off_b), i32(inp.holes_b), i32(inp.parts_b)]
    nw, ng = pa.shape[0], L.shape[0]
    bits = (1 if "ovlp" in want else 0) | (2 if "fb" in want else 0) | (4 if "energy" in want else 0)
    ovlp = np.full(nw, np.nan, dtype=np.complex128)
    fb = np.full((nw, ng), np.nan, dtype=np.complex128)
    E = np.full((nw, 3), np.nan, dtype=np.complex128)
    p = lambda a: a.ctypes.data_as(ctypes.c_void_p)
    rc = lib.msd_wick_cpu(inp.N, inp.n_alpha, inp.n_beta, ng, inp.n_det, nw, p(h1), p(L), float(inp.e0),
                          *[p(a) for a in arrs], p(ci), p(pa), p(pb), bits, p(ovlp), p(fb), p(E), int(nthreads))
    if rc != 0:
        raise RuntimeError("msd_wick_cpu failed rc=%d" % rc)
    return dict(ovlp=ovlp, fb=fb, E=E)
