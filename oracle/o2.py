"""ctypes wrapper of oracle tier O2 (oracle/o2.c).  TEST INFRASTRUCTURE (see oracle/__init__.py)."""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle_o2.so")
_SO_LD = os.path.join(_HERE, "liboracle_o2_ld.so")
_libs = {}


def build(force: bool = False, long_double: bool = False) -> str:
    """gcc -O2 -fopenmp, no -ffast-math.  -fcx-limited-range only drops the C99 Annex G NaN/Inf recovery of complex
    multiply/divide (plain (ac-bd, ad+bc) formulas); every real operation stays IEEE.  long_double=True builds the same
    source with -DREAL="long double" (x87 80-bit) for the noise-floor pin P12."""
    src = os.path.join(_HERE, "o2.c")
    so = _SO_LD if long_double else _SO
    if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
        cmd = ["gcc", "-O2", "-march=native", "-fopenmp", "-fcx-limited-range", "-std=c99", "-shared", "-fPIC"]
        if long_double:
            cmd.append('-DREAL=long double')
        subprocess.check_call(cmd + ["-o", so, src, "-lm"])
    return so


def _load(long_double: bool = False):
    if long_double not in _libs:
        lib = ctypes.CDLL(build(long_double=long_double))
        c = ctypes
        lib.msd_oracle_o2.restype = c.c_int
        lib.msd_oracle_o2.argtypes = [c.c_int, c.c_int, c.c_int, c.c_int, c.c_long, c.c_int,
                                      c.c_void_p, c.c_void_p, c.c_double,
                                      c.c_void_p, c.c_void_p, c.c_void_p,
                                      c.c_void_p, c.c_void_p, c.c_int,
                                      c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p, c.c_int]
        lib.msd_oracle_o2_threads.restype = c.c_int
        _libs[long_double] = lib
    return _libs[long_double]


def threads() -> int:
    return int(_load().msd_oracle_o2_threads())


def o2(h1, L, e0, occa, occb, ci, phi_a, phi_b, want=("ovlp", "greens", "energy"), return_G=True, nthreads=0,
       long_double=False):
    """Returns dict(ovlp[nw], G[nw,2,N,N] (if greens and return_G), fb[nw,ng], E[nw,3], kappa[nw]).
    long_double: run the 80-bit build (results are rounded to float64 on output)."""
    lib = _load(long_double)
    h1 = np.ascontiguousarray(h1, dtype=np.float64)
    L = np.ascontiguousarray(L, dtype=np.float64)
    occa = np.ascontiguousarray(occa, dtype=np.int32)
    occb = np.ascontiguousarray(occb, dtype=np.int32)
    ci = np.ascontiguousarray(ci, dtype=np.float64)
    phi_a = np.ascontiguousarray(phi_a, dtype=np.complex128)
    phi_b = np.ascontiguousarray(phi_b, dtype=np.complex128)
    nw, N, na = phi_a.shape
    nb = phi_b.shape[2]
    ng = L.shape[0]
    nd = len(ci)
    assert occa.shape == (nd, na) and occb.shape == (nd, nb) and L.shape == (ng, N, N)
    bits = 1 | (2 if "greens" in want else 0) | (4 if "energy" in want else 0)
    ovlp = np.zeros(nw, dtype=np.complex128)
    kappa = np.zeros(nw, dtype=np.float64)
    fb = np.full((nw, ng), np.nan, dtype=np.complex128)
    E = np.full((nw, 3), np.nan, dtype=np.complex128)
    G = np.zeros((nw, 2, N, N), dtype=np.complex128) if (bits & 2 and return_G) else None
    p = lambda a: a.ctypes.data_as(ctypes.c_void_p) if a is not None else None
    rc = lib.msd_oracle_o2(N, na, nb, ng, nd, nw, p(h1), p(L), float(e0), p(occa), p(occb), p(ci),
                           p(phi_a), p(phi_b), bits, p(ovlp), p(G), p(fb), p(E), p(kappa), int(nthreads))
    if rc != 0:
        raise RuntimeError("msd_oracle_o2 failed rc=%d" % rc)
    out = dict(ovlp=ovlp, fb=fb, E=E, kappa=kappa)
    if G is not None:
        out["G"] = G
    return out


def run(inp, walkers=None, want=("ovlp", "greens", "energy"), return_G=True, nthreads=0, long_double=False):
    pa, pb = inp.phi_a, inp.phi_b
    if walkers is not None:
        pa, pb = pa[walkers], pb[walkers]
    return o2(inp.h1, inp.L, inp.e0, inp.occa, inp.occb, inp.ci, pa, pb, want=want, return_G=return_G,
              nthreads=nthreads, long_double=long_double)
