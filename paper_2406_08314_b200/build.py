"""Build libmsd_b200.so in-tree with nvcc for sm_100a.

The library has a plain C ABI (include/msd.h), so no torch extension machinery is involved:
    nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo -O3 ... -shared -o libmsd_b200.so
The .so is git-ignored but travels to the GPU box with the gpurun snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libmsd_b200.so")
SOURCES = ["msd_api.cu", "pack.cu", "reference.cu", "dets.cu", "dense.cu", "gemm.cu", "propagate.cu"]
# bench-side peak probes (FP64 DMMA/DFMA, L2 gather): a separate library that only bench.py loads, not the product ABI
PROBES_SO = os.path.join(HERE, "libmsd_probes.so")
PROBES_SRC = "probes.cu"
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
              "-Xcompiler", "-fPIC", "-diag-suppress", "128"]


def _nvcc() -> str:
    cand = os.environ.get("NVCC")
    if cand:
        return cand
    if os.path.exists("/usr/local/cuda/bin/nvcc"):
        return "/usr/local/cuda/bin/nvcc"
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(SO) or not os.path.exists(PROBES_SO):
        return True
    t = os.path.getmtime(SO)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    deps.append(os.path.join(HERE, "..", "include", "msd.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return SO
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    procs, objs = [], []
    for src in SOURCES + [PROBES_SRC]:
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
              ["-c", os.path.join(CSRC, src), "-o", obj]
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    failed = False
    for src, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0:
            failed = True
            sys.stderr.write("nvcc failed for %s:\n%s\n" % (src, out))
        elif verbose or out.strip():
            sys.stderr.write(out)
    if failed:
        raise RuntimeError("nvcc compilation failed")
    link = [_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o"]
    subprocess.check_call(link + [SO] + objs[:-1] + ["-lcudart"])
    subprocess.check_call(link + [PROBES_SO] + objs[-1:] + ["-lcudart"])
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
