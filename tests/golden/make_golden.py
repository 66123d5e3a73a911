"""Writes tests/golden/<config>_seed<seed>.json: oracle values at BASELINE.json's FULL sizes.

Calls only ``oracle/`` (tier O2) and ``msd_inputs``; never the CUDA path.  The brute-force oracle costs
~20 TFLOP per walker at the Fe2S2-shaped config, so the expected values of a few sampled
walkers are computed once here and stored as text; tests/test_parity_gpu.py compares the full-batch GPU
result on those walkers.

    python tests/golden/make_golden.py fe2s2 0 57 99        # ~10 min per walker on 8 cores
    python tests/golden/make_golden.py cu2o2 0 1 7 8 100 199
"""
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import msd_inputs as mi  # noqa: E402
from oracle import o2  # noqa: E402


def main():
    name = sys.argv[1]
    walkers = [int(a) for a in sys.argv[2:]]
    nthreads = int(os.environ.get("ORACLE_THREADS", "0"))
    x = mi.generate(name)
    t = time.time()
    r = o2.run(x, walkers=walkers, return_G=False, nthreads=nthreads)
    dt = time.time() - t
    gs = list(range(0, x.n_chol, 8))
    out = {
        "config": name, "seed": x.params["seed"], "input_sha256": x.sha256(), "walkers": walkers,
        "oracle": "oracle/o2.c (tier O2), float64", "oracle_seconds": dt, "threads": o2.threads(),
        "fb_gamma_sample": gs,
        "ovlp": [[float(v.real), float(v.imag)] for v in r["ovlp"]],
        "kappa": [float(v) for v in r["kappa"]],
        "E": [[[float(v.real), float(v.imag)] for v in row] for row in r["E"]],
        "fb": [[[float(v.real), float(v.imag)] for v in row[gs]] for row in r["fb"]],
        "fb_max_abs": [float(np.abs(row).max()) for row in r["fb"]],
    }
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "%s_seed%d.json" % (name, x.params["seed"]))
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    print("wrote", path, "in %.0f s" % dt)


if __name__ == "__main__":
    main()
