"""Writes tests/golden/<case>.json: oracle values at BASELINE.json's FULL sizes.

Calls only ``oracle/`` (tier O2) and ``msd_inputs``; never the CUDA path.  The brute-force oracle costs
~20 TFLOP per walker at the Fe2S2-shaped config, so the expected values of sampled
walkers are computed once here and stored as text; tests/test_parity_gpu.py compares the full-batch GPU
result with them.  Per file (plan of SURVEY.md 8(d) "Oracle timing beside it"):

    walkers / ovlp / E / fb (every 8th gamma)   energy walkers (the L loop per determinant: minutes per walker)
    fb_walkers / fb_full                         force bias on >= 16 walkers, every gamma (no L loop per determinant)
    ovlp_all                                     overlap of EVERY walker of the batch

    python tests/golden/make_golden.py fe2s2 --energy 0 7 8 57 99 --fb 0-15 --ovlp-all     # ~10 min per energy walker on 8 cores
    python tests/golden/make_golden.py cu2o2 --energy 0 1 7 8 100 199
    python tests/golden/make_golden.py sweep --n-det 100000 --max-level 8 --energy 64 --fb 7 8 --ovlp-all
    python tests/golden/make_golden.py sweep --n-det 1000000 --max-level 10 --ovlp-all

An existing file is extended: sections that are not requested are kept as they are (their inputs are identified by
input_sha256, which must match).
"""
import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import msd_inputs as mi  # noqa: E402
from oracle import o2  # noqa: E402


def _ids(tokens):
    out = []
    for t in tokens:
        if "-" in t:
            a, b = t.split("-")
            out += list(range(int(a), int(b) + 1))
        else:
            out.append(int(t))
    return out


def _c(v):
    return [float(v.real), float(v.imag)]


def case_name(name, seed, n_det=None, max_level=None):
    tag = name
    if n_det is not None:
        tag += "_nd%d" % n_det
    if max_level is not None:
        tag += "_K%d" % max_level
    return "%s_seed%d" % (tag, seed)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("name")
    ap.add_argument("--n-det", type=int, default=None)
    ap.add_argument("--max-level", type=int, default=None)
    ap.add_argument("--energy", nargs="*", default=[])
    ap.add_argument("--fb", nargs="*", default=[])
    ap.add_argument("--ovlp-all", action="store_true")
    a = ap.parse_args()
    over = {}
    if a.n_det is not None:
        over["n_det"] = a.n_det
    if a.max_level is not None:
        over["max_level"] = a.max_level
    nthreads = int(os.environ.get("ORACLE_THREADS", "0"))
    x = mi.generate(a.name, **over)
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)),
                        case_name(a.name, x.params["seed"], a.n_det, a.max_level) + ".json")
    out = {}
    if os.path.exists(path):
        out = json.load(open(path))
        assert out["input_sha256"] == x.sha256(), "existing golden file belongs to other inputs"
    out.update({"config": a.name, "overrides": over, "seed": x.params["seed"], "input_sha256": x.sha256(),
                "oracle": "oracle/o2.c (tier O2), float64", "threads": o2.threads()})
    ew, fw = _ids(a.energy), _ids(a.fb)
    if ew:
        t = time.time()
        r = o2.run(x, walkers=ew, return_G=False, nthreads=nthreads)
        gs = list(range(0, x.n_chol, 8))
        new = {"walkers": ew, "ovlp": [_c(v) for v in r["ovlp"]], "kappa": [float(v) for v in r["kappa"]],
               "E": [[_c(v) for v in row] for row in r["E"]], "fb": [[_c(v) for v in row[gs]] for row in r["fb"]],
               "fb_max_abs": [float(np.abs(row).max()) for row in r["fb"]]}
        # energy walkers already stored (same inputs, same oracle) are kept; the new ones are merged in by walker index
        old = {w: i for i, w in enumerate(out.get("walkers", []))} if out.get("fb_gamma_sample", gs) == gs else {}
        merged = sorted(set(old) | set(ew))
        for key in ("ovlp", "kappa", "E", "fb", "fb_max_abs"):
            out[key] = [new[key][ew.index(w)] if w in ew else out[key][old[w]] for w in merged]
        out.update({"walkers": merged, "fb_gamma_sample": gs,
                    "oracle_seconds": out.get("oracle_seconds", 0.0) + time.time() - t})
        print("energy walkers %s: %.0f s" % (ew, time.time() - t), flush=True)
    if fw:
        t = time.time()
        r = o2.run(x, walkers=fw, want=("ovlp", "greens"), return_G=False, nthreads=nthreads)
        out.update({"fb_walkers": fw, "fb_full": [[_c(v) for v in row] for row in r["fb"]]})
        print("force-bias walkers %s: %.0f s" % (fw, time.time() - t), flush=True)
    if a.ovlp_all:
        t = time.time()
        r = o2.run(x, want=("ovlp",), nthreads=nthreads)
        out.update({"ovlp_all": [_c(v) for v in r["ovlp"]], "kappa_all": [float(v) for v in r["kappa"]]})
        print("overlap of all %d walkers: %.0f s" % (x.n_w, time.time() - t), flush=True)
    with open(path, "w") as f:
        json.dump(out, f, separators=(",", ":"))
    print("wrote", path)


if __name__ == "__main__":
    main()
