#!/usr/bin/env python
"""bench.py -- walker x determinant local-energy + force-bias evaluations per second (BASELINE.json metric).

A "step" is one pass of the whole hot path over one walker batch: msd_force_bias + msd_local_energy
(S1-S9 of SURVEY.md 8(a)) on synthetic inputs shaped like the paper's Fe2S2 workload (BASELINE.json configs[3],
the largest fully specified single-GPU config; stands in for PAPER.md:L315, whose integrals are unavailable).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config fe2s2] [--impl ours|reference]

N > 1 (torchrun): replicas only -- walkers are independent, every rank holds the trial and its
own walker batch (seed + rank), no data-path collective; value = units of all ranks / max-over-ranks time.
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "walker x determinant local-energy + force-bias evaluations per second"
UNIT = "walker*det/s"
FP64_PEAK_DERIVED = 148 * 64 * 2 * 1.965e9 / 1e12     # 148 SMs x 64 FP64 FMA/clk x 2 flop x 1.965 GHz = 37.2 TF


def shard_info(n_gpus: int):
    """(rank, world, local_rank) from the torchrun environment; (0, 1, 0) when run as a plain script."""
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != max(1, n_gpus) and world > 1:
        raise SystemExit("WORLD_SIZE %d does not match --gpus %d" % (world, n_gpus))
    return rank, world, local


def reduce_max_time(ms: float, world: int, device=None) -> float:
    """max over ranks of a per-rank duration (the job is as slow as its slowest replica)."""
    if world == 1:
        return ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


NCU_RAW = os.path.join(ROOT, "profiles", "r02_ncu_raw.csv")


def ncu_traffic(kernel_prefix: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the kernels whose name starts with `kernel_prefix`,
    averaged over their launches, parsed from the RAW page of one `ncu --set full` capture of this same command
    (profiles/r02_ncu_raw.csv = `ncu -i ... --page raw --csv`, command in profiles/r02_ncu_full.md).  Returns
    (bytes per launch, launches) or (None, 0) when the capture is absent."""
    import csv
    try:
        rows = list(csv.reader(open(NCU_RAW)))
    except OSError:
        return None, 0
    hdr = next((r for r in rows if "Kernel Name" in r), None)
    if hdr is None:
        return None, 0
    units = rows[rows.index(hdr) + 1]
    k, rd, wr = hdr.index("Kernel Name"), hdr.index("dram__bytes_read.sum"), hdr.index("dram__bytes_write.sum")
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    tot, n = 0.0, 0
    for r in rows[rows.index(hdr) + 2:]:
        name = r[k][5:] if len(r) > k and r[k].startswith("void ") else (r[k] if len(r) > k else "")   # templated kernels print as "void k<...>"
        if len(r) > max(k, rd, wr) and name.startswith(kernel_prefix):
            tot += float(r[rd].replace(",", "")) * scale.get(units[rd], 1.0) + \
                   float(r[wr].replace(",", "")) * scale.get(units[wr], 1.0)
            n += 1
    return (tot / n, n) if n else (None, 0)


_probes = None


def probes():
    """libmsd_probes.so (paper_2406_08314_b200/csrc/probes.cu): bench-side peak probes, not part of the product ABI."""
    global _probes
    if _probes is None:
        import ctypes as C
        lib = C.CDLL(os.path.join(ROOT, "paper_2406_08314_b200", "libmsd_probes.so"))
        lib.msd_probe_fp64_tflops.restype = C.c_double
        lib.msd_probe_fp64_tflops.argtypes = [C.c_int, C.c_double, C.c_void_p]
        lib.msd_probe_l2_gather_gbs.restype = C.c_double
        lib.msd_probe_l2_gather_gbs.argtypes = [C.c_int, C.c_double, C.c_void_p]
        _probes = lib
    return _probes


def fb_dets_flops(ka: np.ndarray, kb: np.ndarray) -> float:
    """Real FP64 flops of one (walker, determinant) unit of the force-bias determinant pass (W2-W4: minors, adjugates, the
    products c~ R^sbar A[b][a] and their accumulation), from the closed forms of csrc/dets.cu: complex mul = 6, complex
    fma = 8.  k = 1: 0; 2: 14; 3: 9 minors + expansion = 148; 4: 12 two-by-two minors + R + 16 cofactors = 566;
    k >= 5: Gauss-Jordan with the pivot row in registers, 8 k^3 + 14 k^2.  Per unit also W (12) and (ka^2 + kb^2) x 8."""
    def spin(k):
        out = np.zeros_like(k, dtype=np.float64)
        for lev, f in ((2, 14.0), (3, 148.0), (4, 566.0)):
            out[k == lev] = f
        big = k >= 5
        out[big] = 8.0 * k[big] ** 3 + 14.0 * k[big] ** 2
        return out
    return float(np.sum(spin(ka) + spin(kb) + 12.0 + 8.0 * (ka * ka + kb * kb)))


def total_units(n_w: int, n_det: int, steps: int, world: int) -> float:
    return float(n_w) * float(n_det) * steps * world


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        def pump():
            for line in self.proc.stdout:
                self.rows.append(line.strip())
        self.thread = threading.Thread(target=pump, daemon=True)
        self.thread.start()

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [t.strip() for t in r.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def cpu_oracle_sample(inp, n_det_sample: int, steps: int = 1, warmup: int = 0):
    """The oracle as it stands (tier O2, oracle/o2.c) on walker 0 and the first n_det_sample determinants
    (force bias + local energy).  Returns (walker*det/s, seconds per step, threads)."""
    from oracle import o2
    sub = inp.subset_dets(np.arange(min(n_det_sample, inp.n_det)))
    for _ in range(warmup):
        o2.run(sub, walkers=[0], return_G=False)
    ts = []
    for _ in range(steps):
        t = time.perf_counter()
        o2.run(sub, walkers=[0], return_G=False)
        ts.append(time.perf_counter() - t)
    sec = sum(ts) / len(ts)
    return sub.n_det / sec, sec, o2.threads()


def cpu_wick_sample(inp, n_walkers: int):
    """the same Wick's-theorem algorithm restated for the CPU (oracle/wick_cpu.c, OpenMP), force bias
    and local energy of the first n_walkers walkers against ALL determinants.  Returns (walker*det/s, seconds, threads)."""
    from oracle import wick
    ws = list(range(min(n_walkers, inp.n_w)))
    wick.run(inp, walkers=ws[:1])              # warm-up (page in L, build the library)
    t = time.perf_counter()
    wick.run(inp, walkers=ws, want=("fb", "energy"))
    sec = time.perf_counter() - t
    return len(ws) * inp.n_det / sec, sec, wick.threads()


def run_reference(args, rank):
    """--impl reference: the CPU oracle, timed on the host cores on a bounded sample of the same workload."""
    if rank != 0:
        return
    import msd_inputs as mi
    inp = mi.generate(args.config)
    nsamp = args.oracle_dets
    thr, sec, cores = cpu_oracle_sample(inp, nsamp, steps=args.steps, warmup=min(args.warmup, 1))
    sample = "walker 0 x first %d of %d determinants of '%s' per step (force bias + local energy, tier O2)" % (
        min(nsamp, inp.n_det), inp.n_det, args.config)
    line = {"impl": "reference", "metric": METRIC, "value": thr, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64 (complex128)", "data": "synthetic",
            "config": {"workload": args.config, "N": inp.N, "n_alpha": inp.n_alpha, "n_beta": inp.n_beta,
                       "n_chol": inp.n_chol, "n_det": inp.n_det, "n_w": inp.n_w, "sample": sample},
            "cpu_baseline": {"value": thr, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": thr, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="fe2s2")
    ap.add_argument("--oracle-dets", type=int, default=4000, help="determinants in the CPU-oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--n-det", type=int, default=None, help="override the determinant count (kernel sweep, configs[4])")
    ap.add_argument("--max-level", type=int, default=None, help="override the maximum excitation level (kernel sweep)")
    ap.add_argument("--shard", default="replicas", choices=["replicas", "dets"],
                    help="N > 1: 'replicas' (default; every rank its own walker batch, no collective, weak scaling) or 'dets' "
                         "(SURVEY.md 8(f) f4: every rank 1/N of every level bucket of the determinant list and the SAME walkers, "
                         "one NCCL all-reduce of the partial W / C / E sums per determinant pass, strong scaling)")
    args = ap.parse_args()
    rank, world, local = shard_info(args.gpus)
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.warmup < 3:
        args.warmup = 3

    import torch
    import msd_inputs as mi
    from paper_2406_08314_b200 import build as _build
    _build.build()                  # no-op when libmsd_b200.so is up to date (nvcc, sm_100a, in-tree)
    import paper_2406_08314_b200 as msd

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    over = {}
    if args.n_det is not None:
        over["n_det"] = args.n_det
    if args.max_level is not None:
        over["max_level"] = args.max_level
    inp = mi.generate(args.config, **over)
    shard_dets = args.shard == "dets" and world > 1
    if rank > 0 and not shard_dets:   # replicas: same trial, a different walker batch per rank
        rng = np.random.default_rng(inp.params["seed"] + 7919 * rank)
        inp = inp.with_walkers(mi.walkers_from_rng(rng, inp.n_w, inp.N, inp.n_alpha),
                               mi.walkers_from_rng(rng, inp.n_w, inp.N, inp.n_beta))
    trial = msd.setup_from_inputs(inp, shard=(rank, world) if shard_dets else (0, 1))
    if shard_dets:
        trial.set_allreduce(msd.dist_allreduce())
    units_world = 1 if shard_dets else world          # determinant shards work on ONE batch together
    info = trial.info()
    stream = torch.cuda.current_stream()
    h_a = torch.from_numpy(inp.phi_a).pin_memory()
    h_b = torch.from_numpy(inp.phi_b).pin_memory()
    d_a = h_a.to(dev)
    d_b = h_b.to(dev)
    fb = torch.empty((inp.n_w, inp.n_chol), dtype=torch.complex128, device=dev)
    en = torch.empty((inp.n_w, 3), dtype=torch.complex128, device=dev)
    h_fb = torch.empty((inp.n_w, inp.n_chol), dtype=torch.complex128).pin_memory()
    h_en = torch.empty((inp.n_w, 3), dtype=torch.complex128).pin_memory()
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device=dev)   # > 126 MB L2

    def step():
        trial.force_bias(d_a, d_b, out=fb)
        trial.local_energy(d_a, d_b, out=en)

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    # ---- timed region: K steps, CUDA events on the launching stream, L2 flushed between steps ----
    sampler = ClockSampler(local)
    sampler.start()
    l0 = trial.launch_count()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    for a, b in evs:
        flush.zero_()
        a.record(stream)
        step()
        b.record(stream)
    barrier()
    launches = trial.launch_count() - l0
    clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in evs]
    total_ms = reduce_max_time(sum(step_ms), world, dev)
    value = total_units(inp.n_w, inp.n_det, args.steps, units_world) / (total_ms * 1e-3)

    # ---- the same two outputs from the fused call msd_force_bias_energy (one pass of the determinant kernels) ----
    fused_out = torch.empty((inp.n_w, inp.n_chol + 3), dtype=torch.complex128, device=dev)
    for _ in range(2):
        trial.force_bias_energy(d_a, d_b, out=fused_out)
    barrier()
    fev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for a, b in fev:
        flush.zero_()
        a.record(stream)
        trial.force_bias_energy(d_a, d_b, out=fused_out)
        b.record(stream)
    barrier()
    fused_ms = reduce_max_time(sum(a.elapsed_time(b) for a, b in fev), world, dev)
    fused = {"call": "msd_force_bias_energy (force bias and local energy of the batch from ONE pass: the energy-mode "
                     "determinant kernels also accumulate C, fb = X0 + C.B/W, SURVEY.md 8(c) W6)",
             "value": total_units(inp.n_w, inp.n_det, args.steps, units_world) / (fused_ms * 1e-3), "unit": UNIT,
             "ms_per_step": fused_ms / args.steps,
             "max_rel_diff_fb_vs_separate_calls": float(((fused_out[:, :inp.n_chol] - fb).abs().amax(dim=1)
                                                         / fb.abs().amax(dim=1)).max().item()),
             "max_abs_diff_E_vs_separate_calls": float((fused_out[:, inp.n_chol:] - en).abs().max().item())}

    # ---- per-call throughputs and the paper's block mix (a block = 25 propagation
    # steps, each needing one force bias and one overlap, + 1 energy estimate) ----
    ov = torch.empty(inp.n_w, dtype=torch.complex128, device=dev)
    calls = {"msd_overlap": lambda: trial.overlap(d_a, d_b, out=ov),
             "msd_force_bias": lambda: trial.force_bias(d_a, d_b, out=fb),
             "msd_local_energy": lambda: trial.local_energy(d_a, d_b, out=en),
             "msd_force_bias_overlap": lambda: trial.force_bias_overlap(d_a, d_b, out=fb, out_ovlp=ov)}
    per_call = {}
    for cname, fn in calls.items():
        fn()
        barrier()
        cev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        for a, b in cev:
            flush.zero_()
            a.record(stream)
            fn()
            b.record(stream)
        barrier()
        cms = reduce_max_time(sum(a.elapsed_time(b) for a, b in cev), world, dev) / args.steps
        per_call[cname] = {"ms": cms, "value": total_units(inp.n_w, inp.n_det, 1, units_world) / (cms * 1e-3), "unit": UNIT}
    t_ov, t_fb, t_e = (per_call[k]["ms"] for k in ("msd_overlap", "msd_force_bias", "msd_local_energy"))
    block_mix = {"definition": "N_w N_d 25 / (25 (t_fb + t_ovlp) + t_E): walker x determinant propagation-step evaluations "
                               "per second in the paper's block of 25 steps + 1 energy estimate (PAPER.md:L303-309)",
                 "value": total_units(inp.n_w, inp.n_det, 25, units_world) / ((25.0 * (t_fb + t_ov) + t_e) * 1e-3),
                 "unit": "walker*det*step/s", "block_ms": 25.0 * (t_fb + t_ov) + t_e,
                 "energy_share_of_block": t_e / (25.0 * (t_fb + t_ov) + t_e)}
    # the same block when every step takes its force bias and overlap from ONE determinant pass (msd_force_bias_overlap)
    t_fbo = per_call["msd_force_bias_overlap"]["ms"]
    block_mix["one_pass"] = {"definition": "N_w N_d 25 / (25 t_fb+ovlp + t_E) with msd_force_bias_overlap (force bias and overlap of "
                                           "the step's walkers from one determinant pass)",
                             "value": total_units(inp.n_w, inp.n_det, 25, units_world) / ((25.0 * t_fbo + t_e) * 1e-3),
                             "unit": "walker*det*step/s", "block_ms": 25.0 * t_fbo + t_e}

    # ---- one propagation step around the path (force bias, B(x - xbar), new overlap, Eq. 8-12) ----
    trial.propagator_setup(0.005, 6, inp.h1, inp.L)
    xf = torch.randn((inp.n_w, inp.n_chol), dtype=torch.float64, device=dev,
                     generator=torch.Generator(device=dev).manual_seed(1234 + rank))
    wts = torch.ones(inp.n_w, dtype=torch.float64, device=dev)
    sout = torch.empty((inp.n_w, 8), dtype=torch.float64, device=dev)
    pa_w, pb_w = d_a.clone(), d_b.clone()
    trial.propagate(pa_w, pb_w, xf, weights=wts, out=sout)
    barrier()
    pev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for a, b in pev:
        pa_w.copy_(d_a); pb_w.copy_(d_b)          # every timed step starts from the orthonormal walkers
        flush.zero_()
        a.record(stream)
        trial.propagate(pa_w, pb_w, xf, weights=wts, out=sout)
        b.record(stream)
    barrier()
    pms = reduce_max_time(sum(a.elapsed_time(b) for a, b in pev), world, dev) / args.steps
    propagation = {"call": "msd_propagate: force bias + overlap of the walkers, field matrices (DMMA), orbital update with a "
                           "6th-order Taylor series, overlap of the new walkers, Eq. 8-12 (dt = 0.005)",
                   "ms_per_step": pms, "value": total_units(inp.n_w, inp.n_det, 1, units_world) / (pms * 1e-3),
                   "unit": "walker*det*step/s", "finite": bool(torch.isfinite(sout).all().item())}

    # ---- end to end: the C-ABI *_host calls (pinned HOST buffers; H2D + kernels + D2H inside each call) ----
    def e2e_step():
        trial.force_bias_host(h_a, h_b, out=h_fb)
        trial.local_energy_host(h_a, h_b, out=h_en)

    e2e_step()
    barrier()
    ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n_e2e = max(3, min(args.steps, 10))
    ea.record(stream)
    for _ in range(n_e2e):
        e2e_step()
    eb.record(stream)
    barrier()
    e2e_ms = reduce_max_time(ea.elapsed_time(eb), world, dev)
    e2e_val = total_units(inp.n_w, inp.n_det, n_e2e, units_world) / (e2e_ms * 1e-3)
    h2d = 2 * (h_a.numel() * 16 + h_b.numel() * 16)      # each of the two host calls copies the walkers in
    d2h = h_fb.numel() * 16 + h_en.numel() * 16

    # ---- roofline of the dominant kernel (phase timings from CUDA events inside the library, same stream) ----
    roofline = None
    phases = None
    roofline_dets = roofline_fb_dets = roofline_other = None
    if rank == 0 and not shard_dets:      # (the profiled calls below would be collectives in determinant-shard mode)
        peak = float(probes().msd_probe_fp64_tflops(1, 30.0, None))
        l2_gather = float(probes().msd_probe_l2_gather_gbs(32, 20.0, None))
        trial.set_profiling(True)
        acc = {}
        reps = 3
        for _ in range(reps):
            flush.zero_()
            trial.local_energy(d_a, d_b, out=en)
            for k, v in trial.phase_ms().items():
                acc[k] = acc.get(k, 0.0) + v / reps
        fbacc = {}
        for _ in range(reps):
            flush.zero_()
            trial.force_bias(d_a, d_b, out=fb)
            for k, v in trial.phase_ms().items():
                fbacc[k] = fbacc.get(k, 0.0) + v / reps
        trial.set_profiling(False)
        Pa = info["n_o_alpha"] * info["n_v_alpha"]
        Pb = info["n_o_beta"] * info["n_v_beta"]
        nr_a = inp.n_alpha + info["n_v_alpha"]
        nr_b = inp.n_beta + info["n_v_beta"]
        ng, nw, N = inp.n_chol, inp.n_w, inp.N
        # complex MAC = 8 flops (the method's work; the V kernel executes 6 per complex MAC by the 3-multiplication scheme);
        # the same-spin products are symmetric: only x <= y is algorithmic work
        flops_v = 8.0 * ng * nw * (Pa * Pb + Pa * (Pa + 1) / 2 + Pb * (Pb + 1) / 2)
        # S7 (fused kernel): Lambda = L_sub Theta over the N - n_sigma virtual orbitals when the reference is the first n
        # orbitals (Theta[occ] = 1), real x complex MAC = 4; dense steps per (walker, slice, spin): Theta_v T (8 n_v n n),
        # Bfull T[:, pos] (8 n_v n n_o), tr(T T) (8 n^2)
        contiguous = (list(inp.occ_ref_a) == list(range(inp.n_alpha)) and list(inp.occ_ref_b) == list(range(inp.n_beta))
                      and inp.n_alpha == inp.n_beta and inp.n_alpha % 2 == 0)
        kv_a = N - inp.n_alpha if contiguous else N
        kv_b = N - inp.n_beta if contiguous else N
        flops_lam = 4.0 * (ng + 1) * nw * (kv_a * nr_a * inp.n_alpha + kv_b * nr_b * inp.n_beta)
        nva, nvb, noa, nob = info["n_v_alpha"], info["n_v_beta"], info["n_o_alpha"], info["n_o_beta"]
        flops_dense = 8.0 * ng * nw * (nva * inp.n_alpha * (inp.n_alpha + noa) + inp.n_alpha ** 2
                                       + nvb * inp.n_beta * (inp.n_beta + nob) + inp.n_beta ** 2)
        phases = {"energy_ms": {"reference": acc["reference"], "s7_lambda_and_dense": acc["p1"] + acc["p2"],
                                "v_gemm": acc["p3"], "dets": acc["p4"], "assemble": acc["p5"]},
                  "force_bias_ms": {"reference": fbacc["reference"], "dets": fbacc["p1"], "greens_fb_gemm": fbacc["p2"]}}
        step_mean = sum(step_ms) / len(step_ms)
        s7_ms, v_ms = acc["p1"] + acc["p2"], acc["p3"]
        src = ("measured live by the bench-side probe (csrc/probes.cu, libmsd_probes.so): register-resident DMMA m8n8k4 "
               "loop; MEASURED_PEAKS.json has no FP64 entry; derived 148 SM x 64 FMA/clk x 1.965 GHz = %.1f" % FP64_PEAK_DERIVED)

        def tensor_roofline(kernel, prefix, flops, ms, note):
            tr, nl = ncu_traffic(prefix)
            return {"kernel": kernel, "bound": "tensor", "achieved": flops / (ms * 1e-3) / 1e12, "peak": peak,
                    "unit": "TFLOP/s", "frac": flops / (ms * 1e-3) / 1e12 / peak if peak > 0 else None, "peak_source": src,
                    "traffic": tr, "traffic_note": "dram__bytes_read.sum + dram__bytes_write.sum per launch, mean over the %d "
                    "launches of this kernel in profiles/r02_ncu_raw.csv (raw page of one ncu --set full capture of this "
                    "command; null when absent)" % nl, "ms": ms, "share_of_step": ms / step_mean,
                    "algorithmic_flops_per_step": flops, "note": note}
        r_s7 = tensor_roofline("k_energy_fused (S7: Lambda = L_sub Theta by FP64 DMMA + dense intermediates, 1 launch)",
                               "k_energy_fused", flops_lam + flops_dense, s7_ms,
                               "executes (40/35 padded rows) more DMMA than the algorithmic count")
        r_v = tensor_roofline("k_vgemm3m (V contractions alpha-beta, alpha-alpha, beta-beta: 3 launches on forked streams; the walkers with an "
                              "ill-conditioned reference block go through the 4-multiplication k_gemm_tn instead: DESIGN.md section 7)",
                              "k_vgemm3m", flops_v, v_ms,
                              "achieved counts 8 flops per complex MAC (the method's work); the kernel executes 6 (3-multiplication "
                              "scheme), i.e. %.2f TFLOP/s of executed DMMA on 48 x 48 tiles" % (0.75 * flops_v / (v_ms * 1e-3) / 1e12))
        # the dominant kernel = the one with the larger share of the step
        roofline, roofline_other = (r_s7, r_v) if s7_ms >= v_ms else (r_v, r_s7)

        # energy-mode dets kernels: bound by the L2 -> SM gathers of V / Vbar; algorithmic bytes =
        # 16 B x (ka^2 kb^2 + C(ka,2)^2 + C(kb,2)^2) per walker x determinant, from the level histogram of the inputs
        ka = np.diff(inp.exc_off_a).astype(np.float64)
        kb = np.diff(inp.exc_off_b).astype(np.float64)
        gathers = float(np.sum(ka * ka * kb * kb + (ka * (ka - 1) / 2) ** 2 + (kb * (kb - 1) / 2) ** 2))
        l2_bytes = 16.0 * gathers * nw
        roofline_dets = {"kernel": "k_dets_cf<2> + k_dets_gen<2> + k_dets_coop<2> (energy mode, forked over side streams)",
                         "bound": "l2", "achieved": l2_bytes / (acc["p4"] * 1e-3) / 1e9, "peak": l2_gather, "unit": "GB/s",
                         "frac": l2_bytes / (acc["p4"] * 1e-3) / 1e9 / l2_gather if l2_gather > 0 else None,
                         "peak_source": "measured live by the bench-side probe (csrc/probes.cu): random 128-byte lines of a "
                                        "32 MB L2-resident buffer, 16 B per lane, 8 independent loads in flight per lane",
                         "algorithmic_l2_bytes_per_step": l2_bytes, "share_of_step": acc["p4"] / (sum(step_ms) / len(step_ms))}
        # force-bias determinant pass (k_dets_pull + k_dets_gen<1>): plain FP64 ALU work against the FP64 peak
        fl = fb_dets_flops(ka, kb) * nw
        roofline_fb_dets = {"kernel": "k_dets_pull + k_dets_gen<1> (force-bias mode: minors, adjugates, CI reduction)",
                            "bound": "alu", "achieved": fl / (fbacc["p1"] * 1e-3) / 1e12, "peak": peak, "unit": "TFLOP/s",
                            "frac": fl / (fbacc["p1"] * 1e-3) / 1e12 / peak if peak > 0 else None,
                            "peak_source": "FP64 pipe (DFMA and DMMA share it): the live DMMA probe",
                            "algorithmic_flops_per_step": fl, "ms": fbacc["p1"],
                            "share_of_step": fbacc["p1"] / (sum(step_ms) / len(step_ms))}

    if rank != 0:
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
            dist.destroy_process_group()
        return

    cpu_baseline = None
    if not args.no_cpu_baseline:
        thr, sec, cores = cpu_oracle_sample(inp, args.oracle_dets)
        cpu_baseline = {"value": thr, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": "walker 0 x first %d of %d determinants (force bias + local energy, tier O2), %.1f s"
                                  % (min(args.oracle_dets, inp.n_det), inp.n_det, sec)}
    cpu_wick = None
    if not args.no_cpu_baseline:
        thr, sec, cores = cpu_wick_sample(inp, inp.n_w)
        cpu_wick = {"value": thr, "unit": UNIT, "cores": cores, "kind": "wick (same algorithm on the CPU, oracle/wick_cpu.c)",
                    "sample": "all %d walkers x all %d determinants (force bias + local energy in one pass), %.1f s"
                              % (inp.n_w, inp.n_det, sec)}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "strong" if shard_dets else "weak",
            "vs_baseline": None, "dtype": "f64 (complex128)", "data": "synthetic",
            "config": {"workload": args.config, "N": inp.N, "n_alpha": inp.n_alpha, "n_beta": inp.n_beta,
                       "n_chol": inp.n_chol, "n_det": inp.n_det, "n_w": inp.n_w, "active_window": info,
                       "step": "msd_force_bias + msd_local_energy (two calls; the fused one-pass call is reported under 'fused')", "l2": "flushed between timed steps (256 MB write)",
                       "parallelism": ("determinant shards x%d (one all-reduce per determinant pass)" if shard_dets else "replicas x%d") % world, "input_sha256": inp.sha256()[:16]},
            "clocks": clocks,
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": n_e2e},
            "gpu_launches": int(launches),
            "fused": fused, "per_call": per_call, "block_mix": block_mix, "propagation": propagation,
            "roofline": roofline, "roofline_second_tensor_kernel": roofline_other, "roofline_dets": roofline_dets,
            "roofline_fb_dets": roofline_fb_dets,
            "cpu_baseline": cpu_baseline, "cpu_wick_baseline": cpu_wick, "phases": phases,
            "step_ms": {"min": min(step_ms), "median": statistics.median(step_ms), "max": max(step_ms)}}
    print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
