"""Host-side logic of bench.py's multi-GPU mode ("replicas only"): world_size-2 gloo on CPU."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch, torch.distributed as dist
import bench
rank, world, local = bench.shard_info(2)
dist.init_process_group("gloo", rank=rank, world_size=world)
ms = bench.reduce_max_time(10.0 + 5.0 * rank, world)          # slowest replica decides
units = bench.total_units(100, 2000, 3, world)
if rank == 0:
    print(json.dumps({"ms": ms, "units": units, "world": world}))
dist.barrier()
dist.destroy_process_group()
"""


def test_two_rank_gloo_max_time_and_units(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29731", WORLD_SIZE="2")
    procs = []
    for r in range(2):
        e = dict(env, RANK=str(r), LOCAL_RANK=str(r))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=e, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=300) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e
    res = json.loads(outs[0][0].strip().splitlines()[-1])
    assert res["world"] == 2
    assert res["ms"] == 15.0                      # max over ranks, not rank 0's own 10 ms
    assert res["units"] == 100 * 2000 * 3 * 2     # whole-job units: every replica's walkers count


def test_shard_info_defaults(monkeypatch):
    sys.path.insert(0, ROOT)
    import bench
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        monkeypatch.delenv(k, raising=False)
    assert bench.shard_info(1) == (0, 1, 0)
    monkeypatch.setenv("WORLD_SIZE", "4"); monkeypatch.setenv("RANK", "3"); monkeypatch.setenv("LOCAL_RANK", "3")
    assert bench.shard_info(4) == (3, 4, 3)
    with pytest.raises(SystemExit):
        bench.shard_info(2)


def test_reference_arm_prints_one_json_line():
    """--impl reference times the oracle on the host cores (bounded sample) and needs no GPU."""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "small",
                          "--steps", "1", "--warmup", "0", "--oracle-dets", "200"], capture_output=True, text=True,
                         timeout=600)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0


SHARD_WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import numpy as np, torch, torch.distributed as dist
import msd_inputs as mi
from oracle import o2
from paper_2406_08314_b200.binding import dist_allreduce
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
x = mi.generate("open-shell")
# slice `rank` of every (k_alpha, k_beta) level bucket, buckets in ascending key order, stable inside (include/msd.h msd_setup_sharded)
ka, kb = np.diff(x.exc_off_a), np.diff(x.exc_off_b)
key = ka * 17 + kb
mine = []
for k in np.unique(key):
    idx = np.nonzero(key == k)[0]
    mine += list(idx[len(idx) * rank // world: len(idx) * (rank + 1) // world])
sub = x.subset_dets(np.array(sorted(mine)))
r = o2.run(sub, want=("ovlp",))
t = torch.from_numpy(np.ascontiguousarray(r["ovlp"]).view(np.float64).copy())      # this rank's partial sum_I c_I d_I^a d_I^b
dist_allreduce()(t)                                                                 # the hook MSDTrial.set_allreduce is given
full = o2.run(x, want=("ovlp",))["ovlp"]
err = float(np.abs(t.numpy().view(np.complex128) - full).max() / np.abs(full).max())
counts = torch.tensor([len(mine)]); dist.all_reduce(counts)
if rank == 0:
    print(json.dumps({"err": err, "n_det_total": int(counts.item()), "n_det": x.n_det}))
dist.barrier()
dist.destroy_process_group()
"""


def test_two_rank_gloo_determinant_shards_sum_to_the_whole(tmp_path):
    """SURVEY.md 8(e)(ii) / 8(f) f4 on CPU: the level-bucket slices of two ranks partition the determinant list, and the
    all-reduce hook turns their partial overlaps (oracle O2 on each slice) into the overlap of the whole trial."""
    script = tmp_path / "shard_worker.py"
    script.write_text(SHARD_WORKER % ROOT)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29733", WORLD_SIZE="2")
    procs = []
    for r in range(2):
        e = dict(env, RANK=str(r), LOCAL_RANK=str(r))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=e, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=300) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e
    res = json.loads(outs[0][0].strip().splitlines()[-1])
    assert res["n_det_total"] == res["n_det"]
    assert res["err"] < 1e-13
