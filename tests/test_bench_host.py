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
