"""N > 1 host logic on CPU (gloo, world_size 2): the path does not shard (BASELINE north_star: one GPU, no
collectives), so bench.py runs N independent replicas and only reduces the TIME (max over ranks); the reference arm
runs on rank 0 alone.  DESIGN.md section 9."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
mine = 1.0 + 0.5 * rank                       # rank 1 is the slow replica
t = bench.max_over_ranks(mine, dist, torch.device("cpu"))
v = bench.replica_throughput(world, 10, t)
dist.barrier()
# one file per rank: two ranks printing to one pipe can interleave inside a line
with open(os.path.join({out!r}, "rank%d.json" % rank), "w") as f:
    json.dump({{"rank": rank, "t": t, "value": v}}, f)
dist.destroy_process_group()
"""


def _launch(code, extra_env=None, nproc=2, args=()):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", **(extra_env or {}))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={nproc}",
           "--master-addr", "127.0.0.1", "--master-port", "29617"] + list(code) + list(args)
    return subprocess.run(cmd, capture_output=True, text=True, env=env, cwd=ROOT, timeout=600)


def test_time_is_max_over_ranks_and_value_counts_all_replicas(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(WORKER.format(root=ROOT, out=str(tmp_path)))
    r = _launch([str(w)])
    assert r.returncode == 0, r.stderr[-2000:]
    rows = [json.loads((tmp_path / f"rank{q}.json").read_text()) for q in range(2)]
    assert sorted(x["rank"] for x in rows) == [0, 1]
    for x in rows:
        assert x["t"] == pytest.approx(1.5)            # the slowest replica's time on every rank
        assert x["value"] == pytest.approx(2 * 10 / 1.5)  # both replicas' iterations over that time


def test_reference_arm_prints_once_under_torchrun():
    """`bench.py --impl reference` launched like the driver does for N = 2: rank 0 prints the line, rank 1 exits 0."""
    r = _launch([os.path.join(ROOT, "bench.py")], args=["--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                                                        "--workload", "C1"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
