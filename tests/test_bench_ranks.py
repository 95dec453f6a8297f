"""The N > 1 path of bench.py is "replicas only": no data-path collective, rank r
works on its own 64 events, the reported time is the maximum over ranks.  Covered here with a
world_size-2 gloo group on CPU; the reference arm must print on rank 0 only."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, sys.argv[1])
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
mine = 10.0 + 5.0 * rank                                   # this rank's "timed region", ms
slowest = bench.max_over_ranks(mine, dist, torch.device("cpu"))
seeds = list(range(bench.rank_seed0(rank), bench.rank_seed0(rank) + bench.N_EVENTS))
gathered = [None] * world
dist.all_gather_object(gathered, seeds)
dist.barrier()
if rank == 0:
    print(json.dumps({"slowest": slowest, "value": bench.whole_job_events_per_s(world, 3, slowest),
                      "seeds": gathered, "world": world}))
dist.destroy_process_group()
"""


def test_replicas_shard_by_seed_and_time_is_max_over_ranks(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                        "--master-addr", "127.0.0.1", "--master-port", "29631", str(w), ROOT],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    line = [ln for ln in r.stdout.splitlines() if ln.startswith("{")][-1]
    d = json.loads(line)
    assert d["world"] == 2 and d["slowest"] == 15.0                       # max over ranks, not mean or rank 0's
    assert d["value"] == pytest.approx(2 * 64 * 3 / 15e-3)                # whole-job events / slowest time
    a, b = d["seeds"]
    assert a == list(range(0, 64)) and b == list(range(64, 128))         # disjoint events per replica


def test_reference_arm_prints_on_rank_0_only():
    """--impl reference under torchrun: rank 0 alone runs the oracle and prints; other ranks exit 0 silently."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0"], capture_output=True, text=True, env=env, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_reference_arm_line(tmp_path):
    """One JSON line with the keys the contract names; the value is the oracle's own events/s."""
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    d = json.loads(r.stdout.strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["unit"] == "events/s" and d["value"] > 0 and d["higher_is_better"]
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["config"]["workload"].startswith("BASELINE.json configs[2]")
