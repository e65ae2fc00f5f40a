"""Host-side logic of the N > 1 path on CPU (gloo, world_size 2): the per-rank template shards are
distinct and seeded, whole-job time is the MAX and work the SUM over ranks, and the reference arm
runs on rank 0 only.  The data path itself has no collective."""
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys, json
sys.path.insert(0, os.environ["SFT_ROOT"])
import torch, torch.distributed as dist
import bench
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
ms_dev, ms_host, pairs = bench.aggregate_over_ranks(10.0 + rank, 20.0 - rank, 1000 * (rank + 1), torch.device("cpu"), world)
w = bench.make_workload("config1", rank=rank)
w2 = bench.make_workload("config2", rank=rank, n_templates=8, n_sft=64)
print(json.dumps(dict(rank=rank, ms_dev=ms_dev, ms_host=ms_host, pairs=pairs, p2=float(w2.params[1:, 0].sum()))), flush=True)
dist.destroy_process_group()
'''


def _torchrun(code, nproc=2, extra_env=None):
    env = dict(os.environ, SFT_ROOT=ROOT, **(extra_env or {}))
    path = os.path.join(ROOT, "tests", "_worker_tmp.py")
    with open(path, "w") as f:
        f.write(code)
    try:
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(nproc),
               "--master-addr", "127.0.0.1", "--master-port", "29541", path]
        return subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=600)
    finally:
        os.remove(path)


def test_aggregation_and_shards_world2():
    import json
    r = _torchrun(WORKER)
    assert r.returncode == 0, r.stderr[-2000:]
    rows = sorted((json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")), key=lambda d: d["rank"])
    assert len(rows) == 2
    for d in rows:
        assert d["ms_dev"] == 11.0 and d["ms_host"] == 20.0 and d["pairs"] == 3000.0     # max, max, sum
    assert rows[0]["p2"] != rows[1]["p2"]                                                # distinct seeded shards


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
