"""The N > 1 path of bench.py on CPU: world_size 2 over gloo (replicas only — the ranks never
exchange field data; the only cross-rank step is the MAX over the ranks' device times)."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks([10.0 + rank, 7.0 - rank], world, "cpu")
    val = bench.aggregate_value(1000, world, ms[0], steps=2)
    dist.barrier()
    dist.destroy_process_group()
    json.dump({"ms": ms, "value": val}, open(os.path.join(out_dir, "r%d.json" % rank), "w"))


def test_max_over_ranks_and_aggregate_gloo_world2(tmp_path):
    port = 29500 + (os.getpid() % 2000)
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r = [json.load(open(tmp_path / ("r%d.json" % k))) for k in range(2)]
    assert r[0] == r[1]                       # every rank sees the same maxima
    assert r[0]["ms"] == [11.0, 7.0]          # slowest rank decides
    assert r[0]["value"] == 2 * 1000 * 2 / (11.0e-3) / 1e9   # whole-job units / max time


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([3.5, 1.0], 1) == [3.5, 1.0]


def test_reference_arm_other_ranks_exit_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert p.returncode == 0 and p.stdout.strip() == ""
