"""World-size-2 gloo test (CPU) of bench.py's multi-replica aggregation: value = sum of the units
all ranks processed / max over ranks of the time ("replicas only"), and of the
reference arm's rule that only rank 0 prints."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dt, sums = bench.reduce_over_ranks(dist, 0.1 * (rank + 1), [100.0 + rank, 7.0], "cpu")
    dist.barrier()
    dist.destroy_process_group()
    json.dump({"dt": dt, "sums": sums}, open(out % rank, "w"))


def test_reduce_over_ranks_gloo(tmp_path):
    out = str(tmp_path / "r%d.json")
    mp.spawn(_worker, args=(2, 29631, out), nprocs=2, join=True)
    for r in range(2):
        d = json.load(open(out % r))
        assert abs(d["dt"] - 0.2) < 1e-12          # max over ranks
        assert d["sums"] == [201.0, 14.0]          # whole-job totals


def test_single_process_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks(None, 0.5, [1.0, 2.0], "cpu") == (0.5, [1.0, 2.0])


def test_reference_arm_nonzero_rank_prints_nothing():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert p.returncode == 0 and p.stdout.strip() == ""
