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


def test_gpus_n_without_torchrun_spawns_n_ranks():
    """`python bench.py --gpus N` with no WORLD_SIZE in the environment must launch N ranks itself
    and the line must say n_gpus = N (launch plumbing only: the selftest arm joins a gloo group and does no work)."""
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "selftest", "--gpus", "2"],
                       env=env, capture_output=True, text=True, timeout=300)
    assert p.returncode == 0, p.stderr[-500:]
    lines = [ln for ln in p.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1 and json.loads(lines[0])["n_gpus"] == 2
    sys.path.insert(0, ROOT)
    import argparse
    import bench
    a = argparse.Namespace(gpus=4, steps=7, warmup=3, impl="ours", no_sweep=True, no_extras=False, no_cpu=True)
    cmd = bench.spawn_command(a, port=12345)
    assert cmd[1:4] == ["-m", "torch.distributed.run", "--nnodes=1"] and "--nproc-per-node" in cmd and "4" in cmd
    assert cmd[-2:] == ["--no-sweep", "--no-cpu"] and "127.0.0.1" in cmd


# ---- column-sharded propagator: host logic on gloo, world size 2 and 3 -------------
class _Res:
    def __init__(self, it):
        self.iterations = it


def _shard_worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    from paper_2411_08461_b200 import lqcd
    dist.init_process_group("gloo", rank=rank, world_size=world)
    g = torch.Generator().manual_seed(5)
    src = torch.complex(torch.randn(12, 2, 3, 4, generator=g, dtype=torch.float64),
                        torch.randn(12, 2, 3, 4, generator=g, dtype=torch.float64))
    lo, hi = lqcd.shard_columns(12, rank, world)
    calls = []

    def solve(blk):  # stands for the batched GPU solve: x = (2 + i) b, column c "takes" 10 + c iterations
        calls.append(blk.shape[0])
        return (2 + 1j) * blk, [_Res(10 + lo + k) for k in range(blk.shape[0])], (1 if rank == world - 1 else 0)

    x, iters, rc = lqcd.sharded_solve(src, solve)
    ok = bool(torch.equal(x, (2 + 1j) * src)) and iters == [10 + c for c in range(12)] and calls == [hi - lo]
    dist.barrier()
    dist.destroy_process_group()
    json.dump({"ok": ok, "rc": rc, "lo": lo, "hi": hi}, open(out % rank, "w"))


def test_sharded_solve_gloo(tmp_path):
    for world, port in ((2, 29641), (3, 29651)):
        out = str(tmp_path / ("w%d_" % world + "r%d.json"))
        mp.spawn(_shard_worker, args=(world, port, out), nprocs=world, join=True)
        got = [json.load(open(out % r)) for r in range(world)]
        assert all(d["ok"] for d in got)
        assert all(d["rc"] == 1 for d in got)                      # NOT_CONVERGED on one rank is everybody's status
        assert [d["lo"] for d in got] == [r * 12 // world for r in range(world)]
        assert got[-1]["hi"] == 12


def test_shard_columns_covers_every_column_once():
    sys.path.insert(0, ROOT)
    from paper_2411_08461_b200 import lqcd
    for n in (1, 5, 12, 16):
        for world in (1, 2, 3, 5, 8, 16):
            blocks = [lqcd.shard_columns(n, r, world) for r in range(world)]
            cover = [c for lo, hi in blocks for c in range(lo, hi)]
            assert cover == list(range(n))
            sizes = [hi - lo for lo, hi in blocks]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    x, iters, rc = lqcd.sharded_solve(torch.ones(3, 2), lambda b: (b * 3, [_Res(7)] * 3, -7))   # no process group
    assert torch.equal(x, torch.full((3, 2), 3.0)) and iters == [7, 7, 7] and rc == -7
