"""Host logic of the 4-D domain decomposition (paper_2411_08461_b200/dd.py): rank
grid with t fastest, neighbour table, seam weights, split / join of cb2 fields, and the exchange schedule run over a
world-size-2 gloo group (CPU tensors stand in for the packed faces)."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from paper_2411_08461_b200 import dd  # noqa: E402
from latt import coords  # noqa: E402


def test_rank_grid_runs_fastest_in_t():
    p = dd.Partition((8, 8, 16, 16), (1, 2, 2, 4))
    assert p.local == (8, 4, 8, 4) and p.size == 16
    assert [p.coords(r) for r in range(5)] == [(0, 0, 0, 0), (0, 0, 0, 1), (0, 0, 0, 2), (0, 0, 0, 3), (0, 0, 1, 0)]
    for r in range(p.size):
        assert p.rank(p.coords(r)) == r
        for mu in range(4):
            assert p.neighbour(p.neighbour(r, mu, +1), mu, -1) == r
    assert p.neighbour(3, 3, +1) == 0 and p.neighbour(0, 3, -1) == 3 and p.neighbour(0, 2, +1) == 4
    assert p.partitioned == [False, True, True, True] and p.local_t_boundary() == 1
    # the antiperiodic sign sits on the two hops across global t = Lt-1 | 0 only
    assert p.ghost_weight(3, 3, +1) == -1.0 and p.ghost_weight(0, 3, -1) == -1.0
    assert p.ghost_weight(0, 3, +1) == 1.0 and p.ghost_weight(3, 3, -1) == 1.0 and p.ghost_weight(3, 1, +1, ws=0.7) == 0.7
    with pytest.raises(ValueError):
        dd.Partition((8, 8, 8, 16), (1, 1, 1, 8))      # local extent 2
    assert dd.Partition((12, 8, 8, 16), (2, 1, 1, 1)).local[0] == 6
    with pytest.raises(ValueError):
        dd.Partition((12, 8, 8, 16), (4, 1, 1, 1))     # local extent 3


def test_every_face_sent_is_expected_by_its_receiver():
    for grid in ((1, 1, 1, 2), (1, 1, 2, 2), (2, 1, 1, 4), (2, 2, 2, 2)):
        p = dd.Partition((8, 8, 8, 16), grid)
        for r in range(p.size):
            sends, recvs = p.messages(r)
            assert len(sends) == len(recvs) == 2 * sum(p.partitioned)
            for mu, kind, peer, tag in sends:
                assert (mu, kind, r, tag) in p.messages(peer)[1]
            assert len({tag for _, _, _, tag in recvs}) == len(recvs)


def test_split_join_round_trip_and_parity():
    dims, grid = (8, 8, 8, 16), (2, 1, 2, 2)
    p = dd.Partition(dims, grid)
    x, y, z, t = coords(dims)
    f = (x + 100 * y + 10000 * z + 1000000 * t).astype(np.float64)[..., None]
    pieces = dd.split_field(p, f)
    assert np.array_equal(dd.join_field(p, pieces), f)
    lx, ly, lz, lt = coords(p.local)
    for r, piece in enumerate(pieces):
        ox, oy, oz, ot = p.origin(r)
        # slot (par, t, z, y, xh) of the local array holds the global site origin + local coordinates
        assert np.array_equal(piece[..., 0], (lx + ox) + 100 * (ly + oy) + 10000 * (lz + oz) + 1000000 * (lt + ot))


def _worker(rank, world, port, grid, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    p = dd.Partition((8, 8, 8, 16), grid)
    faces = {tag: (torch.full((5,), 1000.0 * rank + tag), peer) for mu, kind, peer, tag in p.messages(rank)[0]}
    got = dd.exchange(p, rank, faces)
    ok = True
    for mu, kind, peer, tag in p.messages(rank)[1]:
        ok = ok and bool((got[tag] == 1000.0 * peer + tag).all())
    # the reductions of a decomposed solve: one value per held sub-lattice, summed over all ranks
    D = dd.Decomposed(p, [rank], [None], [None], [None], [None], group=dist.group.WORLD)
    ok = ok and D.allsum([rank + 1 + 2j]) == 3 + 4j
    dist.barrier()
    dist.destroy_process_group()
    open(out % rank, "w").write("ok" if ok and len(got) == 2 * sum(p.partitioned) else "bad")


@pytest.mark.parametrize("grid,port", [((1, 1, 1, 2), 29641), ((1, 2, 1, 1), 29642)])
def test_exchange_schedule_world_size_2_gloo(grid, port, tmp_path):
    """Two ranks in one direction: both neighbours of a rank are the SAME rank, the forward and the backward ghost are
    told apart by their tags."""
    out = str(tmp_path / "r%d.txt")
    mp.spawn(_worker, args=(2, port, grid, out), nprocs=2, join=True)
    assert [open(out % r).read() for r in range(2)] == ["ok", "ok"]
