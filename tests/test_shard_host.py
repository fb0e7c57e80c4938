"""Host side of NEXT-4 (paper_1912_10192_b200/shard.py) on CPU: the contiguous x1 partition, the neighbour ring, and the
N > 1 reduction over a world_size-2 gloo group (the MAX of the Courant maxima every rank contributes, PAPER.md:93 fn. 2)."""
import os
import socket
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

from paper_1912_10192_b200 import shard

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_partition_covers_the_grid_in_contiguous_ranges_of_at_least_three_zones():
    for n1 in (9, 32, 40, 256, 257, 1000):
        for parts in (1, 2, 3, 8):
            if n1 < 3 * parts:
                continue
            r = shard.partition_x1(n1, parts)
            assert len(r) == parts and r[0][0] == 0 and sum(n for _, n in r) == n1
            assert all(r[q][0] + r[q][1] == r[q + 1][0] for q in range(parts - 1))
            assert min(n for _, n in r) >= 3
            assert max(n for _, n in r) - min(n for _, n in r) <= 1          # uniform cost: balanced to one plane
    with pytest.raises(ValueError):
        shard.partition_x1(8, 3)
    with pytest.raises(ValueError):
        shard.partition_x1(32, 2, cost=np.zeros(32))


def test_partition_by_cost_balances_the_cost_not_the_zone_count():
    cost = np.r_[np.full(64, 4.0), np.full(192, 1.0)]        # the inner quarter of the planes costs four times as much
    r = shard.partition_x1(256, 4, cost)
    w = [cost[lo:lo + n].sum() for lo, n in r]
    assert max(w) - min(w) <= 4.0                              # to one (expensive) plane
    assert r[0][1] < r[-1][1]
    # every cut is the plane nearest its target: moving any cut by one plane does not lower the largest share
    cuts = [lo for lo, _ in r[1:]]
    for q, c in enumerate(cuts):
        for dc in (-1, 1):
            cc = cuts[:q] + [c + dc] + cuts[q + 1:]
            edges = [0] + cc + [256]
            w2 = [cost[edges[t]:edges[t + 1]].sum() for t in range(4)]
            assert max(w2) >= max(w) - 1e-12


def test_neighbour_ring():
    assert [shard.neighbours(r, 3, False) for r in range(3)] == [(None, 1), (0, 2), (1, None)]
    assert [shard.neighbours(r, 3, True) for r in range(3)] == [(2, 1), (0, 2), (1, 0)]
    assert [shard.neighbours(r, 2, True) for r in range(2)] == [(1, 1), (0, 0)]     # two slabs: neighbours on both sides
    assert shard.neighbours(0, 1, True) == (None, None)                             # one slab wraps onto itself


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    red = shard.Reducer()
    ct = torch.tensor([0.5, 0.25, 0.9] if rank == 0 else [0.7, 0.125, 0.3], dtype=torch.float64)
    red.max_(ct)
    fence = torch.zeros(1, dtype=torch.float64)
    red.max_(fence)
    out.put((rank, red.rank, red.world, red.on_stream, ct.tolist(), shard.partition_x1(32, world)[rank]))
    dist.barrier()
    dist.destroy_process_group()


def test_reduction_over_two_ranks_with_gloo():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, rr, world, on_stream, ct, part in res:
        assert rr == rank and world == 2 and not on_stream
        assert ct == [0.7, 0.25, 0.9]
        assert part == ((0, 16) if rank == 0 else (16, 16))
