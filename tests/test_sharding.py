"""Host logic of the multi-GPU path: the plane partition of the library
(rick_partition_planes: pure host arithmetic in librick_b200.so, no device needed) against brute force, and
the reduction plumbing of paper_2601_19714_b200/sharded.py in a world-size-2 gloo run on the CPU."""
import itertools
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2601_19714_b200 import rick, sharded


def _brute(hist, parts, cost):
    n = len(hist)
    c = np.asarray(hist, dtype=np.float64) + cost
    best = None
    for cuts in itertools.combinations(range(1, n), parts - 1):
        b = (0,) + cuts + (n,)
        m = max(c[b[i]:b[i + 1]].sum() for i in range(parts))
        best = m if best is None or m < best else best
    return best


def test_partition_matches_brute_force_and_covers_every_plane():
    rng = np.random.default_rng(7)
    for trial in range(40):
        n = int(rng.integers(1, 10))
        hist = (rng.pareto(0.7, n) * 1000).astype(np.int64)          # heavy-tailed, like the w distribution
        cost = float(rng.choice([0.0, 10.0, 5000.0]))
        for parts in range(1, n + 1):
            b = rick.rick_partition_planes(hist, parts, cost)
            assert b[0] == 0 and b[-1] == n and np.all(np.diff(b) >= 1)   # contiguous, every part non-empty
            got = max((hist[b[i]:b[i + 1]].sum() + cost * (b[i + 1] - b[i])) for i in range(parts))
            assert got <= _brute(hist, parts, cost) * (1 + 1e-9) + 1e-6


def test_partition_edge_cases():
    h = np.array([5, 0, 0, 7], np.int64)
    b = rick.rick_partition_planes(h, 6, 1.0)                            # more parts than planes: trailing parts empty
    assert list(b) == [0, 1, 2, 3, 4, 4, 4]
    assert list(rick.rick_partition_planes(h, 1, 0.0)) == [0, 4]
    assert list(rick.rick_partition_planes(np.zeros(8, np.int64), 4, 1.0)) == [0, 2, 4, 6, 8]   # equal planes
    with pytest.raises(rick.RickError):
        rick.rick_partition_planes(np.array([-1], np.int64), 1, 0.0)
    with pytest.raises(rick.RickError):
        rick.rick_partition_planes(h, 0, 0.0)
    # the cfg-2-like histogram: one plane with half of all visibilities ends up alone
    h2 = np.array([31, 100, 8_000_000, 500_000, 20, 10, 900_000, 4_000_000], np.int64)
    b2 = rick.rick_partition_planes(h2, 3, 1e6)
    costs = [h2[b2[i]:b2[i + 1]].sum() + 1e6 * (b2[i + 1] - b2[i]) for i in range(3)]
    assert max(costs) == 10_400_030.0 and list(sharded.channel_bounds(128, 3)) == [0, 42, 85, 128]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # both ranks derive the same bounds from the same histogram (no communication needed for them)
        hist = np.array([3, 50, 4000, 300, 2, 1, 900, 2500], np.int64)
        b = sharded.shard_bounds(hist, world, 100.0)
        # stand-in for the ranks' shares: plane z contributes (z + 1) * pattern; the reduction must give the sum
        n = 16
        pattern = torch.arange(n * n, dtype=torch.float64).reshape(n, n)
        share = torch.zeros(n, n, dtype=torch.float64)
        for z in range(int(b[rank]), int(b[rank + 1])):
            share += (z + 1) * pattern
        sharded.reduce_image(share, dst=0)
        ok = True
        if rank == 0:
            ok = torch.equal(share, pattern * sum(z + 1 for z in range(len(hist))))
        q.put((rank, list(map(int, b)), bool(ok)))
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo_bounds_and_reduction():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] == res[1][1] and res[0][1][0] == 0 and res[0][1][-1] == 8
    assert all(r[2] for r in res)
