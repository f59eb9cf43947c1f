"""Host-side measurement plumbing: clock parsing and the N>1 rank reduction (gloo, world size 2)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2601_19714_b200 import benchutil as bu


def test_parse_clock_lines():
    lines = ["1965, 1965, 180.0, Not Active, Not Active, Not Active, Not Active",
             "1500, 1965, 900.5, Not Active, Not Active, Not Active, Active",
             "1320, 1965, 1001.0, Not Active, Not Active, Not Active, Active",
             "garbage"]
    c = bu.parse_clock_lines(lines)
    assert c["sm_max_mhz"] == 1965 and c["reasons"] == ["sw_power_cap"]
    assert c["sm_mhz"] == 1410.0          # median of the samples under load (900 W, 1001 W)
    assert bu.parse_clock_lines([])["sm_mhz"] is None
    hot = bu.parse_clock_lines(["1000, 1965, 500, Active, Active, Not Active, Not Active"])
    assert "hw_slowdown" in hot["reasons"] and "hw_thermal_slowdown" in hot["reasons"]


def test_measured_peaks_fallback(tmp_path):
    p = bu.measured_peaks(str(tmp_path))
    assert p["hbm_gbs"] == 6650.0 and "fallback" in p["source"]
    (tmp_path / "MEASURED_PEAKS.json").write_text('{"hbm_gbs": 6455.3}')
    p = bu.measured_peaks(str(tmp_path))
    assert p["hbm_gbs"] == 6455.3 and "measured" in p["source"]


def test_single_process_identity():
    assert bu.dist_max(3.5) == 3.5 and bu.dist_sum(2.0) == 2.0
    a = bu.aggregate_replicas(1000.0, 10.0)
    assert a["units"] == 1000.0 and a["ms"] == 10.0 and abs(a["per_s"] - 1e5) < 1e-6


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    assert bu.dist_env() == (rank, rank, world)
    bu.dist_barrier()
    # replicas: each rank processed 1000 units; rank 1 was slower
    a = bu.aggregate_replicas(1000.0, 10.0 + 5.0 * rank)
    q.put((rank, a["units"], a["ms"], a["per_s"], bu.dist_max(float(rank))))
    dist.destroy_process_group()


def test_replica_aggregation_world2_gloo():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, units, ms, per_s, mx in res:
        assert units == 2000.0 and ms == 15.0 and abs(per_s - 2000.0 / 0.015) < 1e-6 and mx == 1.0
