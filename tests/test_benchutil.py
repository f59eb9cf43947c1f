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


def test_byte_model_counts_what_the_pruned_method_moves():
    """bench.py's byte model on hand-made counts: the row pass is charged the occupied tiles it reads and the
    occupied rows it writes; the fused column pass the stack once -- at N = 8192 fp64 only the occupied 256-row
    windows --, plus the image (and its read-modify-write for every plane batch but the first)."""
    import types
    import numpy as np
    import bench
    def wl(n, nw, prec, batch=0):
        return types.SimpleNamespace(n=n, support=7, n_wplanes=nw, n_chan=4, n_rows=1000, n_vis=4000, cube=0,
                                     grid_prec=prec, plane_batch=batch, weights=None, vis=np.zeros(1, np.complex64))
    # N = 8192 fp64, 2 planes: 10 occupied windows of 64, 3000 occupied rows, 500 occupied tiles
    st = dict(n_planes=2, occ_rows=3000, occ_tiles=500, occ_windows=10, n_gridded=3900)
    prof = {"fft_cols_wcorrect": (1.0, 1), "fft_rows": (1.0, 1), "radix_scatter": (1.0, 4)}
    m, sizes = bench.byte_model(wl(8192, 2, "f64"), st, prof, 1)
    E, N = 16, 8192
    assert m["fft_rows"]["bytes"] == 500 * 16 * 16 * E + 3000 * N * E
    assert m["fft_cols_wcorrect"]["bytes"] == 10 * 256 * N * E + N * N * 8
    assert m["fft_cols_wcorrect"]["dense_bytes"] == N * N * 2 * E + N * N * 8 == sizes["stack"] + sizes["image"]
    assert m["radix_scatter"]["bytes"] == 16 * 4000 * 4
    # N = 4096 fp64: the whole stack, whatever the windows say
    st4 = dict(st, occ_windows=1)
    m4, _ = bench.byte_model(wl(4096, 2, "f64"), st4, prof, 1)
    assert m4["fft_cols_wcorrect"]["bytes"] == 4096 * 4096 * 2 * 16 + 4096 * 4096 * 8
    # fp32 sparse fused pass in 2 plane batches: occupied rows gathered, transposed image written, then read + written
    st32 = dict(n_planes=4, occ_rows=5000, occ_tiles=700, occ_windows=0, n_gridded=3900)
    m32, _ = bench.byte_model(wl(16384, 4, "f32", batch=2), st32, prof, 1)
    assert m32["fft_cols_wcorrect"]["bytes"] == 5000 * 16384 * 8 + 16384 * 16384 * 8 * 3 and m32["fft_cols_wcorrect"]["alu"]
