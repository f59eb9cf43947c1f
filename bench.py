#!/usr/bin/env python
"""bench.py -- one JSON line for the w-stacking hot path (see the contract in DESIGN.md).

A "step" is one pass of the whole hot path (a0..a6: w range, index/key, radix sort, zero,
grid, w-plane FFT, w-correction + plane sum, taper) over one batch of synthetic visibilities,
through the C ABI (rick_image).  Workload at N=1: BASELINE.json configs[1] (MeerKAT-like,
4096^2 x 32 planes fp64, ~16.5M visibilities).  With --gpus N every rank images its own
replica (north_star: no multi-GPU path; "replicas only").

  python bench.py --gpus 1 --steps 10 --warmup 3
  python bench.py --impl reference ...     # the CPU oracle on a bounded sample, same metric
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "Mvis/s imaged end to end (rick_image: sort+grid, w-plane FFT, w-correct+sum, taper)"
WORKLOAD = "configs[1] MeerKAT-like: 64 ant, 2016 bl x 512 t x 16 ch = 16515072 vis (c64), 4096^2 grid, 32 w-planes, S=7, fp64 grid"


def make_workload(args, device):
    from paper_2601_19714_b200 import synth
    kw = {}
    if args.small:
        kw = dict(n_times=32, n=1024, n_wplanes=8)
    if args.grid:
        kw["n"] = args.grid          # e.g. --config 2 --grid 8192: the paper's 8192^2 x 32-plane shape (context only)
    return synth.make_config(args.config, device=device, **kw)


def cpu_sample(wl, frac):
    """Bounded sample for the oracle: every `frac`-th row and N_w/frac planes -> 1/frac of the
    work of every stage at the full grid size."""
    import dataclasses
    out = dataclasses.replace(wl)
    out.uvw_m = wl.uvw_m[::frac].copy()
    out.vis = wl.vis[::frac].copy()
    out.weights = None if wl.weights is None else wl.weights[::frac].copy()
    out.n_wplanes = max(1, wl.n_wplanes // frac)
    return out


def run_oracle_sample(wl, frac):
    import oracle
    s = cpu_sample(wl, frac)
    t0 = time.perf_counter()
    r = oracle.image(s.uvw_m, s.freq_hz, s.vis, s.weights, s.n, s.n_wplanes, s.support, s.pixel_rad,
                     cube=s.cube)
    dt = time.perf_counter() - t0
    return s, r, dt


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--small", action="store_true", help="scaled-down workload (debug only)")
    ap.add_argument("--grid", type=int, default=0, help="override the grid edge N of the config (context runs only)")
    ap.add_argument("--cpu-frac", type=int, default=4, help="oracle sample: 1/frac of the workload")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()

    from paper_2601_19714_b200 import benchutil as bu
    rank, local_rank, world = bu.dist_env()

    # ------------------------------------------------------------------ reference arm = oracle
    if args.impl == "reference":
        if rank != 0:
            return 0
        import torch
        import oracle
        dev = "cuda" if torch.cuda.is_available() else "cpu"
        wl = make_workload(args, dev)
        for _ in range(min(args.warmup, 1)):
            run_oracle_sample(wl, args.cpu_frac * 4)
        times = []
        for _ in range(args.steps):
            s, r, dt = run_oracle_sample(wl, args.cpu_frac)
            times.append(dt)
        ms = 1e3 * sum(times) / len(times)
        val = s.n_vis / (ms * 1e-3) / 1e6
        sample = (f"rows r mod {args.cpu_frac} = 0 ({s.n_vis} vis) and {s.n_wplanes} of {wl.n_wplanes} w-planes "
                  f"at the full {wl.n}^2 grid: 1/{args.cpu_frac} of every stage")
        line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "Mvis/s", "n_gpus": args.gpus,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": WORKLOAD if not args.small else "small debug", "sample": sample},
                "cpu_baseline": {"value": val, "unit": "Mvis/s", "cores": oracle.num_threads(),
                                 "kind": "oracle", "sample": sample},
                "e2e": {"value": val, "unit": "Mvis/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                "gpu_launches": 0}
        print(json.dumps(line))
        return 0

    # ------------------------------------------------------------------ our arm
    import numpy as np
    import torch
    import torch.distributed as dist
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    from paper_2601_19714_b200 import build, rick
    if rank == 0:
        build.build()
    bu.dist_barrier()

    wl = make_workload(args, "cuda")
    vis, uvw, wgt = rick.to_device(wl)
    plan = rick.plan_from_workload(wl)
    image = torch.empty((wl.n_chan, wl.n, wl.n) if wl.cube else (wl.n, wl.n), dtype=torch.float64, device="cuda")
    E = 8 if wl.grid_prec == "f32" else 16
    stack_bytes = wl.n * wl.n * wl.n_wplanes * E
    image_bytes = wl.n * wl.n * 8

    def step():
        plan.rick_image(vis, uvw, wgt, wl.freq_hz, image)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    n_gridded = plan.rick_get_stats()["n_gridded"]

    sampler = bu.ClockSampler(gpu_index=local_rank).start()
    # timed region: K steps, CUDA events on the launching stream, per-kernel events inside the library
    plan.rick_profile(True)
    l0 = plan.rick_get_stats()["n_launches"]
    bu.dist_barrier()
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(args.steps):
        step()
    ev1.record()
    torch.cuda.synchronize()
    bu.dist_barrier()
    ms_total = ev0.elapsed_time(ev1)
    prof = plan.rick_profile_read()
    plan.rick_profile(False)
    launches = plan.rick_get_stats()["n_launches"] - l0
    agg = bu.aggregate_replicas(wl.n_vis * args.steps, ms_total, device="cuda")
    ms_per_step = agg["ms"] / args.steps
    value = agg["per_s"] / 1e6

    # stage numbers (BASELINE.json's three-part metric), from the per-kernel events
    def ms_of(*names):
        return sum(prof[n][0] for n in names if n in prof) / args.steps
    fused = ms_of("fft_cols_wcorrect") > 0
    t_sortgrid = ms_of("reset", "wrange", "index_key", "radix_hist", "scan", "radix_scatter", "plane_starts",
                       "zero", "grid", "row_occupancy")
    stages = {
        "grid_mvis_s_a0_a3": n_gridded / (t_sortgrid * 1e-3) / 1e6 if t_sortgrid else None,
        "grid_kernel_mvis_s": n_gridded / (ms_of("grid") * 1e-3) / 1e6 if ms_of("grid") else None,
        # a4 + a5 + a6 move 3 x stack + image when the column pass is fused with the correction
        # (rows: read + write; columns+correction: read), else 5 x stack + image
        "fft_rows_gb_s": 2 * stack_bytes / (ms_of("fft_rows") * 1e-3) / 1e9 if ms_of("fft_rows") else None,
        "fft_plus_wcorrect_gb_s": ((3 if fused else 5) * stack_bytes + image_bytes) /
                                  (ms_of("fft_rows", "fft_cols", "wcorrect", "taper", "fft_cols_wcorrect") * 1e-3) / 1e9,
        "fft_plus_wcorrect_ms": ms_of("fft_rows", "fft_cols", "wcorrect", "taper", "fft_cols_wcorrect"),
        "fused_cols_wcorrect": fused,
        "image_s": ms_per_step * 1e-3,
        "kernel_ms_per_step": {k: round(v[0] / args.steps, 4) for k, v in prof.items() if v[1]},
    }

    # roofline of the dominant kernel (algorithmic bytes per launch: DESIGN.md "Kernels")
    peaks = bu.measured_peaks(ROOT)
    # BASELINE.json's "FFT + correction GB/s vs 8 TB/s": dense algorithmic bytes of a4..a6 over their time,
    # against the nominal 8 TB/s the metric names and against this pool's measured copy rate (the row pass
    # skips rows no visibility reaches, so the bytes actually moved are fewer: profiles/)
    stages["fft_plus_wcorrect_frac_of_8tbs"] = stages["fft_plus_wcorrect_gb_s"] / 8000.0
    stages["fft_plus_wcorrect_frac_of_measured_peak"] = stages["fft_plus_wcorrect_gb_s"] / peaks["hbm_gbs"]
    alg_bytes = {"fft_rows": 2 * stack_bytes, "fft_cols": 2 * stack_bytes, "zero": stack_bytes,
                 "wcorrect": stack_bytes + image_bytes, "fft_cols_wcorrect": stack_bytes + image_bytes}
    dom = max((k for k in prof if prof[k][1]), key=lambda k: prof[k][0])
    # dram__bytes_read.sum + dram__bytes_write.sum per launch, from profiles/r1f_ncu_full.md (configs[1] only;
    # the row pass transforms occupied rows only, so its traffic is below its dense algorithmic bytes)
    traffic_ncu = {}
    if args.config == 2 and not args.small and not args.grid:
        traffic_ncu = {"fft_rows": 4.629e9, "fft_cols_wcorrect": 8.925e9, "grid": 0.781e9}
    if dom in alg_bytes:
        avg_ms = prof[dom][0] / prof[dom][1]
        ach = alg_bytes[dom] / (avg_ms * 1e-3) / 1e9
        roofline = {"kernel": dom, "bound": "hbm", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                    "frac": ach / peaks["hbm_gbs"], "traffic": traffic_ncu.get(dom), "peak_source": peaks["source"],
                    "avg_launch_ms": avg_ms, "algorithmic_bytes_per_launch": alg_bytes[dom]}
    else:  # the gridder: shared-memory accumulate rate (DESIGN.md derives the peak)
        avg_ms = prof[dom][0] / prof[dom][1]
        S2 = wl.support * wl.support
        ach = n_gridded * S2 * 2 / (avg_ms * 1e-3) / 1e9            # G scalar accumulations / s
        peak = 148 * 1.965 * 16.0                                    # 16 fp64 RMW / clk / SM (128 B/clk smem)
        roofline = {"kernel": dom, "bound": "alu", "achieved": ach, "peak": peak, "unit": "Gacc/s",
                    "frac": ach / peak, "traffic": traffic_ncu.get(dom), "avg_launch_ms": avg_ms}
    roofline["share_of_step"] = prof[dom][0] / args.steps / ms_per_step

    # end to end through the public host-buffer call: pinned host inputs, image read back
    hv = torch.from_numpy(np.ascontiguousarray(wl.vis)).pin_memory()
    hu = torch.from_numpy(np.ascontiguousarray(wl.uvw_m)).pin_memory()
    hw = None if wl.weights is None else torch.from_numpy(wl.weights).pin_memory()
    nimg = wl.n_chan if wl.cube else 1
    hout = torch.empty((nimg, wl.n, wl.n), dtype=torch.float64).pin_memory()
    plan.rick_image_host(hv, hu, hw, wl.freq_hz, hout)          # warm (allocates staging)
    k_e2e = max(1, min(args.steps, 5))
    bu.dist_barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(k_e2e):
        plan.rick_image_host(hv, hu, hw, wl.freq_hz, hout)
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    e2e = bu.aggregate_replicas(wl.n_vis * k_e2e, e2e_ms, device="cuda")
    h2d = hv.numel() * hv.element_size() + hu.numel() * 8 + (0 if hw is None else hw.numel() * 4)
    # out-of-core visibilities (rick_image_stream_host): the same host buffers in 8 chunks of rows, the copy
    # of chunk c+1 under index + sort + gridding of chunk c (whole stack resident, cube = 0 only)
    if not wl.cube and not wl.plane_batch:
        rpc = (wl.n_rows + 7) // 8
        plan.rick_image_stream_host(hv, hu, hw, wl.freq_hz, hout[0], rpc)      # warm (grows the staging)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(k_e2e):
            plan.rick_image_stream_host(hv, hu, hw, wl.freq_hz, hout[0], rpc)
        torch.cuda.synchronize()
        st_ms = (time.perf_counter() - t0) * 1e3 / k_e2e
        stages["stream_host"] = {"ms_per_step": st_ms, "mvis_s": wl.n_vis / st_ms / 1e3, "rows_per_chunk": rpc, "chunks": 8}
    clocks = sampler.stop()

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        s, r, dt = run_oracle_sample(wl, args.cpu_frac)
        cpu_baseline = {"value": s.n_vis / dt / 1e6, "unit": "Mvis/s", "cores": oracle.num_threads(),
                        "kind": "oracle", "seconds": dt,
                        "sample": f"rows r mod {args.cpu_frac} = 0 ({s.n_vis} vis) and {s.n_wplanes} of "
                                  f"{wl.n_wplanes} w-planes at the full {wl.n}^2 grid: 1/{args.cpu_frac} of every stage",
                        "stage_seconds": r["timings"]}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": "Mvis/s", "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64" if wl.grid_prec == "f64" else "f32",
                "data": "synthetic",
                "config": {"workload": WORKLOAD if not args.small and not args.grid and args.config == 2 else wl.name,
                           "n_vis": wl.n_vis, "grid": wl.n, "w_planes": wl.n_wplanes, "support": wl.support,
                           "parallelism": f"replicas x{world}" if world > 1 else "single GPU",
                           "l2": "inputs larger than L2 (stack %.2f GB, visibilities %.0f MB); no flush needed"
                                 % (stack_bytes / 1e9, h2d / 1e6)},
                "clocks": clocks,
                "e2e": {"value": e2e["per_s"] / 1e6, "unit": "Mvis/s", "h2d_bytes_per_step": h2d,
                        "d2h_bytes_per_step": hout.numel() * 8, "ms_per_step": e2e["ms"] / k_e2e, "steps": k_e2e},
                "gpu_launches": int(launches),
                "roofline": roofline, "cpu_baseline": cpu_baseline, "stages": stages}
        print(json.dumps(line))
    plan.destroy()
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
