#!/usr/bin/env python
"""bench.py -- one JSON line for the w-stacking hot path (contract: DESIGN.md section 9).

A "step" is one pass of the whole hot path (a0..a6: w range, index/key, radix sort, zero,
grid, w-plane FFT, w-correction + plane sum, taper) over one batch of synthetic visibilities,
through the C ABI (rick_image).

Headline workload at N=1: BASELINE.json configs[2] (LOFAR-like, 8192^2 x 64 planes fp64, 68.7 GB
resident: the largest fp64 single-GPU config and the closest to the paper's own 8192^2 x 32 test,
PAPER.md:216).  The same line carries a `configs` array with one record for each of configs[1]
(MeerKAT-like), configs[3] (large-pixel fp32, streamed plane batches) and configs[4] (128-channel
cube): north_star asks for MeerKAT- AND LOFAR-shaped throughput.  With --gpus N every rank images
its own replica of the headline workload ("replicas only").

  python bench.py                               # N=1: headline + the other configs, oracle baseline
  python bench.py --config 2 --only             # one config only
  python bench.py --impl reference ...          # the CPU oracle on a bounded sample, same metric

Byte model (every figure is per step; DESIGN.md section 6 derives it):
  dense_equiv = 3 * stack + image      what a4..a6 move when nothing is pruned and the column pass is
                                       fused with the correction -- for comparison only
  moved       = the bytes the pruned method has to move: the row pass reads the occupied B x B tiles and
                writes the occupied rows (counts from rick_get_stats: occ_tiles, occ_rows), the column
                pass reads what its kernel reads (the whole stack, or the occupied rows) -- every
                fraction of the HBM peak is quoted on `moved`, per launch.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "Mvis/s imaged end to end (rick_image: sort+grid, w-plane FFT, w-correct+sum, taper)"
WORKLOADS = {
    2: "configs[1] MeerKAT-like: 64 ant, 2016 bl x 512 t x 16 ch = 16515072 vis (c64), 4096^2 grid, 32 w-planes, S=7, fp64 grid",
    3: "configs[2] LOFAR-like: 60 stations, 1770 bl x 1024 t x 8 ch = 14499840 vis (c64), 8192^2 grid, 64 w-planes, S=7, fp64 grid (68.7 GB stack resident)",
    4: "configs[3] large-pixel: 2016 bl x 2048 t x 16 ch = 66060288 vis (c64), 16384^2 grid, 32 w-planes in streamed batches of 8, S=7, fp32 grid",
    5: "configs[4] cube: 2016 bl x 256 t x 128 ch = 66060288 vis (c64), 128 images of 4096^2 x 16 w-planes, S=7, fp64 grid",
}
HEADLINE = 3
CPU_FRAC = {2: 4, 3: 8, 4: 16, 5: 32}      # oracle sample: 1/frac of every stage (about 10-30 s of host work)
SM_CLOCK_GHZ = 1.965                       # clocks.max.sm of this pool's B200 (B200_PROFILING.md)
N_SM = 148


def make_workload(cfg, args, device):
    from paper_2601_19714_b200 import synth
    kw = {}
    if args.small:
        kw = dict(n_times=16, n=1024 if cfg != 3 else 2048, n_wplanes=8)
        if cfg == 5:
            kw["n_chan"] = 8
    return synth.make_config(cfg, device=device, **kw)


def cpu_sample(wl, frac):
    """Bounded sample for the oracle: every `frac`-th row and N_w/frac planes at the full grid size
    (1/frac of every stage); for a cube every frac-th channel with all its planes."""
    import dataclasses
    import numpy as np
    out = dataclasses.replace(wl)
    if wl.cube:
        out.freq_hz = wl.freq_hz[::frac].copy()
        out.vis = np.ascontiguousarray(wl.vis[:, ::frac])
        out.weights = None if wl.weights is None else np.ascontiguousarray(wl.weights[:, ::frac])
        return out, (f"channels c mod {frac} = 0 ({out.n_chan} of {wl.n_chan} images, all rows, all "
                     f"{wl.n_wplanes} w-planes each, full {wl.n}^2 grid): 1/{frac} of every stage")
    out.uvw_m = wl.uvw_m[::frac].copy()
    out.vis = wl.vis[::frac].copy()
    out.weights = None if wl.weights is None else wl.weights[::frac].copy()
    out.n_wplanes = max(1, wl.n_wplanes // frac)
    return out, (f"rows r mod {frac} = 0 ({out.n_vis} vis) and {out.n_wplanes} of {wl.n_wplanes} w-planes "
                 f"at the full {wl.n}^2 grid: 1/{frac} of every stage")


def run_oracle_sample(wl, frac):
    import oracle
    s, desc = cpu_sample(wl, frac)
    t0 = time.perf_counter()
    r = oracle.image(s.uvw_m, s.freq_hz, s.vis, s.weights, s.n, s.n_wplanes, s.support, s.pixel_rad,
                     cube=s.cube)
    dt = time.perf_counter() - t0
    return s, r, dt, desc


# --------------------------------------------------------------------------------------------------
def byte_model(wl, st, prof, steps):
    """Bytes (and FFT flops) every kernel class has to move per step -> {class: dict}.  `prof` is
    {class: (total_ms, launches)} over `steps` profiled steps; which column path ran is read off it."""
    N, S, B = wl.n, wl.support, 16
    E = 8 if wl.grid_prec == "f32" else 16
    P = int(st["n_planes"])                                   # planes of all images
    n_img = wl.n_chan if wl.cube else 1
    M = wl.n_vis
    stack = N * N * P * E
    img = N * N * 8 * n_img
    batch = wl.plane_batch or wl.n_wplanes
    n_batches = math.ceil(wl.n_wplanes / batch)
    rmw = (n_batches - 1) * 2 * img                           # image read + write of every batch but the first
    occ_rows, occ_tiles = int(st["occ_rows"]), int(st["occ_tiles"])
    vis_b = wl.vis.dtype.itemsize
    launched = lambda k: k in prof and prof[k][1] > 0
    fft_flops = lambda n_transforms: 5.0 * N * math.log2(N) * n_transforms
    m = {}
    m["index_key"] = dict(bytes=24 * wl.n_rows + 8 * M + (4 * M if wl.weights is not None else 0))
    m["radix_scatter"] = dict(bytes=16 * M * (prof["radix_scatter"][1] / steps if launched("radix_scatter") else 0))
    m["zero"] = dict(bytes=occ_tiles * B * B * E)             # lower bound: stale rows come on top
    m["grid"] = dict(bytes=M * (8 + vis_b + 16 + (4 if wl.weights is not None else 0)) + 2 * occ_tiles * B * B * E,
                     acc=2.0 * S * S * int(st["n_gridded"]))
    m["fft_rows"] = dict(bytes=occ_tiles * B * B * E + occ_rows * N * E, flops=fft_flops(occ_rows),
                         dense_bytes=2 * stack)
    fused = launched("fft_cols_wcorrect")
    sparse = fused and wl.grid_prec == "f32"
    if sparse:         # fp32 long columns: one fused pass that GATHERS the occupied rows only and accumulates a
        #                transposed image (read + written by every batch but the first); `taper` = transpose + a6
        m["fft_cols_wcorrect"] = dict(bytes=occ_rows * N * E + img * (2 * n_batches - 1),
                                      flops=fft_flops(N * P) + 8.0 * N * N * P, dense_bytes=stack + img, alu=True)
        m["taper"] = dict(bytes=2 * img)
    elif fused:        # single pass over the stack fused with a5 (+ a6): the planes are never written
        # (N = 8192: only the windows of N/32 rows that hold an occupied row are fetched)
        read = int(st["occ_windows"]) * (N // 32) * N * E if N == 8192 else stack
        m["fft_cols_wcorrect"] = dict(bytes=read + img + rmw, flops=fft_flops(N * P) + 8.0 * N * N * P,
                                      dense_bytes=stack + img)
    elif N >= 8192:    # two passes: A in place (reads occupied rows, writes every row), B fused with a5 (+ a6)
        m["fft_cols"] = dict(bytes=occ_rows * N * E + stack, flops=fft_flops(N * P) * (math.log2(N) - 4) / math.log2(N),
                             dense_bytes=2 * stack)
        m["wcorrect"] = dict(bytes=stack + img + rmw, flops=fft_flops(N * P) * 4 / math.log2(N) + 8.0 * N * N * P,
                             dense_bytes=stack + img)
    else:              # generic: in-place column pass, then the correction pass
        m["fft_cols"] = dict(bytes=2 * stack, flops=fft_flops(N * P), dense_bytes=2 * stack)
        m["wcorrect"] = dict(bytes=stack + img + rmw, flops=8.0 * N * N * P, dense_bytes=stack + img)
    return m, dict(stack=stack, image=img, dense_equiv=3 * stack + img, fused=fused)


def load_traffic(cfg):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu captures
    (profiles/r2_traffic.csv, written when a capture is summarised; profiles/r2_traffic.md says how): only valid
    for the kernels as they were when captured, so every row names the sha256 of the csrc tree it was taken at
    and rows of another tree are ignored."""
    import csv
    path = os.path.join(ROOT, "profiles", "r2_traffic.csv")
    from paper_2601_19714_b200 import benchutil as bu
    out = {}
    try:
        sha = bu.csrc_sha256(ROOT)
        with open(path) as f:
            for row in csv.DictReader(f):
                if row["csrc_sha256"] == sha and row["config"] == str(cfg):
                    out[row["kernel_class"]] = float(row["dram_bytes_per_launch"])
    except (OSError, KeyError, ValueError):
        return {}
    return out


def measure(cfg, args, rank, world, headline):
    """Time rick_image (device-resident inputs), per-kernel classes, the host-buffer entry and cuFFT on
    config `cfg`; returns the record (rank 0's view, times are max over ranks)."""
    import numpy as np
    import torch
    from paper_2601_19714_b200 import benchutil as bu
    from paper_2601_19714_b200 import rick

    wl = make_workload(cfg, args, "cuda")
    shard = None
    if world > 1:
        # strong scaling: this rank's share of the ONE problem.  Set-up (untimed, once per visibility set):
        # the per-plane histogram, the plane bounds, this rank's plan.
        import dataclasses
        from paper_2601_19714_b200 import sharded
        if wl.cube:
            cb = sharded.channel_bounds(wl.n_chan, world)
            c0, c1 = int(cb[rank]), max(int(cb[rank + 1]), int(cb[rank]) + 1)
            wl = dataclasses.replace(wl, freq_hz=wl.freq_hz[c0:c1].copy(), vis=np.ascontiguousarray(wl.vis[:, c0:c1]),
                                     weights=None if wl.weights is None else np.ascontiguousarray(wl.weights[:, c0:c1]))
            shard = {"kind": "channels", "bounds": cb.tolist()}
    if world > 1 and not wl.cube and world > wl.n_wplanes:       # the same on every rank: nobody enters a collective
        raise SystemExit(f"--gpus {world}: more ranks than w-planes ({wl.n_wplanes})")
    vis, uvw, wgt = rick.to_device(wl)
    if world > 1 and not wl.cube:
        sh = sharded.ShardedImager(dict(n=wl.n, n_wplanes=wl.n_wplanes, support=wl.support, pixel_rad=wl.pixel_rad,
                                        grid_prec=wl.grid_prec, plane_batch=wl.plane_batch), rank, world)
        bounds = sh.prepare(uvw, wl.freq_hz)
        shard = {"kind": "w-planes", "bounds": bounds.tolist(), "plane_cost_vis": sh.cost,
                 "hist_max": int(sh.hist.max()), "hist_min": int(sh.hist.min())}
        plan = sh.plan                      # (never None: every rank owns at least one plane when world <= N_w)
    else:
        plan = rick.plan_from_workload(wl)
    image = torch.empty((wl.n_chan, wl.n, wl.n) if wl.cube else (wl.n, wl.n), dtype=torch.float64, device="cuda")
    steps = args.steps if headline else max(1, min(args.steps, args.secondary_steps))
    warmup = max(args.warmup, 3) if headline else 2

    def step():
        plan.rick_image(vis, uvw, wgt, wl.freq_hz, image)
        if world > 1 and not wl.cube:
            sharded.reduce_image(image, dst=0)          # the one collective of the path: the N x N real image

    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    st = plan.rick_get_stats()
    n_gridded = st["n_gridded"]

    sampler = bu.ClockSampler(gpu_index=torch.cuda.current_device()).start()
    # ---- timed region: K steps, CUDA events on the launching stream, per-kernel profiling OFF
    l0 = st["n_launches"]
    bu.dist_barrier()
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(steps):
        step()
    ev1.record()
    torch.cuda.synchronize()
    bu.dist_barrier()
    ms_total = ev0.elapsed_time(ev1)
    launches = plan.rick_get_stats()["n_launches"] - l0
    n_vis_total = bu.dist_sum(wl.n_vis, "cuda") if (world > 1 and wl.cube) else wl.n_vis     # the whole problem
    ms_max = bu.dist_max(ms_total, "cuda")              # max over ranks
    ms_per_step = ms_max / steps
    value = n_vis_total * steps / (ms_max * 1e-3) / 1e6

    # ---- second loop: the library brackets every launch with CUDA events on the stream it launches on
    # (read back after every step: the per-kernel figure is the MEDIAN over the profiled steps -- a single disturbed
    # step, seen on this pool when the clock sampler's nvidia-smi starts up under the loop, does not move it; the
    # per-step values of the larger kernels are kept in stages.kernel_ms_steps)
    psteps = max(1, min(steps, 5))
    plan.rick_profile(True)
    per_step, prev = [], {}
    for _ in range(psteps):
        step()
        cur = plan.rick_profile_read()
        per_step.append({k: v[0] - prev.get(k, (0.0, 0))[0] for k, v in cur.items() if v[1]})
        prev = cur
    prof = cur
    plan.rick_profile(False)
    import statistics
    kms = {k: statistics.median(d.get(k, 0.0) for d in per_step) for k, v in prof.items() if v[1]}
    prof_step_ms = sum(kms.values())

    model, sizes = byte_model(wl, st, prof, psteps)
    peaks = bu.measured_peaks(ROOT)
    traffic = load_traffic(cfg)
    f32 = wl.grid_prec == "f32"
    alu_peak_tflops = N_SM * (128 if f32 else 64) * 2 * SM_CLOCK_GHZ / 1e3      # FMA lanes x 2 flop x clock
    rooflines = []
    for k, ms in sorted(kms.items(), key=lambda kv: -kv[1]):
        share = ms / prof_step_ms
        if (share < 0.05 and k != "grid") or k not in model:      # (the gridder always: north_star asks for its fraction)
            continue
        n_l = prof[k][1] / psteps
        mk = model[k]
        if k == "grid":
            # not a contraction, not HBM-bound: shared-memory accumulate model.  One 128 B/clk port per SM
            # serves 16 fp64 reads OR writes per clock; a read-modify-write is two accesses -> 8 RMW/clk/SM
            # (16 for the fp32 grid).  `achieved` counts the 2 S^2 scalar accumulations Eq. 3 asks for per
            # visibility; run accumulation in registers (reading R22) does fewer tile updates than that.
            peak = N_SM * SM_CLOCK_GHZ * (16.0 if f32 else 8.0)
            ach = mk["acc"] / (ms * 1e-3) / 1e9
            rooflines.append({"kernel": k, "bound": "alu", "model": "shared-memory read-modify-write: 8 fp64 (16 fp32) per clk per SM",
                              "achieved": ach, "peak": peak, "unit": "Gacc/s", "frac": ach / peak,
                              "hbm_gb_s_moved": mk["bytes"] / (ms * 1e-3) / 1e9, "gvis_s": n_gridded / (ms * 1e-3) / 1e9,
                              "traffic": traffic.get(k), "avg_launch_ms": ms / n_l, "launches_per_step": n_l,
                              "share_of_step": share})
            continue
        ach = mk["bytes"] / (ms * 1e-3) / 1e9
        r = {"kernel": k, "bound": "hbm", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s",
             "frac": ach / peaks["hbm_gbs"], "traffic": traffic.get(k), "peak_source": peaks["source"],
             "avg_launch_ms": ms / n_l, "launches_per_step": n_l,
             "algorithmic_bytes_per_launch": mk["bytes"] / n_l, "share_of_step": share}
        if "dense_bytes" in mk:
            r["dense_equiv_gb_s"] = mk["dense_bytes"] / (ms * 1e-3) / 1e9
        if "flops" in mk:      # secondary ceiling: the FFT's own arithmetic on the plain FMA pipe
            r["fft_tflops"] = mk["flops"] / (ms * 1e-3) / 1e12
            r["fft_frac_of_fma_peak"] = r["fft_tflops"] / alu_peak_tflops
        t_hbm = mk["bytes"] / (peaks["hbm_gbs"] * 1e9)
        t_alu = mk["flops"] / (alu_peak_tflops * 1e12) if "flops" in mk else 0.0
        if mk.get("alu") or t_alu > t_hbm:
            # The roof is the lower of the two at the kernel's arithmetic intensity.  A kernel that skips the known-zero
            # part of the stack (the occupied rows of the fp32 pass, the occupied windows of the N = 8192 fp64 pass) moves
            # so few bytes that its arithmetic floor (5 N log2 N flop per transform + the Horner step against lanes x
            # 2 flop x clock) lies above its HBM floor: its roofline is the arithmetic one; the HBM
            # figures stay beside it.
            r.update({"bound": "alu", "hbm_gb_s_moved": r["achieved"], "hbm_frac": r["frac"],
                      "achieved": r["fft_tflops"], "peak": alu_peak_tflops, "unit": "TFLOP/s",
                      "frac": r["fft_frac_of_fma_peak"],
                      "peak_source": "148 SMs x %d %s lanes x 2 flop x 1.965 GHz" % (128 if f32 else 64, "fp32" if f32 else "fp64"),
                      "floor_ms": {"hbm": round(t_hbm * 1e3, 3), "alu": round(t_alu * 1e3, 3)}})
        rooflines.append(r)

    def ms_of(*names):
        return sum(kms.get(n, 0.0) for n in names)
    a46 = ("fft_rows", "fft_cols", "wcorrect", "taper", "fft_cols_wcorrect")
    t_a46 = ms_of(*a46)
    moved_a46 = sum(model[k]["bytes"] for k in a46 if k in model and k in kms)
    t_sortgrid = ms_of("reset", "wrange", "index_key", "radix_hist", "scan", "radix_scatter", "plane_starts",
                       "zero", "grid", "row_occupancy")
    stages = {
        "grid_mvis_s_a0_a3": n_gridded / (t_sortgrid * 1e-3) / 1e6 if t_sortgrid else None,
        "grid_kernel_mvis_s": n_gridded / (ms_of("grid") * 1e-3) / 1e6 if ms_of("grid") else None,
        "fft_plus_wcorrect_ms": t_a46,
        # the fraction of the HBM peak is quoted on MOVED bytes only; dense_equiv is for comparison with
        # SURVEY.md's table (it credits the pruned row pass with bytes it does not move)
        "fft_plus_wcorrect_moved_gb_s": moved_a46 / (t_a46 * 1e-3) / 1e9 if t_a46 else None,
        "fft_plus_wcorrect_frac_of_measured_peak": moved_a46 / (t_a46 * 1e-3) / 1e9 / peaks["hbm_gbs"] if t_a46 else None,
        "fft_plus_wcorrect_frac_of_8tbs": moved_a46 / (t_a46 * 1e-3) / 1e9 / 8000.0 if t_a46 else None,
        "fft_plus_wcorrect_dense_equiv_gb_s": sizes["dense_equiv"] / (t_a46 * 1e-3) / 1e9 if t_a46 else None,
        "fused_cols_wcorrect": sizes["fused"],
        "occupied_rows_frac": st["occ_rows"] / (st["n_planes"] * wl.n),
        "occupied_tiles_frac": st["occ_tiles"] / (st["n_planes"] * (wl.n // 16) ** 2),
        "image_s": ms_per_step * 1e-3,
        "kernel_ms_per_step": {k: round(v, 4) for k, v in kms.items()},
        "kernel_ms_steps": {k: [round(d.get(k, 0.0), 3) for d in per_step] for k, v in kms.items() if v >= 0.05 * prof_step_ms},
        "profiled_step_ms": prof_step_ms,
    }

    # ---- end to end through the public host-buffer call: pinned host inputs, image read back
    hv = torch.from_numpy(np.ascontiguousarray(wl.vis)).pin_memory()
    hu = torch.from_numpy(np.ascontiguousarray(wl.uvw_m)).pin_memory()
    hw = None if wl.weights is None else torch.from_numpy(wl.weights).pin_memory()
    nimg = wl.n_chan if wl.cube else 1
    hout = torch.empty((nimg, wl.n, wl.n), dtype=torch.float64).pin_memory()
    plan.rick_image_host(hv, hu, hw, wl.freq_hz, hout)          # warm (allocates staging)
    k_e2e = max(1, min(steps, 5 if not wl.cube else 2))
    bu.dist_barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(k_e2e):
        plan.rick_image_host(hv, hu, hw, wl.freq_hz, hout)
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    if world > 1 and not wl.cube:
        # end to end over the shards: every rank copies the inputs from pinned host memory, images its planes,
        # the images are reduced, rank 0 reads the result back
        t0 = time.perf_counter()
        for _ in range(k_e2e):
            dv, du = hv.to("cuda", non_blocking=True), hu.to("cuda", non_blocking=True)
            dw = None if hw is None else hw.to("cuda", non_blocking=True)
            plan.rick_image(dv, du, dw, wl.freq_hz, image)
            sharded.reduce_image(image, dst=0)
            if rank == 0:
                hout[0].copy_(image, non_blocking=True)
            torch.cuda.synchronize()
        e2e_ms = (time.perf_counter() - t0) * 1e3
    e2e_max = bu.dist_max(e2e_ms, "cuda")
    e2e = {"ms": e2e_max, "per_s": n_vis_total * k_e2e / (e2e_max * 1e-3)}
    h2d = hv.numel() * hv.element_size() + hu.numel() * 8 + (0 if hw is None else hw.numel() * 4)
    # out-of-core visibilities (rick_image_stream_host): the same host buffers in 8 chunks of rows
    if headline and world == 1 and not wl.cube and not wl.plane_batch:
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
    plan.destroy()
    del plan, image, vis, uvw, wgt, hv, hu, hout
    torch.cuda.empty_cache()

    # ---- cuFFT on a dense stack of the same shape (GPU-side baseline for a4 only; the paper's own GPU FFT is
    # cuFFT under HeFFTe).  bench.py only: never linked into librick_b200.so.
    if not args.no_cufft and rank == 0:
        try:
            plane_bytes = wl.n * wl.n * (8 if f32 else 16)
            n_pl = sizes["stack"] // plane_bytes
            nb = int(max(1, min(n_pl, (16 << 30) // plane_bytes)))
            t = bu.time_cufft_2d(wl.n, nb, double=not f32, reps=3)
            stages["cufft"] = {"ms_per_stack": t * n_pl / nb, "planes_timed": nb, "planes": n_pl,
                               "dense_gb_s": 4 * plane_bytes * nb / (t * 1e-3) / 1e9,
                               "type": "C2C" if f32 else "Z2Z", "in_place": True,
                               "ours_a4_ms": ms_of("fft_rows", "fft_cols") if not sizes["fused"] else None,
                               "ours_a4_a5_a6_ms": t_a46,
                               "ratio_cufft_a4_over_ours_a4_a6": (t * n_pl / nb) / t_a46 if t_a46 else None}
        except Exception as ex:      # a missing library is reported, never silently skipped
            stages["cufft"] = {"unavailable": repr(ex)}
        torch.cuda.empty_cache()

    dom = rooflines[0] if rooflines else None
    rec = {"workload": WORKLOADS[cfg] if not args.small else wl.name + " (small debug)",
           "value": value, "unit": "Mvis/s", "steps": steps, "warmup": warmup, "ms_per_step": ms_per_step,
           "dtype": "f32" if f32 else "f64",
           "n_vis": wl.n_vis, "grid": wl.n, "w_planes": wl.n_wplanes, "support": wl.support,
           "l2": "inputs larger than L2 (stack %.2f GB resident, visibilities %.0f MB); no flush needed"
                 % (min(sizes["stack"], plan_resident_bytes(wl)) / 1e9, h2d / 1e6),
           "clocks": clocks,
           "e2e": {"value": e2e["per_s"] / 1e6, "unit": "Mvis/s", "h2d_bytes_per_step": h2d,
                   "d2h_bytes_per_step": nimg * wl.n * wl.n * 8, "ms_per_step": e2e["ms"] / k_e2e, "steps": k_e2e},
           "gpu_launches": int(launches), "roofline": dom, "rooflines": rooflines, "stages": stages, "shard": shard,
           "n_vis_total": int(n_vis_total)}
    return rec, wl


def plan_resident_bytes(wl):
    E = 8 if wl.grid_prec == "f32" else 16
    batch = wl.plane_batch or wl.n_wplanes
    per_img = wl.n * wl.n * E * batch
    if wl.cube and not wl.plane_batch:
        return per_img * max(1, min(8, int(48e9 // per_img)))
    return per_img


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=HEADLINE, help="headline config 2..5 (SURVEY numbering: configs[k-1])")
    ap.add_argument("--only", action="store_true", help="headline config only (no `configs` array)")
    ap.add_argument("--secondary-steps", type=int, default=3, help="timed steps of the non-headline configs")
    ap.add_argument("--small", action="store_true", help="scaled-down workloads (debug only)")
    ap.add_argument("--cpu-frac", type=int, default=0, help="oracle sample: 1/frac of the workload (0: per config)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cufft", action="store_true")
    args = ap.parse_args()
    cfg = args.config
    frac = args.cpu_frac or CPU_FRAC[cfg]

    from paper_2601_19714_b200 import benchutil as bu
    rank, local_rank, world = bu.dist_env()

    # ------------------------------------------------------------------ reference arm = oracle
    if args.impl == "reference":
        if rank != 0:
            return 0
        import torch
        import oracle
        dev = "cuda" if torch.cuda.is_available() else "cpu"
        wl = make_workload(cfg, args, dev)
        for _ in range(min(args.warmup, 1)):
            run_oracle_sample(wl, frac * 4)
        times = []
        for _ in range(args.steps):
            s, r, dt, sample = run_oracle_sample(wl, frac)
            times.append(dt)
        ms = 1e3 * sum(times) / len(times)
        val = s.n_vis / (ms * 1e-3) / 1e6
        line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "Mvis/s", "n_gpus": args.gpus,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": WORKLOADS[cfg] if not args.small else "small debug", "sample": sample},
                "cpu_baseline": {"value": val, "unit": "Mvis/s", "cores": oracle.num_threads(),
                                 "kind": "oracle", "sample": sample},
                "e2e": {"value": val, "unit": "Mvis/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                "gpu_launches": 0}
        print(json.dumps(line))
        return 0

    # ------------------------------------------------------------------ our arm
    import torch
    import torch.distributed as dist
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    from paper_2601_19714_b200 import build
    if rank == 0:
        build.build()
    bu.dist_barrier()

    rec, wl = measure(cfg, args, rank, world, headline=True)

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        s, r, dt, sample = run_oracle_sample(wl, frac)
        cpu_baseline = {"value": s.n_vis / dt / 1e6, "unit": "Mvis/s", "cores": oracle.num_threads(),
                        "kind": "oracle", "seconds": dt, "sample": sample, "stage_seconds": r["timings"]}
    del wl

    others = []
    if world == 1 and not args.only:
        for c in (2, 3, 4, 5):
            if c == cfg:
                continue
            r2, w2 = measure(c, args, rank, world, headline=False)
            del w2
            others.append(r2)

    if rank == 0:
        line = {"metric": METRIC, "value": rec["value"], "unit": "Mvis/s", "n_gpus": world, "steps": rec["steps"],
                "warmup": rec["warmup"], "ms_per_step": rec["ms_per_step"], "higher_is_better": True,
                "scaling": "strong" if world > 1 else "weak", "vs_baseline": None, "dtype": rec["dtype"], "data": "synthetic",
                "config": {"workload": rec["workload"], "n_vis": rec["n_vis_total"], "grid": rec["grid"],
                           "w_planes": rec["w_planes"], "support": rec["support"],
                           "parallelism": (f"{rec['shard']['kind']} sharded over {world} GPUs, one reduction of the image"
                                           if world > 1 else "single GPU"),
                           "shard": rec["shard"], "l2": rec["l2"]},
                "clocks": rec["clocks"], "e2e": rec["e2e"], "gpu_launches": rec["gpu_launches"],
                "roofline": rec["roofline"], "rooflines": rec["rooflines"], "cpu_baseline": cpu_baseline,
                "stages": rec["stages"], "configs": others}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
