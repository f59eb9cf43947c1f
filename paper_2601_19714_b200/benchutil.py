"""Measurement plumbing for bench.py: clock sampling, rank reduction, peaks.  No method arithmetic."""
from __future__ import annotations

import json
import os
import statistics
import subprocess
import threading
from typing import Optional

_FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
           "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
           "clocks_event_reasons.sw_power_cap")


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons of one GPU while a timed region runs."""

    def __init__(self, gpu_index: int = 0, period_ms: int = 100):
        self.gpu_index, self.period_ms = gpu_index, period_ms
        self.proc: Optional[subprocess.Popen] = None
        self.lines = []
        self._t = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={_FIELDS}", "--format=csv,noheader,nounits",
                 "-lms", str(self.period_ms), "-i", str(self.gpu_index)],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return self
        self._t = threading.Thread(target=self._read, daemon=True)
        self._t.start()
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        return parse_clock_lines(self.lines)


def parse_clock_lines(lines) -> dict:
    sm, smax, power, reasons = [], [], [], set()
    names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
    for ln in lines:
        parts = [p.strip() for p in ln.split(",")]
        if len(parts) < 7:
            continue
        try:
            sm.append(float(parts[0]))
            smax.append(float(parts[1]))
            power.append(float(parts[2]))
        except ValueError:
            continue
        for name, val in zip(names, parts[3:7]):
            if val.lower().startswith("active"):
                reasons.add(name)
    if not sm:
        return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
    # "under load": samples whose power is above the midpoint of the observed range
    thr = (min(power) + max(power)) / 2.0
    loaded = [c for c, p in zip(sm, power) if p >= thr] or sm
    return {"sm_mhz": statistics.median(loaded), "sm_max_mhz": max(smax), "samples": len(sm),
            "power_w_max": max(power), "reasons": sorted(reasons)}


def measured_peaks(root: str) -> dict:
    """HBM peak for the roofline: MEASURED_PEAKS.json (driver-written) or the guide's fallback."""
    path = os.path.join(root, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "source": "measured (MEASURED_PEAKS.json)"}
    except (OSError, KeyError, ValueError):
        return {"hbm_gbs": 6650.0, "source": "fallback (B200_PROFILING.md: 6.65 TB/s)"}


def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), \
        int(os.environ.get("WORLD_SIZE", "1"))


def dist_max(value: float, device="cpu") -> float:
    """Max over ranks of a scalar (identity when not distributed)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def dist_sum(value: float, device="cpu") -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def dist_barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()


def aggregate_replicas(units_per_rank: float, ms_local: float, device="cpu") -> dict:
    """Replicas-only scaling: every rank images its own copy of the
    workload; value = units all ranks processed / max-over-ranks time."""
    total_units = dist_sum(units_per_rank, device)
    ms = dist_max(ms_local, device)
    return {"units": total_units, "ms": ms, "per_s": total_units / (ms * 1e-3)}


def csrc_sha256(root: str) -> str:
    """Hash of the kernel sources: ncu traffic figures in profiles/r2_traffic.csv are valid only for the
    sources they were captured at."""
    import hashlib
    d = os.path.join(root, "paper_2601_19714_b200", "csrc")
    h = hashlib.sha256()
    for name in sorted(os.listdir(d)):
        if name.endswith((".cu", ".cuh")):
            with open(os.path.join(d, name), "rb") as f:
                h.update(name.encode() + b"\0" + f.read())
    return h.hexdigest()


# ----------------------------------------------------------------------------------------------
# cuFFT, timed as the GPU-side baseline of a4 (bench.py only; the library never links it)
# ----------------------------------------------------------------------------------------------
_CUFFT_Z2Z, _CUFFT_C2C, _CUFFT_INVERSE = 0x69, 0x29, 1


def _load_cufft():
    import ctypes
    import glob
    import torch
    cands = glob.glob(os.path.join(os.path.dirname(torch.__file__), "..", "nvidia", "cufft", "lib", "libcufft.so*"))
    cands += ["libcufft.so.11", "/usr/local/cuda/lib64/libcufft.so.11", "libcufft.so"]
    err = None
    for c in cands:
        try:
            return ctypes.CDLL(c)
        except OSError as e:
            err = e
    raise RuntimeError(f"libcufft not found: {err}")


def time_cufft_2d(n: int, batch: int, double: bool = True, reps: int = 3) -> float:
    """Milliseconds of one in-place batched 2-D complex transform (cufftPlanMany, Z2Z or C2C, + sign) of
    `batch` dense n x n planes, CUDA events on the current stream, best of `reps` after one warm-up."""
    import ctypes as C
    import torch
    lib = _load_cufft()
    plan = C.c_int(0)
    dims = (C.c_int * 2)(n, n)
    kind = _CUFFT_Z2Z if double else _CUFFT_C2C
    rc = lib.cufftPlanMany(C.byref(plan), 2, dims, None, 1, 0, None, 1, 0, kind, batch)
    if rc != 0:
        raise RuntimeError(f"cufftPlanMany failed: {rc}")
    try:
        stream = torch.cuda.current_stream()
        lib.cufftSetStream(plan, C.c_void_p(stream.cuda_stream))
        buf = torch.zeros((batch, n, n), dtype=torch.complex128 if double else torch.complex64, device="cuda")
        buf[:, n // 2 - 8:n // 2 + 8, n // 2 - 8:n // 2 + 8] = 1.0
        fn = lib.cufftExecZ2Z if double else lib.cufftExecC2C
        ptr = C.c_void_p(buf.data_ptr())
        best = float("inf")
        for i in range(reps + 1):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            rc = fn(plan, ptr, ptr, _CUFFT_INVERSE)
            e1.record()
            torch.cuda.synchronize()
            if rc != 0:
                raise RuntimeError(f"cufftExec failed: {rc}")
            if i > 0:
                best = min(best, e0.elapsed_time(e1))
        del buf
        return best
    finally:
        lib.cufftDestroy(plan)
