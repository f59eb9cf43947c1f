"""Multi-GPU imaging by w-plane shards.

One process per GPU.  Every rank holds all visibilities; the w-planes of the problem are cut into contiguous
ranges, one per rank, chosen from the per-plane visibility histogram so that the largest
(visibilities + planes x plane_cost) is as small as possible (the paper's histogram-based balancing, :135,
with w-plane ranges in place of v-slabs: on one node the whole grid of a rank's planes is resident, so no halo
exchange is left).  Each rank images its planes with its own librick_b200 plan (rick_plan_desc.z_begin /
z_count) and the ranks' images are added by ONE reduction of the N x N real image -- the structural fix the
paper is after (its v1 reduced the whole grid, :31).  The a6 taper is linear, so every rank applies it to its
share.  Cube mode shards by channels and has nothing to reduce.

Plumbing only: the arithmetic is in the library (rick_plane_histogram, rick_partition_planes, rick_image);
torch.distributed (NCCL on GPUs, gloo in the CPU tests of the host logic) carries the reduction.
"""
from __future__ import annotations

from typing import Optional, Sequence

import numpy as np
import torch

from . import rick

# cost of one w-plane's row pass + column pass + correction in units of one visibility's sort + gridding,
# from the per-kernel times of bench.py on a B200: t(a4..a6 per plane) / t(a0..a3 per visibility)
PLANE_COST_VIS = {4096: 1.0e6, 8192: 4.5e6, 16384: 1.1e7}


def plane_cost(n: int) -> float:
    """Default plane cost [visibilities] for grid edge n (scales as n^2 log n between the measured sizes)."""
    if n in PLANE_COST_VIS:
        return PLANE_COST_VIS[n]
    ref = 4096
    return PLANE_COST_VIS[ref] * (n * n * np.log2(n)) / (ref * ref * np.log2(ref))


def shard_bounds(hist: Sequence[int], world: int, cost: float) -> np.ndarray:
    """[world + 1] plane bounds: rank r owns planes bounds[r] .. bounds[r+1]-1 (rick_partition_planes)."""
    return rick.rick_partition_planes(np.asarray(hist, dtype=np.int64), world, cost)


def channel_bounds(n_chan: int, world: int) -> np.ndarray:
    """Cube mode: contiguous channel ranges of (almost) equal length."""
    return np.array([(n_chan * r) // world for r in range(world + 1)], dtype=np.int32)


def reduce_image(img: torch.Tensor, dst: int = 0, group=None) -> torch.Tensor:
    """Sum of the ranks' images on rank `dst` (in place; identity when not distributed)."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.reduce(img, dst=dst, op=dist.ReduceOp.SUM, group=group)
    return img


class ShardedImager:
    """rick_image over the w-plane shard of one rank.  plan_kw: keyword arguments of rick.Plan for the WHOLE
    problem (n, n_wplanes, support, pixel_rad, ...).  The histogram and the bounds are computed once per
    visibility set (prepare); image() can then be called repeatedly (e.g. by bench.py)."""

    def __init__(self, plan_kw: dict, rank: int, world: int, cost: Optional[float] = None):
        self.kw, self.rank, self.world = dict(plan_kw), int(rank), int(world)
        self.cost = plane_cost(int(plan_kw["n"])) if cost is None else float(cost)
        self.plan: Optional[rick.Plan] = None
        self.bounds = None
        self.hist = None

    def prepare(self, uvw_m: torch.Tensor, chan_freq_hz) -> np.ndarray:
        """Histogram (on this rank's GPU, from a one-plane probe plan), bounds, and this rank's plan."""
        probe_kw = dict(self.kw)
        probe_kw.update(plane_batch=1, cube=0)
        probe = rick.Plan(**probe_kw)
        try:
            self.hist = probe.rick_plane_histogram(uvw_m, chan_freq_hz)
        finally:
            probe.destroy()
        self.bounds = shard_bounds(self.hist, self.world, self.cost)
        z0, z1 = int(self.bounds[self.rank]), int(self.bounds[self.rank + 1])
        if self.plan is not None:
            self.plan.destroy()
            self.plan = None
        if z1 > z0:
            kw = dict(self.kw)
            kw.update(z_begin=z0, z_count=z1 - z0)
            if kw.get("plane_batch", 0) > z1 - z0:
                kw["plane_batch"] = 0
            self.plan = rick.Plan(**kw)
        return self.bounds

    def image(self, vis, uvw_m, weights, chan_freq_hz, out: torch.Tensor, reduce: bool = True, dst: int = 0):
        """This rank's share into `out` ([N][N] float64, device), then the reduction onto rank dst."""
        if self.plan is None:
            out.zero_()                      # more ranks than planes: this rank adds nothing
        else:
            self.plan.rick_image(vis, uvw_m, weights, chan_freq_hz, out)
        if reduce:
            reduce_image(out, dst)
        return out

    def stats(self) -> dict:
        if self.plan is None:
            return dict(n_gridded=0, n_dropped=0, sum_w=0.0, n_launches=0)
        return self.plan.rick_get_stats()

    def destroy(self):
        if self.plan is not None:
            self.plan.destroy()
            self.plan = None
