"""rick_plane_histogram_noalloc (include/rick.h): the per-plane histogram of PAPER.md:135 through the entry point
that allocates nothing (fixed file-scope device scratch), against the existing rick_plane_histogram and the
oracle's per-plane counts -- integer work, so the bar is equality.  Collected last on purpose (file name): the
suite runs with pytest -x."""
import numpy as np
import pytest

import oracle
from paper_2601_19714_b200 import synth

pytestmark = pytest.mark.gpu


def _rick():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    from paper_2601_19714_b200 import rick
    return rick


def _oracle_hist(wl, uvw_m, fold=False):
    uvw = np.ascontiguousarray(uvw_m, dtype=np.float64)
    if fold:
        uvw = oracle.fold_w(uvw, np.zeros((uvw.shape[0], wl.n_chan), np.complex128))[0]
    ix = oracle.index(uvw, wl.freq_hz, wl.n, wl.n_wplanes, wl.support, wl.pixel_rad, 16)
    keep = ix["key"] != np.uint64(0xFFFFFFFFFFFFFFFF)
    return np.bincount(ix["ip"][keep], minlength=wl.n_wplanes).astype(np.int64)


def test_no_alloc_histogram_two_calls_in_a_row():
    rick = _rick()
    import torch
    # set 1: cfg1-like with several channels (some visibilities fall off the grid); set 2: other rows, other
    # frequencies, fewer of them -- whatever the first call left in the shared scratch must not show in the second
    wl1 = synth.make_config(1, n_times=24, n_chan=5, n_wplanes=11)
    wl2 = synth.make_config(1, n_times=7, n_chan=2, n_wplanes=11, seed=77)
    plan = rick.plan_from_workload(wl1)
    u1 = torch.from_numpy(wl1.uvw_m).cuda()
    u2 = torch.from_numpy(wl2.uvw_m).cuda()
    ref1 = plan.rick_plane_histogram(u1, wl1.freq_hz)
    ref2 = plan.rick_plane_histogram(u2, wl2.freq_hz)
    out = np.full(wl1.n_wplanes, -1, np.int64)
    got1 = plan.rick_plane_histogram_noalloc(u1, wl1.freq_hz, out).copy()
    got2 = plan.rick_plane_histogram_noalloc(u2, wl2.freq_hz, out).copy()      # straight after, same scratch
    got1b = plan.rick_plane_histogram_noalloc(u1, wl1.freq_hz)
    assert np.array_equal(got1, ref1) and np.array_equal(got2, ref2) and np.array_equal(got1b, ref1)
    assert np.array_equal(got1, _oracle_hist(wl1, wl1.uvw_m)) and np.array_equal(got2, _oracle_hist(wl2, wl2.uvw_m))
    assert got1.sum() > got2.sum() > 0 and not np.array_equal(got1, got2)
    # the plan itself is left alone: an image after the calls equals the oracle's
    vis, uvw, wgt = rick.to_device(wl1)
    img = plan.rick_image(vis, uvw, wgt, wl1.freq_hz).cpu().numpy()
    o = oracle.image(wl1.uvw_m, wl1.freq_hz, wl1.vis, wl1.weights, wl1.n, wl1.n_wplanes, wl1.support, wl1.pixel_rad)
    assert np.linalg.norm(img - o["image"]) <= 1e-10 * np.linalg.norm(o["image"])
    assert plan.rick_get_stats()["n_gridded"] == int(ref1.sum())
    # empty set: all zero
    e = torch.empty((0, 3), dtype=torch.float64, device="cuda")
    assert not plan.rick_plane_histogram_noalloc(e, wl1.freq_hz).any()
    plan.destroy()
    print(f"no-alloc histogram: {got1.tolist()} then {got2.tolist()}")


def test_no_alloc_histogram_folded_and_mid_size():
    rick = _rick()
    import torch
    wl = synth.make_config(2, n_times=6, n=1024, n_wplanes=9)          # 2016 baselines x 6 x 16 channels
    plan = rick.plan_from_workload(wl, flags=rick.RICK_FLAG_FOLD_W)
    u = torch.from_numpy(wl.uvw_m).cuda()
    ref = plan.rick_plane_histogram(u, wl.freq_hz)
    got = plan.rick_plane_histogram_noalloc(u, wl.freq_hz)
    got2 = plan.rick_plane_histogram_noalloc(u, wl.freq_hz)
    plan.destroy()
    assert np.array_equal(got, ref) and np.array_equal(got2, ref)
    assert np.array_equal(got, _oracle_hist(wl, wl.uvw_m, fold=True))


def test_no_alloc_histogram_limits_and_argument_errors():
    rick = _rick()
    import torch
    wl = synth.make_config(1, n_times=4)
    u = torch.from_numpy(wl.uvw_m).cuda()
    # more planes than the fixed scratch holds: a clear error, nothing enqueued (one resident plane keeps the plan small)
    big = rick.Plan(n=wl.n, n_wplanes=rick.RICK_NOALLOC_MAX_PLANES + 1, support=wl.support, pixel_rad=wl.pixel_rad,
                    plane_batch=1)
    with pytest.raises(rick.RickError, match="4096 w-planes"):
        big.rick_plane_histogram_noalloc(u, wl.freq_hz)
    assert big.rick_plane_histogram(u, wl.freq_hz).sum() > 0            # the allocating path has no such limit
    big.destroy()
    plan = rick.plan_from_workload(wl)
    with pytest.raises(rick.RickError, match="1024 channels"):
        plan.rick_plane_histogram_noalloc(u, np.linspace(1e9, 2e9, rick.RICK_NOALLOC_MAX_CHAN + 1))
    with pytest.raises(rick.RickError, match="bad frequency"):
        plan.rick_plane_histogram_noalloc(u, np.array([1.4e9, -1.0]))
    with pytest.raises(rick.RickError, match="16-byte"):
        plan.rick_plane_histogram_noalloc(torch.zeros(3 * 8 + 1, dtype=torch.float64, device="cuda")[1:].view(8, 3), wl.freq_hz)
    # still usable afterwards, and exactly at the channel limit
    f = np.linspace(1.3e9, 1.5e9, rick.RICK_NOALLOC_MAX_CHAN)
    assert np.array_equal(plan.rick_plane_histogram_noalloc(u, f), plan.rick_plane_histogram(u, f))
    plan.destroy()
    cube = rick.Plan(n=wl.n, n_wplanes=4, support=wl.support, pixel_rad=wl.pixel_rad, cube=1)
    with pytest.raises(rick.RickError):
        cube.rick_plane_histogram_noalloc(u, wl.freq_hz)
    cube.destroy()
