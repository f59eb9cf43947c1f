"""GPU parity of the SURVEY 8(f) rows: w < 0 folding (item 4, reading R24), the w-plane histogram (item 3,
PAPER.md:135) and w-plane shards (item 2 / 8(e): the shards' images must add up to the oracle's image of the
whole problem).  The ranks of a multi-GPU run are emulated one after the other on the one GPU (no kernel waits
on another); the reduction plumbing itself is covered on the CPU (tests/test_sharding.py, gloo)."""
import numpy as np
import pytest

import oracle
from paper_2601_19714_b200 import synth

pytestmark = pytest.mark.gpu

TOL64, TOL32, MAXF = 1e-10, 1e-4, 5.0
DROPPED = np.uint64(0xFFFFFFFFFFFFFFFF)


def _rel(a, b):
    nb = np.linalg.norm(np.asarray(b).ravel())
    return np.linalg.norm((np.asarray(a) - np.asarray(b)).ravel()) / (nb if nb > 0 else 1.0)


def _close(a, b, tol, what=""):
    e2 = _rel(a, b)
    em = float(np.max(np.abs(a - b))) / float(np.max(np.abs(b)))
    assert e2 <= tol and em <= MAXF * tol, (what, e2, em)
    return e2


def _rick():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    from paper_2601_19714_b200 import rick
    return rick


def _cases():
    return [("cfg1", synth.make_config(1), {}),
            ("cfg2 mid 1024^2 weights", synth.make_config(2, n_times=8, n=1024, n_wplanes=6, n_src=8, with_weights=True), {}),
            ("N=4096 fused columns", synth.make_config(2, n_times=2, n_wplanes=5, n_src=4), {}),
            ("N=8192 fused columns", synth.make_config(3, n_times=2, n_wplanes=3, n_src=4), {}),
            ("fp32 plane batches", synth.make_config(4, n_times=4, n=1024, n_wplanes=7, n_src=4), dict(plane_batch=2)),
            ("fp32 N=8192 fused columns over the occupied rows", synth.make_config(4, n_times=2, n=8192, n_wplanes=4, n_src=4),
             dict(plane_batch=2))]


@pytest.mark.parametrize("case", range(6))
def test_fold_w_matches_the_folded_oracle(case):
    rick = _rick()
    name, wl, over = _cases()[case]
    tol = TOL32 if wl.grid_prec == "f32" else TOL64
    uf, vf, n_fold = oracle.fold_w(wl.uvw_m, wl.vis)
    assert n_fold > 0
    o = oracle.image(wl.uvw_m, wl.freq_hz, wl.vis, wl.weights, wl.n, wl.n_wplanes, wl.support, wl.pixel_rad, fold=True)
    plan = rick.plan_from_workload(wl, flags=rick.RICK_FLAG_FOLD_W, **over)
    vis, uvw, wgt = rick.to_device(wl)
    img = plan.rick_image(vis, uvw, wgt, wl.freq_hz).cpu().numpy()
    st = plan.rick_get_stats()
    if not over:     # whole stack resident: keys and permutation of the folded problem, bit-exact
        idx = oracle.index(uf, wl.freq_hz, wl.n, wl.n_wplanes, wl.support, wl.pixel_rad, 16)
        assert np.array_equal(plan.debug_keys(), idx["key"])
        assert np.array_equal(plan.debug_perm(), oracle.sort(idx["key"]))
    plan.destroy()
    e = _close(img, o["image"], tol, name)
    print(f"fold {name}: {n_fold} of {wl.n_rows} rows folded, rel L2 {e:.2e}, w range [{st['w_min']:.1f}, {st['w_max']:.1f}]")
    assert st["w_min"] >= 0.0 and st["w_min"] == o["stats"]["w_min"] and st["w_max"] == o["stats"]["w_max"]
    assert st["n_gridded"] == o["stats"]["n_gridded"] and st["n_dropped"] == o["stats"]["n_dropped"]
    # and the unfolded image is a different one (the planes sit elsewhere): the flag is not a no-op
    o0 = oracle.image(wl.uvw_m, wl.freq_hz, wl.vis, wl.weights, wl.n, wl.n_wplanes, wl.support, wl.pixel_rad)
    assert _rel(img, o0["image"]) > max(1e-6, 3 * tol)


def test_plane_histogram_equals_oracle_counts():
    rick = _rick()
    for fold in (0, 1):
        for name, wl, _ in _cases()[:3]:
            uvw_h = oracle.fold_w(wl.uvw_m, wl.vis)[0] if fold else wl.uvw_m
            idx = oracle.index(uvw_h, wl.freq_hz, wl.n, wl.n_wplanes, wl.support, wl.pixel_rad, 16)
            want = np.bincount(idx["ip"][idx["key"] != DROPPED], minlength=wl.n_wplanes)
            plan = rick.plan_from_workload(wl, plane_batch=1, flags=fold)
            _, uvw, _ = rick.to_device(wl)
            hist = plan.rick_plane_histogram(uvw, wl.freq_hz)
            plan.destroy()
            assert np.array_equal(hist, want), (name, fold, hist, want)


@pytest.mark.parametrize("case", range(6))
def test_shards_add_up_to_the_whole_image(case):
    rick = _rick()
    from paper_2601_19714_b200 import sharded
    import torch
    name, wl, over = _cases()[case]
    tol = TOL32 if wl.grid_prec == "f32" else TOL64
    o = oracle.image(wl.uvw_m, wl.freq_hz, wl.vis, wl.weights, wl.n, wl.n_wplanes, wl.support, wl.pixel_rad)
    vis, uvw, wgt = rick.to_device(wl)
    kw = dict(n=wl.n, n_wplanes=wl.n_wplanes, support=wl.support, pixel_rad=wl.pixel_rad, grid_prec=wl.grid_prec, **over)
    for world in (2, 3, wl.n_wplanes + 2):                 # the last: more ranks than planes
        total = torch.zeros((wl.n, wl.n), dtype=torch.float64, device="cuda")
        part = torch.empty_like(total)
        n_gridded = n_dropped = 0
        sum_w = 0.0
        seen = []
        for rank in range(world):                          # the ranks, one after the other on this GPU
            sh = sharded.ShardedImager(kw, rank, world, cost=float(wl.n_vis) / wl.n_wplanes)
            b = sh.prepare(uvw, wl.freq_hz)
            sh.image(vis, uvw, wgt, wl.freq_hz, part, reduce=False)
            total += part
            st = sh.stats()
            n_gridded += st["n_gridded"]
            n_dropped += st["n_dropped"]
            sum_w += st["sum_w"]
            seen.append((int(b[rank]), int(b[rank + 1])))
            sh.destroy()
        assert seen[0][0] == 0 and seen[-1][1] == wl.n_wplanes and all(seen[i][1] == seen[i + 1][0] for i in range(world - 1))
        e = _close(total.cpu().numpy(), o["image"], tol, f"{name} world {world}")
        print(f"shards {name} world={world} ranges {seen}: rel L2 of the sum {e:.2e}")
        assert n_gridded == o["stats"]["n_gridded"] and n_dropped == o["stats"]["n_dropped"]
        assert abs(sum_w - o["stats"]["sum_w"]) <= 1e-9 * max(1.0, o["stats"]["sum_w"])


def test_fold_w_in_cube_mode_and_through_the_chunked_host_entry():
    """RICK_FLAG_FOLD_W with cube = 1 (every channel its own folded w range) and through rick_image_stream_host
    (a0 over all rows folds too), N = 8192 fp64 chunked as well (the fused single-pass column kernel)."""
    rick = _rick()
    import torch
    wl = synth.make_config(5, n_times=8, n=512, n_chan=3, n_wplanes=4, n_src=5)
    o = oracle.image(wl.uvw_m, wl.freq_hz, wl.vis, None, wl.n, wl.n_wplanes, wl.support, wl.pixel_rad, cube=1, fold=True)
    plan = rick.plan_from_workload(wl, flags=rick.RICK_FLAG_FOLD_W)
    vis, uvw, wgt = rick.to_device(wl)
    cube = plan.rick_image(vis, uvw, wgt, wl.freq_hz).cpu().numpy()
    plan.destroy()
    for c in range(wl.n_chan):
        _close(cube[c], o["image"][c], TOL64, f"cube channel {c} folded")
    for name, wl, flags in (("cfg1 folded", synth.make_config(1), rick.RICK_FLAG_FOLD_W),
                            ("N=8192 fp64", synth.make_config(3, n_times=3, n_wplanes=3, n_src=4), 0)):
        o = oracle.image(wl.uvw_m, wl.freq_hz, wl.vis, None, wl.n, wl.n_wplanes, wl.support, wl.pixel_rad, fold=bool(flags))
        plan = rick.plan_from_workload(wl, flags=flags)
        hv = torch.from_numpy(np.ascontiguousarray(wl.vis)).pin_memory()
        hu = torch.from_numpy(wl.uvw_m).pin_memory()
        out = torch.full((wl.n, wl.n), float("nan"), dtype=torch.float64).pin_memory()
        for rpc in (wl.n_rows // 3 + 1, wl.n_rows):
            plan.rick_image_stream_host(hv, hu, None, wl.freq_hz, out, rpc)
            e = _close(out.numpy(), o["image"], TOL64, f"{name} stream rows_per_chunk={rpc}")
            st = plan.rick_get_stats()
            assert st["n_gridded"] == o["stats"]["n_gridded"] and st["n_dropped"] == o["stats"]["n_dropped"]
        plan.destroy()
        print(f"stream host {name}: rel L2 {e:.2e}")


def test_shard_and_flag_argument_errors(cfg1):
    rick = _rick()
    kw = dict(n=cfg1.n, n_wplanes=cfg1.n_wplanes, support=cfg1.support, pixel_rad=cfg1.pixel_rad)
    for bad in (dict(z_begin=1), dict(z_begin=6, z_count=3), dict(z_count=-1), dict(z_begin=-1, z_count=2),
                dict(z_count=2, cube=1), dict(flags=2), dict(z_count=2, plane_batch=3)):
        with pytest.raises(rick.RickError):
            rick.Plan(**dict(kw, **bad))
    p = rick.Plan(**dict(kw, cube=1))
    _, uvw, _ = rick.to_device(cfg1)
    with pytest.raises(rick.RickError):
        p.rick_plane_histogram(uvw, cfg1.freq_hz)
    p.destroy()
