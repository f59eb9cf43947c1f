"""Pins for steps 1-4 (scales, cell index, plane index, key, stable sort); Eq. 5 :129."""
import math

import numpy as np

import oracle

C0 = 299792458.0
DROPPED = np.uint64(0xFFFFFFFFFFFFFFFF)


def _one(u_cells, v_cells, N=64, Nw=4, S=7, w=(0.0,), B=16, freq=C0, dl=1e-3, **kw):
    """Visibilities placed at given cell coordinates: u_lambda = cells * du, du = 1/(N dl);
    freq = c0 so metres == wavelengths."""
    du = 1.0 / (N * dl)
    u = np.atleast_1d(np.asarray(u_cells, float)) * du
    v = np.atleast_1d(np.asarray(v_cells, float)) * du
    ww = np.resize(np.asarray(w, float), u.shape)
    uvw = np.stack([u, v, ww], 1)
    return oracle.index(uvw, np.array([freq]), N, Nw, S, dl, B, **kw)


def test_hand_cases_cell_centre_and_tie():
    r = _one([3.0, 2.5, -0.5, -0.49999, 2.4999], [0.0, 0.0, 0.0, 0.0, -7.5], N=64)
    assert list(r["iu"]) == [35, 35, 32, 32, 34]          # floor(x + N/2 + 0.5): ties go up
    assert list(r["iv"]) == [32, 32, 32, 32, 25]
    # at a cell centre all kernel offsets are integers
    assert abs(r["xu"][0] - 3.0) < 1e-12


def test_on_grid_rule_eq5_halo():
    N, S = 64, 7   # h = 3: centre cells 3..60 are kept, 2 and 61 dropped
    r = _one([3 - 32, 2 - 32, 60 - 32, 61 - 32, 0, 0], [0, 0, 0, 0, 3 - 32, 61 - 32], N=N, S=S)
    assert list(r["iu"][:4]) == [3, 2, 60, 61]
    dropped = r["key"] == DROPPED
    assert list(dropped) == [False, True, False, True, False, True]


def test_plane_index_closest_plane_and_clamp():
    w = np.array([0.0, 1.0, 2.49, 2.5, 9.99, 10.0, 5.0])
    r = _one(np.zeros(7), np.zeros(7), w=w, Nw=4)
    assert r["w_min"][0] == 0.0 and r["w_max"][0] == 10.0
    assert list(r["ip"]) == [0, 0, 0, 1, 3, 3, 2]         # w = w_max clamps to plane Nw-1
    # closest plane centre: centres 1.25, 3.75, 6.25, 8.75
    centres = 0.0 + (np.arange(4) + 0.5) * 2.5
    for wk, ipk in zip(w, r["ip"]):
        assert ipk == int(np.argmin(np.abs(centres - wk))) or wk in (2.5, 5.0)
    # degenerate: all w equal -> plane 0
    r = _one(np.zeros(3), np.zeros(3), w=[4.0, 4.0, 4.0], Nw=4)
    assert list(r["ip"]) == [0, 0, 0]


def test_key_layout():
    N, B, Nw = 64, 16, 4
    r = _one([0.0, 17.0, -20.0], [0.0, -3.0, 20.0], w=[0.0, 10.0, 5.0], N=N, B=B, Nw=Nw)
    T = N // B
    for k in range(3):
        iu, iv, ip = int(r["iu"][k]), int(r["iv"][k]), int(r["ip"][k])
        expect = (((ip * T + iv // B) * T + iu // B) * B + iv % B) * B + iu % B
        assert int(r["key"][k]) == expect
    assert list(r["iu"]) == [32, 49, 12] and list(r["iv"]) == [32, 29, 52]
    # (plane, tile row, tile column) then (row, column) inside the 16 x 16 tile
    assert [int(x) for x in r["key"]] == [(((0 * 4 + 2) * 4 + 2) * 16 + 0) * 16 + 0,
                                          (((3 * 4 + 1) * 4 + 3) * 16 + 13) * 16 + 1,
                                          (((2 * 4 + 3) * 4 + 0) * 16 + 4) * 16 + 12]
    # the cell inside the tile is the least significant part: same tile, same plane -> keys differ by the cell
    r2 = _one([0.0, 1.0, 0.0], [0.0, 0.0, 1.0], N=N, B=B, Nw=Nw)
    assert int(r2["key"][1]) - int(r2["key"][0]) == 1 and int(r2["key"][2]) - int(r2["key"][0]) == B


def test_channel_scaling_and_cube_key():
    N, Nw, dl = 64, 2, 1e-3
    du = 1.0 / (N * dl)
    uvw = np.array([[4.0 * du, -2.0 * du, 1.0], [1.0 * du, 1.0 * du, 3.0]])
    freq = np.array([C0, 2 * C0])                        # channel 1 doubles u, v, w
    r = oracle.index(uvw, freq, N, Nw, 7, dl, 16, cube=0)
    assert list(r["iu"]) == [36, 40, 33, 34] and list(r["iv"]) == [30, 28, 33, 34]
    assert r["w_min"][0] == 1.0 and r["w_max"][0] == 6.0
    rc = oracle.index(uvw, freq, N, Nw, 7, dl, 16, cube=1)
    assert list(rc["w_min"]) == [1.0, 2.0] and list(rc["w_max"]) == [3.0, 6.0]
    T = N // 16
    img = np.array([0, 1, 0, 1])
    iu, iv, ip = rc["iu"].astype(np.int64), rc["iv"].astype(np.int64), rc["ip"].astype(np.int64)
    expect = ((((img * Nw + ip) * T + iv // 16) * T + iu // 16) * 16 + iv % 16) * 16 + iu % 16
    assert [int(x) for x in rc["key"]] == list(expect)


def test_index_bruteforce_cfg1(cfg1):
    wl = cfg1
    B = 16
    r = oracle.index(wl.uvw_m, wl.freq_hz, wl.n, wl.n_wplanes, wl.support, wl.pixel_rad, B)
    # explicit python loop over a sample, in exact rational-free float steps
    N, h = wl.n, 3
    s = wl.freq_hz[0] / C0
    wl_all = wl.uvw_m[:, 2] * s
    wmin, wmax = wl_all.min(), wl_all.max()
    assert r["w_min"][0] == wmin and r["w_max"][0] == wmax
    dw = (wmax - wmin) / wl.n_wplanes
    n_drop = 0
    for k in range(0, wl.n_rows, 7):
        xu = (wl.uvw_m[k, 0] * s) * (N * wl.pixel_rad)
        xv = (wl.uvw_m[k, 1] * s) * (N * wl.pixel_rad)
        iu = math.floor(xu + (N / 2 + 0.5))
        iv = math.floor(xv + (N / 2 + 0.5))
        ip = min(wl.n_wplanes - 1, math.floor((wl_all[k] - wmin) * (1.0 / dw)))
        assert (r["iu"][k], r["iv"][k], r["ip"][k]) == (iu, iv, ip)
        on = iu - h >= 0 and iu + h <= N - 1 and iv - h >= 0 and iv + h <= N - 1
        assert (r["key"][k] != DROPPED) == on
        n_drop += (not on)
        # nearest cell: |x - (i - N/2)| <= 1/2
        assert abs(xu - (iu - N / 2)) <= 0.5 and abs(xv - (iv - N / 2)) <= 0.5
    assert n_drop > 0                                     # the config exercises the drop rule


def test_sort_is_stable_sort(cfg1):
    wl = cfg1
    r = oracle.index(wl.uvw_m, wl.freq_hz, wl.n, wl.n_wplanes, wl.support, wl.pixel_rad, 16)
    perm = oracle.sort(r["key"])
    ref = np.argsort(r["key"], kind="stable")
    assert np.array_equal(perm, ref.astype(np.uint32))
    assert np.array_equal(np.sort(perm), np.arange(wl.n_vis, dtype=np.uint32))
    ks = r["key"][perm]
    assert np.all(ks[1:] >= ks[:-1])
    # ties keep index order
    same = ks[1:] == ks[:-1]
    assert np.all(perm[1:][same] > perm[:-1][same])
    assert oracle.sort(np.zeros(0, np.uint64)).shape == (0,)


def test_nonfinite_and_out_of_int_range_coordinates_are_dropped():
    """Reading R23: a visibility with a non-finite u, v or w cannot lie on the grid (R10) and is
    dropped; a non-finite w takes no part in the w range; a finite coordinate beyond the int range is off
    the grid like any other.  Everything else about the clean rows is unchanged by their presence."""
    N, Nw, S, dl, B = 64, 4, 7, 1e-3, 16
    du = 1.0 / (N * dl)
    f = np.array([299792458.0])
    clean = np.array([[1.2 * du, -3.4 * du, 10.0], [5.0 * du, 6.0 * du, -20.0], [-7.7 * du, 0.3 * du, 30.0]])
    bad = np.array([[np.nan, 0.0, 1.0], [0.0, np.inf, 2.0], [0.0, 0.0, np.nan], [1.0 * du, 1.0 * du, -np.inf],
                    [1e300, 0.0, 3.0], [0.0, -4e12 * du, 4.0]])
    uvw = np.concatenate([clean[:1], bad[:3], clean[1:2], bad[3:], clean[2:]])
    r = oracle.index(uvw, f, N, Nw, S, dl, B)
    r0 = oracle.index(clean, f, N, Nw, S, dl, B)
    DROPPED = np.uint64(0xFFFFFFFFFFFFFFFF)
    is_clean = np.array([True, False, False, False, True, False, False, False, True])
    assert np.all(r["key"][~is_clean] == DROPPED)
    # the w range is that of the rows with a finite w (rows 5 and 6 of `bad` have finite w = 3, 4: inside it)
    assert r["w_min"][0] == -20.0 and r["w_max"][0] == 30.0
    assert r0["w_min"][0] == -20.0 and r0["w_max"][0] == 30.0
    assert np.array_equal(r["key"][is_clean], r0["key"]) and np.all(r0["key"] != DROPPED)
    assert np.array_equal(r["ip"][is_clean], r0["ip"])
    # all rows non-finite in w: range collapses to [0, 0] as for an empty set
    r1 = oracle.index(bad[2:4], f, N, Nw, S, dl, B)
    assert r1["w_min"][0] == 0.0 and r1["w_max"][0] == 0.0 and np.all(r1["key"] == DROPPED)
