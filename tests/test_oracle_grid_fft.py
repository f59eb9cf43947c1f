"""Pins for the oracle's gridding (Eq. 3), per-plane FFT (:53, :68) and
w-correction (Eq. 2, :50)."""
import math

import numpy as np

import oracle

C0 = 299792458.0
S, BETA = 7, 2.34 * 7


def _idx(uvw, N, Nw=1, dl=1e-3):
    return oracle.index(np.asarray(uvw, float), np.array([C0]), N, Nw, S, dl, 16)


def test_single_visibility_at_cell_centre_is_outer_product():
    N, dl = 64, 1e-3
    du = 1.0 / (N * dl)
    r = _idx([[5 * du, -4 * du, 0.0]], N)
    vis = np.array([2.0 - 3.0j])
    G = oracle.grid_plane([0], vis, None, r["iu"], r["iv"], r["xu"], r["xv"], N, S, BETA)
    g = np.array([oracle.kb(a, S, BETA) for a in range(-3, 4)])
    expect = np.zeros((N, N), complex)
    expect[32 - 4 - 3:32 - 4 + 4, 32 + 5 - 3:32 + 5 + 4] = vis[0] * np.outer(g, g)   # [v][u]
    assert np.abs(G - expect).max() < 1e-15
    assert np.count_nonzero(G) == 49


def test_off_centre_footprint_and_separability():
    N, dl = 64, 1e-3
    du = 1.0 / (N * dl)
    xu, xv = 3.3, -7.45
    r = _idx([[xu * du, xv * du, 0.0]], N)
    assert (r["iu"][0], r["iv"][0]) == (35, 25)
    G = oracle.grid_plane([0], np.array([1.0 + 0j]), None, r["iu"], r["iv"], r["xu"], r["xv"], N, S, BETA)
    gu = np.array([oracle.kb((35 - 32 + a) - r["xu"][0], S, BETA) for a in range(-3, 4)])
    gv = np.array([oracle.kb((25 - 32 + b) - r["xv"][0], S, BETA) for b in range(-3, 4)])
    assert np.abs(G[22:29, 32:39].real - np.outer(gv, gu)).max() < 1e-15
    assert np.abs(G.imag).max() == 0.0
    # u is the fast (column) axis: the footprint is wider where |offset| is smaller
    assert abs(r["xu"][0] - xu) < 1e-12 and abs(r["xv"][0] - xv) < 1e-12


def test_mass_invariant_linearity_weights(cfg1):
    wl = cfg1
    N = wl.n
    r = oracle.index(wl.uvw_m, wl.freq_hz, N, 1, S, wl.pixel_rad, 16)
    keep = np.nonzero(r["key"] != np.uint64(0xFFFFFFFFFFFFFFFF))[0]
    vis = wl.vis.ravel()
    rng = np.random.default_rng(5)
    wgt = rng.uniform(0.5, 2.0, vis.shape[0]).astype(np.float32)
    G = oracle.grid_plane(keep, vis, wgt, r["iu"], r["iv"], r["xu"], r["xv"], N, S, BETA)
    # sum over cells = sum_k w_k V_k K_u(k) K_v(k), K = discrete kernel sum at the offset
    tot = 0j
    for k in keep:
        Ku = sum(oracle.kb((r["iu"][k] - N // 2 + a) - r["xu"][k], S, BETA) for a in range(-3, 4))
        Kv = sum(oracle.kb((r["iv"][k] - N // 2 + a) - r["xv"][k], S, BETA) for a in range(-3, 4))
        tot += float(wgt[k]) * vis[k] * Ku * Kv
    assert abs(G.sum() - tot) < 1e-10 * abs(tot)
    # linearity: grid(A) + grid(B) == grid(A u B)
    A, Bk = keep[::2], keep[1::2]
    GA = oracle.grid_plane(A, vis, wgt, r["iu"], r["iv"], r["xu"], r["xv"], N, S, BETA)
    GB = oracle.grid_plane(Bk, vis, wgt, r["iu"], r["iv"], r["xu"], r["xv"], N, S, BETA)
    assert np.abs(GA + GB - G).max() < 1e-12 * np.abs(G).max()
    # weights NULL == weights of 1
    G1 = oracle.grid_plane(keep, vis, None, r["iu"], r["iv"], r["xu"], r["xv"], N, S, BETA)
    Gw = oracle.grid_plane(keep, vis, np.ones_like(wgt), r["iu"], r["iv"], r["xu"], r["xv"], N, S, BETA)
    assert np.array_equal(G1, Gw)


def test_fft_equals_definition_16():
    N = 16
    rng = np.random.default_rng(1)
    g = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    P = oracle.fft2_centered(g)
    i = np.arange(N) - N // 2
    E = np.exp(2j * np.pi * np.outer(i, i) / N)          # E[p][i]
    ref = E @ g.T                                        # over i -> [p][j]
    ref = (E @ ref.T)                                    # over j -> [q][p]
    # explicit O(N^4) loop on a few outputs
    for (q, p) in [(0, 0), (3, 11), (8, 8), (15, 1)]:
        acc = 0j
        for j in range(N):
            for ii in range(N):
                acc += g[j, ii] * np.exp(2j * np.pi * ((ii - 8) * (p - 8) + (j - 8) * (q - 8)) / N)
        assert abs(P[q, p] - acc) < 1e-12
    assert np.abs(P - ref).max() < 1e-12


def test_fft_against_numpy_and_parseval():
    rng = np.random.default_rng(2)
    for N in (4, 64, 256):
        g = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
        P = oracle.fft2_centered(g)
        ref = np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(g))) * (N * N)
        assert np.abs(P - ref).max() < 1e-13 * np.abs(ref).max() * math.log2(N)
        assert abs((np.abs(P) ** 2).sum() / (N * N * (np.abs(g) ** 2).sum()) - 1) < 1e-13


def test_fft_delta_cases():
    N = 64
    g = np.zeros((N, N), complex)
    g[N // 2, N // 2] = 1.0
    assert np.abs(oracle.fft2_centered(g) - 1.0).max() < 1e-14        # delta at centre -> ones
    a, b = 5, -9
    g = np.zeros((N, N), complex)
    g[N // 2 + b, N // 2 + a] = 1.0                                   # [v=j][u=i]
    p = np.arange(N) - N // 2
    ref = np.exp(2j * np.pi * (a * p[None, :] + b * p[:, None]) / N)   # [q][p]
    assert np.abs(oracle.fft2_centered(g) - ref).max() < 1e-13


def test_fft_rejects_bad_sizes():
    for N in (2, 6, 48):
        try:
            oracle.fft2_centered(np.zeros((N, N), complex))
            assert False
        except ValueError:
            pass


def test_wcorrect_w0_identity_and_screen():
    N, dl = 64, 2e-3
    rng = np.random.default_rng(3)
    P = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    I0 = oracle.wcorrect_accumulate(P, dl, 0.0)
    assert np.array_equal(I0, P.real)
    wz = 1234.5
    I1 = oracle.wcorrect_accumulate(P, dl, wz)
    l = (np.arange(N) - N // 2) * dl
    n = np.sqrt(1 - l[None, :] ** 2 - l[:, None] ** 2)
    ref = (P * np.exp(2j * np.pi * wz * (n - 1))).real
    # n-1 by subtraction loses ~1e-16/|n-1| relative: phase error ~ 2 pi w 1e-16
    assert np.abs(I1 - ref).max() < 1e-11
    # accumulation: calling twice adds
    I2 = oracle.wcorrect_accumulate(P, dl, wz, image=I1.copy())
    assert np.allclose(I2, 2 * I1, rtol=0, atol=1e-13)


def test_wcorrect_horizon_pixels_zero():
    N, dl = 16, 0.2          # l up to 1.6: pixels with l^2+m^2 >= 1 stay zero (R18)
    P = np.ones((N, N), complex)
    I = oracle.wcorrect_accumulate(P, dl, 3.0)
    l = (np.arange(N) - N // 2) * dl
    r2 = l[None, :] ** 2 + l[:, None] ** 2
    assert np.all(I[r2 >= 1.0] == 0.0) and np.all(I[r2 < 0.99] != 0.0)


def test_one_visibility_plane_wave_times_screen():
    """One visibility at a cell centre on plane z: image = taper-corrected plane wave x screen."""
    N, dl, Nw = 64, 1e-3, 4
    du = 1.0 / (N * dl)
    a, b = 6, -3
    uvw = np.array([[a * du, b * du, 7.0], [0.0, 0.0, 0.0], [0.0, 0.0, 40.0]])
    vis = np.array([1.5 + 0.5j, 0.0, 0.0])                 # rows 1,2 only set the w range
    r = oracle.image(uvw, np.array([C0]), vis, None, N, Nw, S, dl, want_raw=True)
    dw = 40.0 / Nw
    wz = 0.0 + (0 + 0.5) * dw                              # w=7 -> plane 0, centre 5
    p = np.arange(N) - N // 2
    l = p * dl
    n = np.sqrt(1 - l[None, :] ** 2 - l[:, None] ** 2)
    g = np.array([oracle.kb(t, S, BETA) for t in range(-3, 4)])
    # FT of the gridded 7x7 outer product: sum_a g(a) e^{2 pi i a p / N} per axis
    cu = np.array([(g * np.exp(2j * np.pi * np.arange(-3, 4) * pp / N)).sum() for pp in p])
    wave = np.exp(2j * np.pi * (a * p[None, :] + b * p[:, None]) / N)
    ref = (vis[0] * wave * cu[None, :] * cu[:, None] * np.exp(2j * np.pi * wz * (n - 1))).real
    assert np.abs(r["raw_image"] - ref).max() < 1e-12
