"""Pins for the oracle's w < 0 folding (reading R24): hand case, identity on w >= 0,
invariance of the direct DFT (V(-u,-v,-w) = conj V, Eq. 1), and the effect on the
w-quantisation error of the w-stacked image against the exact DFT."""
import numpy as np

import oracle

C0 = 299792458.0


def _rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def test_fold_hand_case():
    uvw = np.array([[1.0, 2.0, -3.0], [4.0, -5.0, 6.0], [7.0, 8.0, 0.0], [-1.5, 2.5, -0.25]])
    vis = np.array([[1 + 2j, 3 - 4j], [5 + 6j, 7 + 8j], [9 - 1j, 2 + 2j], [0.5 + 0.25j, -1 - 1j]])
    u2, v2, n = oracle.fold_w(uvw, vis)
    assert n == 2
    assert np.array_equal(u2, np.array([[-1.0, -2.0, 3.0], [4.0, -5.0, 6.0], [7.0, 8.0, 0.0], [1.5, -2.5, 0.25]]))
    assert np.array_equal(v2, np.array([[1 - 2j, 3 + 4j], [5 + 6j, 7 + 8j], [9 - 1j, 2 + 2j], [0.5 - 0.25j, -1 + 1j]]))
    # the inputs are not touched; -0.0 and NaN rows are left alone
    assert uvw[0, 2] == -3.0 and vis[0, 0] == 1 + 2j
    u3, v3, n3 = oracle.fold_w(np.array([[1.0, 1.0, -0.0], [1.0, 1.0, np.nan]]), np.array([[1 + 1j], [2 + 2j]]))
    assert n3 == 0 and v3[0, 0] == 1 + 1j and v3[1, 0] == 2 + 2j


def test_fold_is_identity_for_nonnegative_w(cfg1):
    uvw = cfg1.uvw_m.copy()
    uvw[:, 2] = np.abs(uvw[:, 2])
    u2, v2, n = oracle.fold_w(uvw, cfg1.vis)
    assert n == 0 and np.array_equal(u2, uvw) and np.array_equal(v2, cfg1.vis.astype(np.complex128))


def test_fold_leaves_the_direct_dft_unchanged_and_halves_the_w_error(cfg1, cfg1_oracle):
    wl = cfg1
    N = wl.n
    assert (wl.uvw_m[:, 2] < 0).sum() > wl.n_rows // 4          # the case has rows to fold
    uf, vf, n = oracle.fold_w(wl.uvw_m, wl.vis)
    assert n == int((wl.uvw_m[:, 2] < 0).sum()) and (uf[:, 2] >= 0).all()
    s = wl.freq_hz / C0
    lam = lambda uvw, k: (uvw[:, k:k + 1] * s[None, :]).ravel()
    # the plain definition does not see the fold: every term keeps its real part
    Nd = 64
    dl = wl.pixel_rad * N / Nd
    D0 = oracle.dft(lam(wl.uvw_m, 0), lam(wl.uvw_m, 1), lam(wl.uvw_m, 2), wl.vis, None, None, Nd, dl)
    D1 = oracle.dft(lam(uf, 0), lam(uf, 1), lam(uf, 2), vf, None, None, Nd, dl)
    assert _rel(D1, D0) < 1e-12
    # conjugating without negating (u, v) -- or the reverse -- is a different image
    Dbad = oracle.dft(lam(wl.uvw_m, 0), lam(wl.uvw_m, 1), lam(uf, 2), vf, None, None, Nd, dl)
    assert _rel(Dbad, D0) > 1e-2

    # w-stacked images against the exact DFT of the gridded visibilities, inner half (reading R14)
    idx = oracle.index(wl.uvw_m, wl.freq_hz, N, wl.n_wplanes, wl.support, wl.pixel_rad, 16)
    keep = idx["key"] != np.uint64(0xFFFFFFFFFFFFFFFF)
    idf = oracle.index(uf, wl.freq_hz, N, wl.n_wplanes, wl.support, wl.pixel_rad, 16)
    keepf = idf["key"] != np.uint64(0xFFFFFFFFFFFFFFFF)
    assert idf["w_min"][0] >= 0.0
    assert idf["w_max"][0] - idf["w_min"][0] < 0.6 * (idx["w_max"][0] - idx["w_min"][0])
    both = keep & keepf                                         # the grid is not symmetric: edge cells may differ
    assert both.sum() > 0.98 * keep.sum()
    De = oracle.dft(lam(wl.uvw_m, 0), lam(wl.uvw_m, 1), lam(wl.uvw_m, 2), wl.vis, None, both, N, wl.pixel_rad)
    vis_both = np.where(both.reshape(wl.vis.shape), wl.vis, 0)
    inner = slice(N // 4, 3 * N // 4)
    img = lambda nw, fold: oracle.image(wl.uvw_m, wl.freq_hz, vis_both, None, N, nw, wl.support, wl.pixel_rad, fold=fold)["image"]
    e_unf = _rel(img(wl.n_wplanes, False)[inner, inner], De[inner, inner])
    e_fold = _rel(img(wl.n_wplanes, True)[inner, inner], De[inner, inner])
    e_fold_half = _rel(img(wl.n_wplanes // 2, True)[inner, inner], De[inner, inner])
    print(f"w-stacking error vs exact DFT (inner half): N_w={wl.n_wplanes} unfolded {e_unf:.3e}, folded {e_fold:.3e}; "
          f"N_w={wl.n_wplanes // 2} folded {e_fold_half:.3e}")
    assert e_fold < 0.7 * e_unf                 # half the plane spacing -> about half the phase error
    assert e_fold_half < 1.3 * e_unf            # the same accuracy from half the planes
