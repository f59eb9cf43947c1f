"""Pins for the oracle's Kaiser-Bessel kernel and taper (readings R5, R12)."""
import math
import os

import numpy as np
import scipy.special as sp

import oracle

S, BETA = 7, 2.34 * 7
GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "kaiser_bessel_S7.txt")) as f:
    for line in f:
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            GOLD[k] = float(v)


def test_i0_against_scipy():
    for x in [0.0, 1e-3, 0.5, 1.0, 3.3, 7.0, 12.5, 16.38, 25.0, 35.1]:
        assert oracle.bessel_i0(x) == sp.i0(x) or abs(oracle.bessel_i0(x) / sp.i0(x) - 1) < 5e-15


def test_i0_golden():
    assert abs(oracle.bessel_i0(16.38) - GOLD["i0_beta"]) < 1e-6


def test_kb_special_values():
    assert oracle.kb(0.0, S, BETA) == 1.0
    assert abs(oracle.kb(S / 2, S, BETA) - 1.0 / sp.i0(BETA)) < 1e-20
    assert abs(oracle.kb(-S / 2, S, BETA) - 1.0 / sp.i0(BETA)) < 1e-20
    assert oracle.kb(S / 2 + 0.01, S, BETA) == 0.0
    for t in np.linspace(0, S / 2, 37):
        assert oracle.kb(t, S, BETA) == oracle.kb(-t, S, BETA)          # even
        ref = sp.i0(BETA * math.sqrt(max(0.0, 1 - (2 * t / S) ** 2))) / sp.i0(BETA)
        # condition number of I0(beta sqrt(y)) w.r.t. y is ~beta/2: a few ulp either side
        assert abs(oracle.kb(t, S, BETA) - ref) < 4e-15
    ts = np.linspace(0, S / 2, 200)
    g = [oracle.kb(t, S, BETA) for t in ts]
    assert all(a > b for a, b in zip(g[:-1], g[1:]))                    # decreasing on [0,S/2]


def _closed(nu, s, beta):
    a = beta * beta - (math.pi * s * nu) ** 2
    if a > 0:
        f = math.sinh(math.sqrt(a)) / math.sqrt(a)
    elif a < 0:
        f = math.sin(math.sqrt(-a)) / math.sqrt(-a)
    else:
        f = 1.0
    return s / sp.i0(beta) * f


def test_taper_quadrature_equals_closed_form():
    for nu in np.linspace(-0.5, 0.5, 41):
        assert abs(oracle.taper(nu, S, BETA) / _closed(nu, S, BETA) - 1) < 1e-12
    # oscillatory branch (a < 0) and other supports
    for s, beta in [(7, 5.0), (3, 2.34 * 3), (15, 2.34 * 15), (5, 1.0)]:
        for nu in [0.0, 0.1, 0.3, 0.5]:
            c = _closed(nu, s, beta)
            assert abs(oracle.taper(nu, s, beta) - c) < 1e-13 * max(1.0, abs(_closed(0, s, beta)))


def test_taper_golden():
    assert abs(oracle.taper(0.0, S, BETA) - GOLD["taper_0"]) < 1e-13
    assert abs(oracle.taper(0.25, S, BETA) - GOLD["taper_0.25"]) < 1e-13
    assert abs(oracle.taper(0.5, S, BETA) - GOLD["taper_0.5"]) < 1e-13


def test_taper_is_integral_of_kernel_samples():
    # c(0) = integral of g; the S-term discrete kernel sum at any offset equals it to ~1e-6
    # (2.150692-2.150694), tying the taper to the gridding kernel.
    for off in [0.0, 0.13, -0.37, 0.5]:
        ksum = sum(oracle.kb(a - off, S, BETA) for a in range(-3, 4))
        assert abs(ksum - oracle.taper(0.0, S, BETA)) < 3e-6
