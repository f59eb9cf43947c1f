"""Seeded synthetic interferometer workloads (input generator only).

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path; it
holds none of the imaging method's arithmetic (no indexing, no gridding kernel,
no FFT, no w-correction).  It only produces the arrays the method consumes:

    uvw_m   [R][3] float64   baseline coordinates in metres
    freq_hz [C]    float64   channel centre frequencies
    vis     [R][C] complex64 / complex128
    weights [R][C] float32   (or None == natural weights of 1)

The recipe is the one DESIGN.md states (shapes of the paper's MeerKAT / LOFAR
runs, PAPER.md:151, :216, :280 -- the datasets themselves are not available):
antennas in local East/North, Earth-rotation synthesis, point-source sky
through the measurement equation (Eq. 1) plus Gaussian noise.

Small random draws (antenna positions, sources, noise) come from
``numpy.random.Generator(PCG64(seed))`` on the host so they do not depend on
the device; the deterministic heavy part (the sum over sources) runs in torch
on whatever device is asked for, in float64.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np
import torch

C0 = 299792458.0
SEED_BASE = 20260119
ARCSEC = math.pi / 180.0 / 3600.0
DEG = math.pi / 180.0


@dataclasses.dataclass
class Workload:
    """One imaging problem: inputs + the imaging parameters of the config."""
    name: str
    uvw_m: np.ndarray          # [R][3] f64
    freq_hz: np.ndarray        # [C] f64
    vis: np.ndarray            # [R][C] c64 or c128
    weights: Optional[np.ndarray]  # [R][C] f32 or None
    n: int                     # grid edge N
    n_wplanes: int             # N_w
    support: int               # S
    pixel_rad: float           # delta-l
    grid_prec: str             # "f64" | "f32"
    cube: int                  # 0 MFS, 1 one image per channel
    plane_batch: int           # 0 = all planes resident
    sources: np.ndarray        # [n_src][3]: l, m, flux  (for closed-form tests)

    @property
    def n_rows(self) -> int:
        return int(self.uvw_m.shape[0])

    @property
    def n_chan(self) -> int:
        return int(self.freq_hz.shape[0])

    @property
    def n_vis(self) -> int:
        return self.n_rows * self.n_chan


# ----------------------------------------------------------------------------
# geometry
# ----------------------------------------------------------------------------

def _antennas_disc(rng, n_ant, radius):
    r = radius * np.sqrt(rng.random(n_ant))
    th = 2.0 * math.pi * rng.random(n_ant)
    return np.stack([r * np.cos(th), r * np.sin(th)], axis=1)


def _antennas_core_outer(rng, n_core, core_sigma, n_outer, r_lo, r_hi, max_baseline):
    core = rng.normal(0.0, core_sigma, size=(n_core, 2))
    lr = rng.uniform(math.log(r_lo), math.log(r_hi), size=n_outer)
    th = rng.uniform(0.0, 2.0 * math.pi, size=n_outer)
    outer = np.stack([np.exp(lr) * np.cos(th), np.exp(lr) * np.sin(th)], axis=1)
    pos = np.concatenate([core, outer], axis=0)
    d = pos[:, None, :] - pos[None, :, :]
    longest = float(np.sqrt((d ** 2).sum(-1)).max())
    return pos * (max_baseline / longest)


def _uvw_rows(ant_en, lat_rad, dec_rad, ha_rad):
    """[T*B][3] metres; rows time-major, baseline-minor (i<j)."""
    n_ant = ant_en.shape[0]
    ii, jj = np.triu_indices(n_ant, k=1)
    d_e = ant_en[jj, 0] - ant_en[ii, 0]
    d_n = ant_en[jj, 1] - ant_en[ii, 1]
    X = -math.sin(lat_rad) * d_n
    Y = d_e
    Z = math.cos(lat_rad) * d_n
    sH = np.sin(ha_rad)[:, None]
    cH = np.cos(ha_rad)[:, None]
    sd, cd = math.sin(dec_rad), math.cos(dec_rad)
    u = sH * X + cH * Y
    v = -sd * cH * X + sd * sH * Y + cd * Z
    w = cd * cH * X - cd * sH * Y + sd * Z
    return np.stack([u.ravel(), v.ravel(), w.ravel()], axis=1).astype(np.float64)


def _powerlaw_flux(rng, n, f_lo, f_hi):
    # pdf ~ F^-1.5 on [f_lo, f_hi]
    U = rng.random(n)
    a, b = f_lo ** -0.5, f_hi ** -0.5
    return (a - U * (a - b)) ** -2.0


# ----------------------------------------------------------------------------
# visibilities: measurement equation for point sources
# ----------------------------------------------------------------------------

def _model_vis(uvw_m, freq_hz, src, device, row_chunk=1 << 15):
    """V[r][c] = sum_s F_s/n_s * exp(-2 pi i (u l + v m + w (n-1))), f64."""
    dev = torch.device(device)
    uvw = torch.as_tensor(uvw_m, dtype=torch.float64, device=dev)
    s_c = torch.as_tensor(freq_hz / C0, dtype=torch.float64, device=dev)
    l = torch.as_tensor(src[:, 0], dtype=torch.float64, device=dev)
    m = torch.as_tensor(src[:, 1], dtype=torch.float64, device=dev)
    F = torch.as_tensor(src[:, 2], dtype=torch.float64, device=dev)
    nn = torch.sqrt(1.0 - l * l - m * m)
    amp = F / nn
    nm1 = -(l * l + m * m) / (1.0 + nn)
    R, C = uvw.shape[0], s_c.shape[0]
    out_re = torch.empty((R, C), dtype=torch.float64, device=dev)
    out_im = torch.empty((R, C), dtype=torch.float64, device=dev)
    if dev.type == "cuda":
        row_chunk = max(1, (1 << 24) // max(1, C * src.shape[0]) * 8)
    else:
        row_chunk = max(1, (1 << 22) // max(1, C * src.shape[0]))
    for r0 in range(0, R, row_chunk):
        r1 = min(R, r0 + row_chunk)
        # geometric delay in metres per source: [r][s]
        g = (uvw[r0:r1, 0:1] * l[None, :] + uvw[r0:r1, 1:2] * m[None, :]
             + uvw[r0:r1, 2:3] * nm1[None, :])
        ph = g[:, None, :] * s_c[None, :, None]          # cycles [r][c][s]
        ph = ph - torch.round(ph)
        ang = (-2.0 * math.pi) * ph
        out_re[r0:r1] = (torch.cos(ang) * amp).sum(-1)
        out_im[r0:r1] = (torch.sin(ang) * amp).sum(-1)
    return out_re.cpu().numpy(), out_im.cpu().numpy()


def _finish(name, rng, ant, lat, dec, ha0_h, ha1_h, n_times, freq, src, sigma,
            vis_dtype, device, **img):
    ha = np.linspace(ha0_h, ha1_h, n_times) * (math.pi / 12.0)
    uvw = _uvw_rows(ant, lat * DEG, dec * DEG, ha)
    re, im = _model_vis(uvw, freq, src, device)
    R, C = re.shape
    if sigma > 0:
        # noise in slabs to bound host memory
        step = max(1, (1 << 24) // C)
        for r0 in range(0, R, step):
            r1 = min(R, r0 + step)
            nz = rng.standard_normal(size=(r1 - r0, C, 2))
            re[r0:r1] += sigma * nz[..., 0]
            im[r0:r1] += sigma * nz[..., 1]
    vis = np.empty((R, C), dtype=np.complex128)
    vis.real = re
    vis.imag = im
    if vis_dtype == "c64":
        vis = vis.astype(np.complex64)
    return Workload(name=name, uvw_m=uvw, freq_hz=np.asarray(freq, dtype=np.float64),
                    vis=vis, weights=None, sources=src, **img)


# ----------------------------------------------------------------------------
# the five BASELINE.json configs (+ scaled-down variants for parity tests)
# ----------------------------------------------------------------------------

def make_config(cfg: int, device: str = "cpu", n_times: Optional[int] = None,
                n: Optional[int] = None, n_chan: Optional[int] = None,
                n_wplanes: Optional[int] = None, n_src: Optional[int] = None,
                with_weights: bool = False, seed: Optional[int] = None) -> Workload:
    """Build config ``cfg`` (1..5).  ``n_times`` / ``n`` / ``n_chan`` /
    ``n_wplanes`` / ``n_src`` override the full-size values to obtain a
    scaled-down case with the same structure (the pixel scale is kept, so the
    grid's half-extent 1/(2 dl) in wavelengths -- and with it the fraction of the
    grid the uv coverage fills -- is that of the full-size config; the field of
    view, and the box the sources are drawn in, shrink with ``n``)."""
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + cfg if seed is None else seed))
    if cfg == 1:
        N = n or 256
        ant = _antennas_disc(rng, 16, 2000.0)
        ns = n_src or 5
        dl = 0.5 * DEG / 256
        field = N * dl
        src = np.stack([rng.uniform(-field / 2, field / 2, ns),
                        rng.uniform(-field / 2, field / 2, ns),
                        rng.uniform(0.1, 1.0, ns)], axis=1)
        # one source snapped to a pixel centre in the inner half (closed-form pin)
        src[0, 0] = 20 * dl
        src[0, 1] = -37 * dl
        wl = _finish("cfg1_tiny", rng, ant, -30.0, -30.0, -1.0, 1.0, n_times or 32,
                     np.array([1.4e9]) if not n_chan else np.linspace(1.3e9, 1.5e9, n_chan),
                     src, 0.01, "c128", device,
                     n=N, n_wplanes=n_wplanes or 8, support=7, pixel_rad=dl,
                     grid_prec="f64", cube=0, plane_batch=0)
    elif cfg in (2, 4, 5):
        ant = _antennas_core_outer(rng, 48, 300.0, 16, 1000.0, 4000.0, 8000.0)
        if cfg == 2:
            N0, T0, C0_, Nw0, dl0, prec, cube, pb = 4096, 512, 16, 32, 2.0 * ARCSEC, "f64", 0, 0
        elif cfg == 4:
            N0, T0, C0_, Nw0, dl0, prec, cube, pb = 16384, 2048, 16, 32, 0.5 * ARCSEC, "f32", 0, 8
        else:
            N0, T0, C0_, Nw0, dl0, prec, cube, pb = 4096, 256, 128, 16, 2.0 * ARCSEC, "f64", 1, 0
        N = n or N0
        dl = dl0
        ns = n_src or 200
        C = n_chan or C0_
        freq = np.linspace(856e6, 1712e6, C)
        half = N * dl / 4.0                       # sources in the inner half
        src = np.stack([rng.uniform(-half, half, ns), rng.uniform(-half, half, ns),
                        _powerlaw_flux(rng, ns, 1e-3, 1.0)], axis=1)
        wl = _finish({2: "cfg2_meerkat", 4: "cfg4_largepix", 5: "cfg5_cube"}[cfg], rng, ant,
                     -30.7, -30.0, -2.0, 2.0, n_times or T0, freq, src, 0.01, "c64", device,
                     n=N, n_wplanes=n_wplanes or Nw0, support=7, pixel_rad=dl,
                     grid_prec=prec, cube=cube, plane_batch=pb)
    elif cfg == 3:
        ant = _antennas_core_outer(rng, 40, 1000.0, 20, 5000.0, 50000.0, 100000.0)
        N = n or 8192
        dl = 5.0 * DEG / 8192
        ns = n_src or 500
        C = n_chan or 8
        freq = np.linspace(120e6, 168e6, C)
        half = N * dl / 2.0 * 0.98
        src = np.stack([rng.uniform(-half, half, ns), rng.uniform(-half, half, ns),
                        _powerlaw_flux(rng, ns, 1e-3, 1.0)], axis=1)
        wl = _finish("cfg3_lofar", rng, ant, 52.9, 48.0, -4.0, 4.0, n_times or 1024, freq,
                     src, 0.01, "c64", device,
                     n=N, n_wplanes=n_wplanes or 64, support=7, pixel_rad=dl,
                     grid_prec="f64", cube=0, plane_batch=0)
    else:
        raise ValueError(f"unknown config {cfg}")
    if with_weights:
        wl.weights = rng.uniform(0.25, 1.75, size=wl.vis.shape).astype(np.float32)
    return wl


def unit_vis(wl: Workload) -> Workload:
    """Same geometry, V = 1 everywhere (unit point source at the phase centre)."""
    out = dataclasses.replace(wl)
    out.vis = np.ones_like(wl.vis)
    return out
