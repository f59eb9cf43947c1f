"""ctypes loader for the CPU oracle (``rick_oracle.c``).  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_2601_19714_b200`` and the product never imports it.

All arrays are numpy, fp64 (visibilities are widened exactly to complex128).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import time

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rick_oracle.c")
_LIB = os.path.join(_HERE, "librick_oracle.so")
_lib = None

_f64p = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_i32p = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
_u32p = np.ctypeslib.ndpointer(dtype=np.uint32, flags="C_CONTIGUOUS")
_u64p = np.ctypeslib.ndpointer(dtype=np.uint64, flags="C_CONTIGUOUS")
_i64p = np.ctypeslib.ndpointer(dtype=np.int64, flags="C_CONTIGUOUS")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.rko_bessel_i0.restype = C.c_double
        L.rko_bessel_i0.argtypes = [C.c_double]
        L.rko_kb.restype = C.c_double
        L.rko_kb.argtypes = [C.c_double, C.c_int, C.c_double]
        L.rko_taper.restype = C.c_double
        L.rko_taper.argtypes = [C.c_double, C.c_int, C.c_double]
        L.rko_num_threads.restype = C.c_int
        L.rko_fft2_centered.argtypes = [_f64p, C.c_int32]
        L.rko_sort.argtypes = [C.c_int64, _u64p, _u32p]
        L.rko_wcorrect_accumulate.argtypes = [_f64p, C.c_int32, C.c_double, C.c_double, _f64p]
        L.rko_gridcorrect.argtypes = [_f64p, C.c_int32, C.c_int32, C.c_double]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().rko_num_threads())


def bessel_i0(x: float) -> float:
    return float(lib().rko_bessel_i0(float(x)))


def kb(t: float, S: int, beta: float) -> float:
    return float(lib().rko_kb(float(t), int(S), float(beta)))


def taper(nu: float, S: int, beta: float) -> float:
    return float(lib().rko_taper(float(nu), int(S), float(beta)))


def _vis128(vis) -> np.ndarray:
    v = np.ascontiguousarray(np.asarray(vis).astype(np.complex128, copy=False)).reshape(-1)
    return v.view(np.float64)


def _ptr(a, ctype):
    return a.ctypes.data_as(C.POINTER(ctype)) if a is not None else None


def index(uvw_m, freq_hz, N, Nw, S, dl, B, cube=0, w_min=float("nan"), w_max=float("nan")):
    """Steps 1-4.  Returns dict(iu, iv, ip, key (uint64; all ones = dropped), xu, xv,
    w_min[n_img], w_max[n_img])."""
    uvw = np.ascontiguousarray(uvw_m, dtype=np.float64)
    fr = np.ascontiguousarray(freq_hz, dtype=np.float64)
    R, Cn = uvw.shape[0], fr.shape[0]
    M = R * Cn
    n_img = Cn if cube else 1
    out = dict(iu=np.empty(M, np.int32), iv=np.empty(M, np.int32), ip=np.empty(M, np.int32),
               key=np.empty(M, np.uint64), xu=np.empty(M, np.float64), xv=np.empty(M, np.float64),
               w_min=np.full(n_img, w_min, np.float64), w_max=np.full(n_img, w_max, np.float64))
    L = lib()
    L.rko_index(C.c_int64(R), C.c_int32(Cn), _ptr(uvw, C.c_double), _ptr(fr, C.c_double),
                C.c_int32(N), C.c_int32(Nw), C.c_int32(S), C.c_double(dl), C.c_int32(B),
                C.c_int32(cube), _ptr(out["w_min"], C.c_double), _ptr(out["w_max"], C.c_double),
                _ptr(out["iu"], C.c_int32), _ptr(out["iv"], C.c_int32), _ptr(out["ip"], C.c_int32),
                _ptr(out["key"], C.c_uint64), _ptr(out["xu"], C.c_double), _ptr(out["xv"], C.c_double))
    return out


def fold_w(uvw_m, vis):
    """Reading R24: rows with w < 0 -> (-u, -v, -w) and conjugated visibilities.  Returns fresh arrays
    (uvw [R][3] float64, vis [R][C] complex128) and the number of rows folded."""
    uvw = np.array(uvw_m, dtype=np.float64, order="C", copy=True)
    v = np.array(np.asarray(vis).astype(np.complex128), order="C", copy=True).reshape(uvw.shape[0], -1)
    L = lib()
    L.rko_fold_w.restype = C.c_int64
    n = L.rko_fold_w(C.c_int64(uvw.shape[0]), C.c_int32(v.shape[1]), _ptr(uvw, C.c_double),
                     _ptr(v.view(np.float64), C.c_double))
    return uvw, v, int(n)


def sort(key) -> np.ndarray:
    key = np.ascontiguousarray(key, dtype=np.uint64)
    perm = np.empty(key.shape[0], np.uint32)
    lib().rko_sort(key.shape[0], key, perm)
    return perm


def grid_plane(list_idx, vis, wgt, iu, iv, xu, xv, N, S, beta) -> np.ndarray:
    """Steps 5-6 for the visibilities in list_idx, onto one zeroed plane [N][N] complex128."""
    lst = np.ascontiguousarray(list_idx, dtype=np.int64)
    plane = np.zeros((N, N), np.complex128)
    v = _vis128(vis)
    w = None if wgt is None else np.ascontiguousarray(wgt, dtype=np.float32).reshape(-1)
    lib().rko_grid_plane(C.c_int64(lst.shape[0]), _ptr(lst, C.c_int64), _ptr(v, C.c_double),
                         _ptr(w, C.c_float), _ptr(iu, C.c_int32), _ptr(iv, C.c_int32),
                         _ptr(xu, C.c_double), _ptr(xv, C.c_double), C.c_int32(N), C.c_int32(S),
                         C.c_double(beta), _ptr(plane.view(np.float64), C.c_double))
    return plane


def fft2_centered(plane) -> np.ndarray:
    """Step 7 on a copy of plane [N][N] complex128."""
    p = np.array(plane, dtype=np.complex128, order="C", copy=True)
    rc = lib().rko_fft2_centered(p.view(np.float64).reshape(-1), p.shape[0])
    if rc != 0:
        raise ValueError("N must be a power of two, multiple of 4")
    return p


def wcorrect_accumulate(plane, dl, w_z, image=None) -> np.ndarray:
    p = np.ascontiguousarray(plane, dtype=np.complex128)
    N = p.shape[0]
    img = np.zeros((N, N), np.float64) if image is None else image
    lib().rko_wcorrect_accumulate(p.view(np.float64).reshape(-1), N, float(dl), float(w_z), img.reshape(-1))
    return img


def gridcorrect(image, S, beta) -> np.ndarray:
    img = np.array(image, dtype=np.float64, order="C", copy=True)
    lib().rko_gridcorrect(img.reshape(-1), img.shape[0], int(S), float(beta))
    return img


def image(uvw_m, freq_hz, vis, wgt, N, Nw, S, dl, beta=0.0, B=16, cube=0,
          w_min=float("nan"), w_max=float("nan"), stages=15, want_stacks=False, want_raw=False, fold=False):
    """Whole path a0..a6 (plane-streamed).  Returns dict(image [n_img][N][N] (squeezed when
    n_img == 1), stats, timings, and optionally stack_grid / stack_fft / raw_image).
    fold: reading R24, the rows with w < 0 are folded onto w > 0 first (fold_w)."""
    if fold:
        uvw_m, vis, _ = fold_w(uvw_m, vis)
    uvw = np.ascontiguousarray(uvw_m, dtype=np.float64)
    fr = np.ascontiguousarray(freq_hz, dtype=np.float64)
    R, Cn = uvw.shape[0], fr.shape[0]
    n_img = Cn if cube else 1
    v = _vis128(vis)
    assert v.shape[0] == 2 * R * Cn
    w = None if wgt is None else np.ascontiguousarray(wgt, dtype=np.float32).reshape(-1)
    img = np.zeros((n_img, N, N), np.float64)
    raw = np.zeros((n_img, N, N), np.float64) if want_raw else None
    sg = np.zeros((n_img * Nw, N, N), np.complex128) if want_stacks else None
    sf = np.zeros((n_img * Nw, N, N), np.complex128) if want_stacks else None
    stats = np.zeros(6, np.float64)
    tim = np.zeros(4, np.float64)
    t0 = time.perf_counter()
    rc = lib().rko_image(C.c_int64(R), C.c_int32(Cn), _ptr(uvw, C.c_double), _ptr(fr, C.c_double),
                         _ptr(v, C.c_double), _ptr(w, C.c_float), C.c_int32(N), C.c_int32(Nw),
                         C.c_int32(S), C.c_double(dl), C.c_double(beta), C.c_int32(B), C.c_int32(cube),
                         C.c_double(w_min), C.c_double(w_max), C.c_int32(stages),
                         _ptr(img, C.c_double), _ptr(raw, C.c_double),
                         _ptr(None if sg is None else sg.view(np.float64), C.c_double),
                         _ptr(None if sf is None else sf.view(np.float64), C.c_double),
                         _ptr(stats, C.c_double), _ptr(tim, C.c_double))
    assert rc == 0
    out = dict(image=img[0] if n_img == 1 else img,
               stats=dict(n_vis=int(stats[0]), n_gridded=int(stats[1]), n_dropped=int(stats[2]),
                          sum_w=float(stats[3]), w_min=float(stats[4]), w_max=float(stats[5])),
               timings=dict(grid=float(tim[0]), fft=float(tim[1]), wcorrect=float(tim[2]),
                            taper=float(tim[3]), total=time.perf_counter() - t0))
    if want_stacks:
        out["stack_grid"], out["stack_fft"] = sg, sf
    if want_raw:
        out["raw_image"] = raw[0] if n_img == 1 else raw
    return out


def dft(u_l, v_l, w_l, vis, wgt, keep, N, dl) -> np.ndarray:
    """Direct DFT image (plain definition).  u_l, v_l, w_l in wavelengths, [M]."""
    u = np.ascontiguousarray(u_l, dtype=np.float64).reshape(-1)
    vv = np.ascontiguousarray(v_l, dtype=np.float64).reshape(-1)
    ww = np.ascontiguousarray(w_l, dtype=np.float64).reshape(-1)
    v = _vis128(vis)
    w = None if wgt is None else np.ascontiguousarray(wgt, dtype=np.float32).reshape(-1)
    kp = None if keep is None else np.ascontiguousarray(keep, dtype=np.uint8).reshape(-1)
    img = np.zeros((N, N), np.float64)
    lib().rko_dft(C.c_int64(u.shape[0]), _ptr(u, C.c_double), _ptr(vv, C.c_double),
                  _ptr(ww, C.c_double), _ptr(v, C.c_double), _ptr(w, C.c_float),
                  _ptr(kp, C.c_uint8), C.c_int32(N), C.c_double(dl), _ptr(img, C.c_double))
    return img
