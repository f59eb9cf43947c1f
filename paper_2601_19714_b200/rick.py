"""Thin Python binding of librick_b200 (include/rick.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; torch is used for
device memory and streams.  There is no CPU fallback: if the shared library is missing
or no CUDA device is present, the calls fail loudly.
"""
from __future__ import annotations

import ctypes as C
import math
import os
from typing import Optional

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "librick_b200.so")

RICK_OK, RICK_ERR_INVALID, RICK_ERR_STATE, RICK_ERR_CUDA, RICK_ERR_OOM = 0, -1, -2, -3, -4
RICK_GRID_F64, RICK_GRID_F32 = 0, 1
RICK_VIS_C64, RICK_VIS_C128 = 0, 1
RICK_FLAG_FOLD_W = 1
RICK_NOALLOC_MAX_PLANES, RICK_NOALLOC_MAX_CHAN, RICK_NOALLOC_SCRATCH_BYTES = 4096, 1024, 41216

EXPORTS = ["rick_plan", "rick_plan_destroy", "rick_grid", "rick_fft_wplanes",
           "rick_wcorrect_accumulate", "rick_gridcorrect", "rick_image", "rick_image_host",
           "rick_image_stream_host", "rick_plane_histogram", "rick_plane_histogram_noalloc", "rick_partition_planes",
           "rick_get_image", "rick_get_stats", "rick_last_error", "rick_debug_items",
           "rick_debug_planes", "rick_version", "rick_profile",
           "rick_profile_read", "rick_kernel_name"]


class PlanDesc(C.Structure):
    _fields_ = [("n", C.c_int32), ("n_wplanes", C.c_int32), ("support", C.c_int32),
                ("pixel_rad", C.c_double), ("kb_beta", C.c_double), ("grid_prec", C.c_int32),
                ("tile", C.c_int32), ("plane_batch", C.c_int32), ("cube", C.c_int32),
                ("flags", C.c_int32), ("w_min", C.c_double), ("w_max", C.c_double),
                ("z_begin", C.c_int32), ("z_count", C.c_int32)]


class Stats(C.Structure):
    _fields_ = [("n_vis", C.c_int64), ("n_gridded", C.c_int64), ("n_dropped", C.c_int64),
                ("sum_w", C.c_double), ("w_min", C.c_double), ("w_max", C.c_double),
                ("n_launches", C.c_int64), ("occ_rows", C.c_int64), ("occ_tiles", C.c_int64),
                ("n_planes", C.c_int64), ("occ_windows", C.c_int64)]


class RickError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"librick_b200 error {code}: {msg}")
        self.code = code


_lib = None


def load_library():
    """Load librick_b200.so (built in-tree by paper_2601_19714_b200/build.py)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2601_19714_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    L.rick_plan.argtypes = [C.POINTER(vp), C.POINTER(PlanDesc), vp]
    L.rick_plan_destroy.argtypes = [vp]
    L.rick_grid.argtypes = [vp, vp, i32, vp, vp, C.POINTER(C.c_double), i32, i64]
    L.rick_fft_wplanes.argtypes = [vp]
    L.rick_wcorrect_accumulate.argtypes = [vp]
    L.rick_gridcorrect.argtypes = [vp]
    L.rick_image.argtypes = [vp, vp, i32, vp, vp, C.POINTER(C.c_double), i32, i64, vp]
    L.rick_image_host.argtypes = [vp, vp, i32, vp, vp, C.POINTER(C.c_double), i32, i64, vp]
    L.rick_image_stream_host.argtypes = [vp, vp, i32, vp, vp, C.POINTER(C.c_double), i32, i64, i64, vp]
    L.rick_plane_histogram.argtypes = [vp, vp, C.POINTER(C.c_double), i32, i64, C.POINTER(C.c_int64)]
    L.rick_plane_histogram_noalloc.argtypes = [vp, vp, C.POINTER(C.c_double), i32, i64, C.POINTER(C.c_int64)]
    L.rick_partition_planes.argtypes = [C.POINTER(C.c_int64), i32, i32, C.c_double, C.POINTER(i32)]
    L.rick_get_image.argtypes = [vp, vp]
    L.rick_get_stats.argtypes = [vp, C.POINTER(Stats)]
    L.rick_last_error.argtypes = [vp]
    L.rick_last_error.restype = C.c_char_p
    L.rick_debug_items.argtypes = [vp, i32, C.POINTER(i32), C.POINTER(i32)]
    L.rick_debug_items.restype = vp
    L.rick_debug_planes.argtypes = [vp]
    L.rick_debug_planes.restype = vp
    L.rick_version.restype = C.c_char_p
    L.rick_profile.argtypes = [vp, i32]
    L.rick_profile_read.argtypes = [vp, i32, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
    L.rick_kernel_name.argtypes = [i32]
    L.rick_kernel_name.restype = C.c_char_p
    for name in EXPORTS:
        getattr(L, name)
    _lib = L
    return L


def _dev_ptr(t: Optional[torch.Tensor]):
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous()
    return C.c_void_p(t.data_ptr())


class Plan:
    """rick_plan + the staged calls.  Tensors are torch CUDA tensors unless noted."""

    def __init__(self, n, n_wplanes, support, pixel_rad, kb_beta=0.0, grid_prec="f64", tile=0,
                 plane_batch=0, cube=0, w_min=float("nan"), w_max=float("nan"), stream=None, flags=0,
                 z_begin=0, z_count=0):
        self._lib = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("librick_b200 needs a CUDA device (no CPU fallback)")
        self.desc = PlanDesc(int(n), int(n_wplanes), int(support), float(pixel_rad), float(kb_beta),
                             RICK_GRID_F32 if grid_prec in ("f32", RICK_GRID_F32) else RICK_GRID_F64,
                             int(tile), int(plane_batch), int(cube), int(flags), float(w_min), float(w_max),
                             int(z_begin), int(z_count))
        self.n, self.n_wplanes, self.cube = int(n), int(n_wplanes), int(cube)
        self.n_planes_resident = int(z_count) if z_count else int(n_wplanes)
        self.f32 = self.desc.grid_prec == RICK_GRID_F32
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        self._h = C.c_void_p()
        rc = self._lib.rick_plan(C.byref(self._h), C.byref(self.desc), C.c_void_p(self.stream.cuda_stream))
        if rc != RICK_OK:
            self._h = C.c_void_p()
            raise RickError(rc, "rick_plan failed (bad descriptor, no device, or out of memory)")
        self._keep = None
        self._n_vis = 0

    # -- helpers ---------------------------------------------------------------------------
    def _check(self, rc):
        if rc != RICK_OK:
            raise RickError(rc, self._lib.rick_last_error(self._h).decode())

    @staticmethod
    def _vis_dtype(vis: torch.Tensor) -> int:
        if vis.dtype == torch.complex64:
            return RICK_VIS_C64
        if vis.dtype == torch.complex128:
            return RICK_VIS_C128
        raise TypeError("vis must be complex64 or complex128")

    def _marshal(self, vis, uvw_m, weights, chan_freq_hz):
        freq = np.ascontiguousarray(chan_freq_hz, dtype=np.float64)
        n_chan = int(freq.shape[0])
        n_rows = int(uvw_m.shape[0])
        assert vis.numel() == n_rows * n_chan
        assert uvw_m.dtype == torch.float64 and (weights is None or weights.dtype == torch.float32)
        self._keep = (vis, uvw_m, weights, freq)        # borrowed until the stream work is done
        self._n_vis = n_rows * n_chan
        return freq.ctypes.data_as(C.POINTER(C.c_double)), n_chan, n_rows

    # -- C ABI, same names -----------------------------------------------------------------
    def rick_grid(self, vis, uvw_m, weights, chan_freq_hz):
        fp, n_chan, n_rows = self._marshal(vis, uvw_m, weights, chan_freq_hz)
        self._check(self._lib.rick_grid(self._h, _dev_ptr(vis), self._vis_dtype(vis), _dev_ptr(uvw_m),
                                        _dev_ptr(weights), fp, n_chan, n_rows))

    def rick_fft_wplanes(self):
        self._check(self._lib.rick_fft_wplanes(self._h))

    def rick_wcorrect_accumulate(self):
        self._check(self._lib.rick_wcorrect_accumulate(self._h))

    def rick_gridcorrect(self):
        self._check(self._lib.rick_gridcorrect(self._h))

    def rick_image(self, vis, uvw_m, weights, chan_freq_hz, image_out: Optional[torch.Tensor] = None):
        fp, n_chan, n_rows = self._marshal(vis, uvw_m, weights, chan_freq_hz)
        if image_out is None:
            shape = (n_chan, self.n, self.n) if self.cube else (self.n, self.n)
            image_out = torch.empty(shape, dtype=torch.float64, device=vis.device)
        assert image_out.dtype == torch.float64 and image_out.is_cuda and image_out.is_contiguous()
        need = (n_chan if self.cube else 1) * self.n * self.n
        if image_out.numel() != need:      # the C ABI cannot see the buffer's size: check it here
            raise ValueError(f"image_out has {image_out.numel()} elements, this plan writes {need}")
        self._check(self._lib.rick_image(self._h, _dev_ptr(vis), self._vis_dtype(vis), _dev_ptr(uvw_m),
                                         _dev_ptr(weights), fp, n_chan, n_rows, _dev_ptr(image_out)))
        return image_out

    def rick_image_host(self, vis, uvw_m, weights, chan_freq_hz, image_out):
        """All buffers HOST (torch CPU tensors, ideally pinned); synchronises."""
        freq = np.ascontiguousarray(chan_freq_hz, dtype=np.float64)
        n_chan, n_rows = int(freq.shape[0]), int(uvw_m.shape[0])
        for t in (vis, uvw_m, image_out) + (() if weights is None else (weights,)):
            assert (not t.is_cuda) and t.is_contiguous()
        self._n_vis = n_rows * n_chan
        need = (n_chan if self.cube else 1) * self.n * self.n
        if image_out.numel() != need or image_out.dtype != torch.float64:
            raise ValueError(f"image_out must hold {need} float64 values")
        self._check(self._lib.rick_image_host(
            self._h, C.c_void_p(vis.data_ptr()), self._vis_dtype(vis), C.c_void_p(uvw_m.data_ptr()),
            None if weights is None else C.c_void_p(weights.data_ptr()),
            freq.ctypes.data_as(C.POINTER(C.c_double)), n_chan, n_rows, C.c_void_p(image_out.data_ptr())))
        return image_out

    def rick_image_stream_host(self, vis, uvw_m, weights, chan_freq_hz, image_out, rows_per_chunk: int):
        """Out-of-core visibilities: all buffers HOST; the visibilities cross in chunks of rows; synchronises."""
        freq = np.ascontiguousarray(chan_freq_hz, dtype=np.float64)
        n_chan, n_rows = int(freq.shape[0]), int(uvw_m.shape[0])
        for t in (vis, uvw_m, image_out) + (() if weights is None else (weights,)):
            assert (not t.is_cuda) and t.is_contiguous()
        self._n_vis = n_rows * n_chan
        if image_out.numel() != self.n * self.n or image_out.dtype != torch.float64:
            raise ValueError(f"image_out must hold {self.n * self.n} float64 values")
        self._check(self._lib.rick_image_stream_host(
            self._h, C.c_void_p(vis.data_ptr()), self._vis_dtype(vis), C.c_void_p(uvw_m.data_ptr()),
            None if weights is None else C.c_void_p(weights.data_ptr()),
            freq.ctypes.data_as(C.POINTER(C.c_double)), n_chan, n_rows, int(rows_per_chunk),
            C.c_void_p(image_out.data_ptr())))
        return image_out

    def rick_plane_histogram(self, uvw_m, chan_freq_hz) -> np.ndarray:
        """[n_wplanes] int64: on-grid visibilities per w-plane of the whole problem (synchronises)."""
        freq = np.ascontiguousarray(chan_freq_hz, dtype=np.float64)
        hist = np.zeros(self.n_wplanes, np.int64)
        self._keep = (uvw_m, freq)
        self._check(self._lib.rick_plane_histogram(self._h, _dev_ptr(uvw_m), freq.ctypes.data_as(C.POINTER(C.c_double)),
                                                   int(freq.shape[0]), int(uvw_m.shape[0]),
                                                   hist.ctypes.data_as(C.POINTER(C.c_int64))))
        return hist

    def rick_plane_histogram_noalloc(self, uvw_m, chan_freq_hz, hist=None) -> np.ndarray:
        """rick_plane_histogram without any device allocation inside the call (fixed scratch array in the library:
        at most RICK_NOALLOC_MAX_PLANES planes and RICK_NOALLOC_MAX_CHAN channels; calls that overlap on the GPU
        race).  `hist`: optional caller-owned [n_wplanes] int64 array to fill."""
        freq = np.ascontiguousarray(chan_freq_hz, dtype=np.float64)
        if hist is None:
            hist = np.zeros(self.n_wplanes, np.int64)
        assert hist.dtype == np.int64 and hist.flags.c_contiguous and hist.shape == (self.n_wplanes,)
        self._keep = (uvw_m, freq)
        self._check(self._lib.rick_plane_histogram_noalloc(self._h, _dev_ptr(uvw_m), freq.ctypes.data_as(C.POINTER(C.c_double)),
                                                           int(freq.shape[0]), int(uvw_m.shape[0]),
                                                           hist.ctypes.data_as(C.POINTER(C.c_int64))))
        return hist

    def rick_get_image(self) -> torch.Tensor:
        out = torch.empty((self.n, self.n), dtype=torch.float64, device="cuda")
        self._check(self._lib.rick_get_image(self._h, _dev_ptr(out)))
        return out

    def rick_get_stats(self) -> dict:
        s = Stats()
        self._check(self._lib.rick_get_stats(self._h, C.byref(s)))
        return {k: getattr(s, k) for k, _ in Stats._fields_}

    def rick_profile(self, enable: bool):
        self._check(self._lib.rick_profile(self._h, 1 if enable else 0))

    def rick_profile_read(self) -> dict:
        """{kernel name: (total_ms, launches)} since profiling was enabled (synchronises)."""
        out, i = {}, 0
        while True:
            name = self._lib.rick_kernel_name(i)
            if name is None:
                return out
            ms, n = C.c_double(), C.c_int64()
            self._check(self._lib.rick_profile_read(self._h, i, C.byref(ms), C.byref(n)))
            out[name.decode()] = (ms.value, n.value)
            i += 1

    # -- debug accessors (copies, synchronising) -------------------------------------------
    def _copy_from(self, ptr, nbytes, dtype, shape):
        if not ptr:
            return None
        typestr = {torch.int64: "<i8", torch.complex64: "<c8", torch.complex128: "<c16"}[dtype]

        class _View:            # zero-copy view of plan-owned device memory
            __cuda_array_interface__ = {"shape": tuple(shape), "typestr": typestr,
                                        "data": (int(ptr), False), "version": 2}
        self.stream.synchronize()
        out = torch.as_tensor(_View(), device="cuda").clone()
        assert out.numel() * out.element_size() == nbytes
        return out

    def debug_items(self, sorted_: bool):
        """(items int64 CUDA tensor [M], idx_bits, key_bits): rick_debug_items (copy, synchronising)."""
        m = self._n_vis
        ib, kb = C.c_int32(), C.c_int32()
        ptr = self._lib.rick_debug_items(self._h, 1 if sorted_ else 0, C.byref(ib), C.byref(kb))
        if not m:
            return torch.empty(0, dtype=torch.int64, device="cuda"), ib.value, kb.value
        return self._copy_from(ptr, 8 * m, torch.int64, (m,)), ib.value, kb.value

    def debug_keys(self) -> np.ndarray:
        """[M] uint64 keys in visibility order; a dropped visibility reads as all ones (64 bits)."""
        items, ib, kb = self.debug_items(False)
        it = items.cpu().numpy().view(np.uint64)
        assert np.array_equal(it & np.uint64((1 << ib) - 1), np.arange(it.shape[0], dtype=np.uint64))
        key = it >> np.uint64(ib)
        key[key == np.uint64((1 << kb) - 1)] = np.uint64(0xFFFFFFFFFFFFFFFF)
        return key

    def debug_perm(self) -> np.ndarray:
        """[M] uint32: visibility index at every sorted position."""
        items, ib, _ = self.debug_items(True)
        return (items.cpu().numpy().view(np.uint64) & np.uint64((1 << ib) - 1)).astype(np.uint32)

    def debug_planes(self) -> Optional[torch.Tensor]:
        dt = torch.complex64 if self.f32 else torch.complex128
        nz = self.n_planes_resident
        nb = (8 if self.f32 else 16) * nz * self.n * self.n
        return self._copy_from(self._lib.rick_debug_planes(self._h), nb, dt, (nz, self.n, self.n))

    def destroy(self):
        if getattr(self, "_h", None) and self._h.value:
            self._lib.rick_plan_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def rick_partition_planes(hist, n_parts: int, plane_cost: float) -> np.ndarray:
    """[n_parts + 1] int32 bounds of contiguous plane ranges with the smallest largest cost (host arithmetic of
    the library; needs no device)."""
    h = np.ascontiguousarray(hist, dtype=np.int64)
    bounds = np.zeros(int(n_parts) + 1, np.int32)
    rc = load_library().rick_partition_planes(h.ctypes.data_as(C.POINTER(C.c_int64)), int(h.shape[0]), int(n_parts),
                                              float(plane_cost), bounds.ctypes.data_as(C.POINTER(C.c_int32)))
    if rc != RICK_OK:
        raise RickError(rc, "rick_partition_planes: bad arguments")
    return bounds


def version() -> str:
    return load_library().rick_version().decode()


def plan_from_workload(wl, **over) -> Plan:
    """Plan with the imaging parameters of a synth.Workload."""
    kw = dict(n=wl.n, n_wplanes=wl.n_wplanes, support=wl.support, pixel_rad=wl.pixel_rad,
              grid_prec=wl.grid_prec, plane_batch=wl.plane_batch, cube=wl.cube)
    kw.update(over)
    return Plan(**kw)


def to_device(wl, device="cuda"):
    """(vis, uvw_m, weights) of a synth.Workload as CUDA tensors."""
    vis = torch.from_numpy(np.ascontiguousarray(wl.vis)).to(device)
    uvw = torch.from_numpy(np.ascontiguousarray(wl.uvw_m)).to(device)
    wgt = None if wl.weights is None else torch.from_numpy(np.ascontiguousarray(wl.weights)).to(device)
    return vis, uvw, wgt
