"""Thin Python binding over the C-ABI of include/hcgrid.h (libhcgrid.so).

Argument marshalling only: every step of the path (pixelise, sort, tables, pack, convolve)
runs in the library's CUDA kernels.  torch is used for device memory and streams.  There
is no CPU fallback: if the library cannot be built or loaded, or a call fails, an
HCGridError is raised.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libhcgrid.so")
_lib = None

F32, F64 = 0, 1
OPT_PROFILE, OPT_SUBPIX_BITS, OPT_COARSEN, OPT_KERNEL, OPT_WARPS_PER_SM, OPT_COARSEN_Y, OPT_SPLIT, OPT_PREORDER = 1, 2, 3, 4, 5, 6, 7, 8
OPT_HOST_CHUNKS = 9
OPT_CELLS_AS_GRID = 10
OPT_GRAPH = 11
PREORDER_AUTO, PREORDER_RADIX, PREORDER_COUNTING = 0, 1, 2
KERNEL_AUTO, KERNEL_SIMPLE, KERNEL_F64PAIR, KERNEL_GENERAL, KERNEL_STAGED, KERNEL_TILE, KERNEL_CUBE, KERNEL_CUBE_TC = 0, 1, 2, 3, 4, 5, 6, 7

EXPORTS = [
    "hcgrid_create", "hcgrid_destroy", "hcgrid_set_option", "hcgrid_set_target_car",
    "hcgrid_set_target_cells", "hcgrid_grid", "hcgrid_grid_host", "hcgrid_ncell",
    "hcgrid_get_stats", "hcgrid_last_error", "hcgrid_debug_preorder",
    "hcgrid_debug_ang2pix_ring", "hcgrid_host_ang2pix_ring", "hcgrid_host_ring_info",
    "hcgrid_measure_peaks", "hcgrid_accumulate", "hcgrid_finalize", "hcgrid_accumulated_batches",
    "hcgrid_set_kernel", "hcgrid_count_hits_static", "hcgrid_static_max_cells",
]
KERNEL_GAUSS, KERNEL_TAPERED_SINC, KERNEL_ELLIPTICAL_GAUSS = 0, 1, 2          # hcgrid_set_kernel types


class HCGridError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"hcgrid status {status}: {message}")
        self.status = status


class Stats(ctypes.Structure):
    _fields_ = [("n_samples", ctypes.c_int64), ("n_kept", ctypes.c_int64), ("n_bins", ctypes.c_int64),
                ("n_rings", ctypes.c_int32), ("subpix_bits", ctypes.c_int32), ("coarsen", ctypes.c_int32),
                ("kernel", ctypes.c_int32), ("gpu_launches", ctypes.c_int32), ("coarsen_y", ctypes.c_int32),
                ("us_pixelise", ctypes.c_float), ("us_sort", ctypes.c_float), ("us_tables", ctypes.c_float),
                ("us_pack", ctypes.c_float), ("us_convolve", ctypes.c_float), ("us_total", ctypes.c_float),
                ("split", ctypes.c_int32), ("preorder", ctypes.c_int32),
                ("n_hit", ctypes.c_int64), ("graph", ctypes.c_int32), ("pad_", ctypes.c_int32),
                ("n_pairs_tested", ctypes.c_int64)]

    def asdict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


def load_library():
    """Load libhcgrid.so, building it in-tree with nvcc first if it is missing or stale.
    Raises if it cannot be built: the product path has no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    from . import build as _build
    try:
        path = _build.build()
    except Exception as exc:  # stale but present library and no nvcc: still refuse silently-old code
        if not os.path.exists(_LIB_PATH):
            raise HCGridError(-4, f"libhcgrid.so is missing and could not be built: {exc}") from exc
        raise
    lib = ctypes.CDLL(path)
    vp, i64, i32, dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_double
    lib.hcgrid_create.argtypes = [ctypes.POINTER(vp), dbl, dbl, i64, ctypes.c_int, ctypes.c_int]
    lib.hcgrid_destroy.argtypes = [vp]
    lib.hcgrid_set_option.argtypes = [vp, ctypes.c_int, i64]
    lib.hcgrid_set_kernel.argtypes = [vp, ctypes.c_int32, ctypes.c_double, ctypes.c_double]
    lib.hcgrid_set_target_car.argtypes = [vp, i32, i32, dbl, dbl, dbl, dbl]
    lib.hcgrid_set_target_cells.argtypes = [vp, i64, vp, vp, vp]
    lib.hcgrid_grid.argtypes = [vp, i64, vp, vp, vp, i32, vp, vp, vp, vp, vp]
    lib.hcgrid_grid_host.argtypes = [vp, i64, vp, vp, vp, i32, vp, vp, vp, vp]
    lib.hcgrid_accumulate.argtypes = [vp, i64, vp, vp, vp, i32, vp, vp]
    lib.hcgrid_finalize.argtypes = [vp, vp, vp, vp, ctypes.c_int, vp]
    lib.hcgrid_accumulated_batches.argtypes = [vp]
    lib.hcgrid_accumulated_batches.restype = i64
    lib.hcgrid_ncell.argtypes = [vp]
    lib.hcgrid_ncell.restype = i64
    lib.hcgrid_get_stats.argtypes = [vp, ctypes.POINTER(Stats)]
    lib.hcgrid_last_error.argtypes = [vp]
    lib.hcgrid_last_error.restype = ctypes.c_char_p
    lib.hcgrid_debug_preorder.argtypes = [vp, vp, vp, ctypes.POINTER(i32), vp]
    lib.hcgrid_debug_ang2pix_ring.argtypes = [i64, i64, vp, vp, vp, vp]
    lib.hcgrid_host_ang2pix_ring.argtypes = [i64, i64, vp, vp, vp]
    lib.hcgrid_host_ring_info.argtypes = [i64, i32, ctypes.POINTER(i64), ctypes.POINTER(i32),
                                          ctypes.POINTER(dbl), ctypes.POINTER(dbl)]
    lib.hcgrid_measure_peaks.argtypes = [ctypes.c_int, ctypes.POINTER(dbl), ctypes.POINTER(dbl)]
    lib.hcgrid_count_hits_static.argtypes = [vp, i64, vp, vp]
    lib.hcgrid_static_max_cells.argtypes = []
    lib.hcgrid_static_max_cells.restype = i64
    for name in EXPORTS:
        if name not in ("hcgrid_ncell", "hcgrid_last_error", "hcgrid_accumulated_batches", "hcgrid_static_max_cells"):
            getattr(lib, name).restype = ctypes.c_int
    _lib = lib
    return lib


def _np_ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def host_ang2pix_ring(nside: int, lon_deg, lat_deg) -> np.ndarray:
    """HEALPix RING pixel index (the library's a2 code compiled for the host; no GPU)."""
    lib = load_library()
    lon = np.ascontiguousarray(lon_deg, dtype=np.float64).ravel()
    lat = np.ascontiguousarray(lat_deg, dtype=np.float64).ravel()
    pix = np.empty(lon.size, dtype=np.int64)
    rc = lib.hcgrid_host_ang2pix_ring(nside, lon.size, _np_ptr(lon), _np_ptr(lat), _np_ptr(pix))
    if rc != 0:
        raise HCGridError(rc, lib.hcgrid_last_error(None).decode())
    return pix


def host_ring_info(nside: int, iring: int):
    """(first_pixel, npix, lat_deg of the ring centre, lon_deg of the centre of pixel 0)."""
    lib = load_library()
    fp, npx = ctypes.c_int64(), ctypes.c_int32()
    la, lo = ctypes.c_double(), ctypes.c_double()
    rc = lib.hcgrid_host_ring_info(nside, iring, ctypes.byref(fp), ctypes.byref(npx), ctypes.byref(la),
                                   ctypes.byref(lo))
    if rc != 0:
        raise HCGridError(rc, lib.hcgrid_last_error(None).decode())
    return fp.value, npx.value, la.value, lo.value


def measure_peaks(device: int = 0):
    """(FP32-pipe thread-instructions/s, MUFU.EX2 thread-instructions/s) measured now."""
    lib = load_library()
    a, b = ctypes.c_double(), ctypes.c_double()
    rc = lib.hcgrid_measure_peaks(device, ctypes.byref(a), ctypes.byref(b))
    if rc != 0:
        raise HCGridError(rc, lib.hcgrid_last_error(None).decode())
    return a.value, b.value


def static_max_cells() -> int:
    return int(load_library().hcgrid_static_max_cells())


def count_hits_static(counts, out=None, ncell: Optional[int] = None):
    """hcgrid_count_hits_static: (sum of counts, cells with counts > 0) of an int32 CUDA tensor into `out`, a uint64-sized
    (torch.int64) CUDA tensor of 2 entries -- allocated here only if the caller passes none.  The library call itself
    allocates nothing; asynchronous on torch's current stream.  Calls that overlap on one GPU race (shared scratch)."""
    import torch
    lib = load_library()
    if not (counts.is_cuda and counts.dtype == torch.int32 and counts.is_contiguous()):
        raise TypeError("counts must be a contiguous CUDA int32 tensor")
    if out is None:
        out = torch.empty(2, dtype=torch.int64, device=counts.device)
    if not (out.is_cuda and out.dtype == torch.int64 and out.numel() >= 2 and out.is_contiguous()):
        raise TypeError("out must be a contiguous CUDA int64 tensor of 2 entries")
    n = counts.numel() if ncell is None else int(ncell)
    with torch.cuda.device(counts.device):
        st = torch.cuda.current_stream().cuda_stream
        rc = lib.hcgrid_count_hits_static(counts.data_ptr(), n, out.data_ptr(), st)
    if rc != 0:
        raise HCGridError(rc, lib.hcgrid_last_error(None).decode())
    return out


def ang2pix_ring(nside: int, lon_deg, lat_deg):
    """Device a2 step alone: torch CUDA float64 tensors in, int64 tensor out."""
    import torch
    lib = load_library()
    lon = lon_deg.contiguous()
    lat = lat_deg.contiguous()
    assert lon.is_cuda and lon.dtype == torch.float64 and lat.dtype == torch.float64
    pix = torch.empty(lon.numel(), dtype=torch.int64, device=lon.device)
    with torch.cuda.device(lon.device):
        st = torch.cuda.current_stream().cuda_stream
        rc = lib.hcgrid_debug_ang2pix_ring(nside, lon.numel(), lon.data_ptr(), lat.data_ptr(), pix.data_ptr(), st)
    if rc != 0:
        raise HCGridError(rc, lib.hcgrid_last_error(None).decode())
    return pix


class HCGrid:
    """hcgrid_create / hcgrid_set_target_* / hcgrid_grid with torch tensors (include/hcgrid.h)."""

    def __init__(self, sigma_deg: float, support_radius_deg: float, nside: int, precision: str = "f32",
                 device: int = 0):
        self._lib = load_library()
        self._ctx = ctypes.c_void_p()
        self.precision = {"f32": F32, "f64": F64}[precision]
        self.device = int(device)
        rc = self._lib.hcgrid_create(ctypes.byref(self._ctx), float(sigma_deg), float(support_radius_deg),
                                     int(nside), self.precision, self.device)
        if rc != 0:
            raise HCGridError(rc, self._lib.hcgrid_last_error(None).decode())

    # -- life cycle
    def close(self):
        if getattr(self, "_ctx", None) and self._ctx.value:
            self._lib.hcgrid_destroy(self._ctx)
            self._ctx = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def _check(self, rc: int):
        if rc != 0:
            raise HCGridError(rc, self._lib.hcgrid_last_error(self._ctx).decode())

    # -- configuration
    def set_option(self, option: int, value: int):
        self._check(self._lib.hcgrid_set_option(self._ctx, option, int(value)))

    def set_kernel(self, kernel_type: int, a: float = 0.0, b: float = 0.0):
        """hcgrid_set_kernel: KERNEL_GAUSS (default), KERNEL_TAPERED_SINC with its a, b, or KERNEL_ELLIPTICAL_GAUSS with
        a = sigma across / sigma along the axis and b = position angle of the axis (degrees, north through east)."""
        self._check(self._lib.hcgrid_set_kernel(self._ctx, int(kernel_type), float(a), float(b)))

    def set_target_car(self, nx: int, ny: int, lon0_deg: float, lat0_deg: float, dlon_deg: float,
                       dlat_deg: float):
        self._check(self._lib.hcgrid_set_target_car(self._ctx, nx, ny, lon0_deg, lat0_deg, dlon_deg, dlat_deg))

    def set_target_cells(self, lon_deg, lat_deg):
        import torch
        lon = lon_deg.contiguous()
        lat = lat_deg.contiguous()
        if not (lon.is_cuda and lat.is_cuda and lon.dtype == torch.float64 and lat.dtype == torch.float64):
            raise TypeError("set_target_cells wants CUDA float64 tensors")
        with torch.cuda.device(self.device):
            st = torch.cuda.current_stream().cuda_stream
            self._check(self._lib.hcgrid_set_target_cells(self._ctx, lon.numel(), lon.data_ptr(), lat.data_ptr(), st))

    @property
    def ncell(self) -> int:
        return int(self._lib.hcgrid_ncell(self._ctx))

    # -- the hot path
    def grid(self, lon_deg, lat_deg, values, weights=None, want_counts: bool = True, out=None):
        """Device tensors in (lon/lat float64 [n], values float32 [n] or [n, nchan], weights
        float32 [n] or None) -> (datacube [ncell, nchan], weightmap [ncell], counts [ncell] or
        None) on the same device.  Asynchronous on torch's current stream."""
        import torch
        n = lon_deg.numel()
        if values.dim() == 1:
            values = values.view(n, 1)
        nchan = values.shape[1]
        for t, dt in ((lon_deg, torch.float64), (lat_deg, torch.float64), (values, torch.float32)):
            if not (t.is_cuda and t.dtype == dt and t.is_contiguous()):
                raise TypeError("grid wants contiguous CUDA tensors: lon/lat float64, values float32")
        if lat_deg.numel() != n or values.shape[0] != n:
            raise ValueError("lon, lat, values disagree on n")
        if weights is not None and not (weights.is_cuda and weights.dtype == torch.float32
                                        and weights.is_contiguous() and weights.numel() == n):
            raise TypeError("weights must be a contiguous CUDA float32 tensor of n entries")
        ncell = self.ncell
        odt = torch.float64 if self.precision == F64 else torch.float32
        dev = lon_deg.device
        if out is None:
            cube = torch.empty((ncell, nchan), dtype=odt, device=dev)
            wmap = torch.empty(ncell, dtype=odt, device=dev)
            cnt = torch.empty(ncell, dtype=torch.int32, device=dev) if want_counts else None
        else:
            cube, wmap, cnt = out
        with torch.cuda.device(self.device):
            st = torch.cuda.current_stream().cuda_stream
            self._check(self._lib.hcgrid_grid(
                self._ctx, n, lon_deg.data_ptr(), lat_deg.data_ptr(), values.data_ptr(), nchan,
                None if weights is None else weights.data_ptr(), cube.data_ptr(), wmap.data_ptr(),
                None if cnt is None else cnt.data_ptr(), st))
        return cube, wmap, cnt

    def accumulate(self, lon_deg, lat_deg, values, weights=None):
        """hcgrid_accumulate: grid one batch (device tensors as in grid) and add its un-normalised
        sums to the context's accumulators.  Asynchronous on torch's current stream."""
        import torch
        n = lon_deg.numel()
        if values.dim() == 1:
            values = values.view(n, 1)
        nchan = values.shape[1]
        for t, dt in ((lon_deg, torch.float64), (lat_deg, torch.float64), (values, torch.float32)):
            if not (t.is_cuda and t.dtype == dt and t.is_contiguous()):
                raise TypeError("accumulate wants contiguous CUDA tensors: lon/lat float64, values float32")
        if lat_deg.numel() != n or values.shape[0] != n:
            raise ValueError("lon, lat, values disagree on n")
        if weights is not None and not (weights.is_cuda and weights.dtype == torch.float32
                                        and weights.is_contiguous() and weights.numel() == n):
            raise TypeError("weights must be a contiguous CUDA float32 tensor of n entries")
        with torch.cuda.device(self.device):
            st = torch.cuda.current_stream().cuda_stream
            self._check(self._lib.hcgrid_accumulate(
                self._ctx, n, lon_deg.data_ptr(), lat_deg.data_ptr(), values.data_ptr(), nchan,
                None if weights is None else weights.data_ptr(), st))
        self._acc_nchan = nchan

    def finalize(self, want_counts: bool = True, reset: bool = True):
        """hcgrid_finalize: (datacube, weightmap, counts or None) of everything accumulated."""
        import torch
        nchan = getattr(self, "_acc_nchan", 0)
        if nchan == 0:
            raise HCGridError(-2, "nothing accumulated")
        odt = torch.float64 if self.precision == F64 else torch.float32
        dev = torch.device("cuda", self.device)
        cube = torch.empty((self.ncell, nchan), dtype=odt, device=dev)
        wmap = torch.empty(self.ncell, dtype=odt, device=dev)
        cnt = torch.empty(self.ncell, dtype=torch.int32, device=dev) if want_counts else None
        with torch.cuda.device(self.device):
            st = torch.cuda.current_stream().cuda_stream
            self._check(self._lib.hcgrid_finalize(self._ctx, cube.data_ptr(), wmap.data_ptr(),
                                                  None if cnt is None else cnt.data_ptr(), 1 if reset else 0, st))
        if reset:
            self._acc_nchan = 0
        return cube, wmap, cnt

    @property
    def accumulated_batches(self) -> int:
        return int(self._lib.hcgrid_accumulated_batches(self._ctx))

    def grid_host(self, lon_deg: np.ndarray, lat_deg: np.ndarray, values: np.ndarray,
                  weights: Optional[np.ndarray] = None, want_counts: bool = True, out=None):
        """Host (numpy) buffers in and out through hcgrid_grid_host: H2D copies, the whole
        device path, D2H copies, synchronised on return."""
        lon = np.ascontiguousarray(lon_deg, dtype=np.float64)
        lat = np.ascontiguousarray(lat_deg, dtype=np.float64)
        n = lon.size
        val = np.ascontiguousarray(values, dtype=np.float32)
        if val.ndim == 1:
            val = val.reshape(n, 1)
        nchan = val.shape[1]
        wts = None if weights is None else np.ascontiguousarray(weights, dtype=np.float32)
        ncell = self.ncell
        odt = np.float64 if self.precision == F64 else np.float32
        if out is None:
            cube = np.empty((ncell, nchan), dtype=odt)
            wmap = np.empty(ncell, dtype=odt)
            cnt = np.empty(ncell, dtype=np.int32) if want_counts else None
        else:
            cube, wmap, cnt = out
        self._check(self._lib.hcgrid_grid_host(self._ctx, n, _np_ptr(lon), _np_ptr(lat), _np_ptr(val), nchan,
                                               _np_ptr(wts), _np_ptr(cube), _np_ptr(wmap), _np_ptr(cnt)))
        return cube, wmap, cnt

    # -- introspection
    def stats(self) -> dict:
        s = Stats()
        self._check(self._lib.hcgrid_get_stats(self._ctx, ctypes.byref(s)))
        return s.asdict()

    def debug_preorder(self):
        """(sorted_pixel, sorted_index, ring_first, ring_start) of the last grid call."""
        st = self.stats()
        nk, nr = st["n_kept"], st["n_rings"]
        pix = np.empty(nk, dtype=np.int64)
        idx = np.empty(nk, dtype=np.int64)
        rs = np.empty(nr + 1, dtype=np.int64)
        rf = ctypes.c_int32()
        self._check(self._lib.hcgrid_debug_preorder(self._ctx, _np_ptr(pix), _np_ptr(idx), ctypes.byref(rf),
                                                    _np_ptr(rs)))
        return pix, idx, rf.value, rs
