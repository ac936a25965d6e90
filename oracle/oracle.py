"""ctypes loader for the brute-force fp64 oracle.  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It shares no code with paper_2012_13173_b200/.

The arithmetic lives in hcgrid_oracle.c (Eq. 1 of the paper); this
file only builds it with gcc and marshals numpy arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hcgrid_oracle.c")
_HDR = os.path.join(_HERE, "hcgrid_oracle.h")
_LIB = os.path.join(_HERE, "libhcgrid_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2 -fopenmp, no fast-math).  Returns the .so path."""
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        cmd = ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c11", "-Wall", "-Wextra",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        d = ctypes.c_double
        lib.hcgrid_oracle_distance.restype = d
        lib.hcgrid_oracle_distance.argtypes = [d, d, d, d]
        p = ctypes.c_void_p
        lib.hcgrid_oracle_grid.restype = ctypes.c_int
        lib.hcgrid_oracle_grid.argtypes = [d, d, ctypes.c_int64, p, p, ctypes.c_int64, p, p, p,
                                           ctypes.c_int32, p, p, p, p, p, p, ctypes.c_int]
        lib.hcgrid_oracle_grid_kernel.restype = ctypes.c_int
        lib.hcgrid_oracle_grid_kernel.argtypes = [ctypes.c_int, d, d, d, d, ctypes.c_int64, p, p, ctypes.c_int64, p, p,
                                                  p, ctypes.c_int32, p, p, p, p, p, p, p, ctypes.c_int]
        lib.hcgrid_oracle_last_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def distance(lon1_deg, lat1_deg, lon2_deg, lat2_deg) -> float:
    """Great-circle angle in radians (the function the gridder calls per pair)."""
    return float(_load().hcgrid_oracle_distance(float(lon1_deg), float(lat1_deg),
                                                float(lon2_deg), float(lat2_deg)))


@dataclass
class OracleResult:
    datacube: np.ndarray       # [ncell, nchan] float64, NaN where weightmap == 0
    weightmap: np.ndarray      # [ncell] float64
    counts: np.ndarray         # [ncell] int64, geometric (ignores per-sample weights)
    absmap: np.ndarray         # [ncell, nchan] float64: sum q w |v| / W
    near_boundary: np.ndarray  # [ncell] int64: pairs with |d - R| < 1e-9 rad
    threads: int
    abswmap: np.ndarray = None  # [ncell] float64: sum |q w| (kernel= calls only)
    vmax: float = 1.0           # largest |value| of the input (finite ones): scale of a boundary pair's effect on V


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


GAUSS, TAPERED_SINC, ELLIPTICAL_GAUSS = 0, 1, 2


def _vmax(values) -> float:
    a = np.abs(values[np.isfinite(values)]) if values.size else values
    return float(a.max()) if a.size else 0.0


def grid(sigma_deg, radius_deg, cell_lon, cell_lat, lon, lat, values, weights=None,
         nthreads: int = 0, kernel=None) -> OracleResult:
    """Brute-force Eq. 1 over every (cell, sample) pair.  Angles in degrees.
    kernel = None (Gaussian, hcgrid_oracle_grid) or (ktype, ka, kb) (hcgrid_oracle_grid_kernel)."""
    lib = _load()
    cell_lon = np.ascontiguousarray(cell_lon, dtype=np.float64).ravel()
    cell_lat = np.ascontiguousarray(cell_lat, dtype=np.float64).ravel()
    lon = np.ascontiguousarray(lon, dtype=np.float64).ravel()
    lat = np.ascontiguousarray(lat, dtype=np.float64).ravel()
    n = lon.size
    ncell = cell_lon.size
    values = np.ascontiguousarray(values, dtype=np.float32)
    if values.ndim == 1:
        values = values.reshape(n, 1)
    nchan = values.shape[1] if values.ndim == 2 and values.shape[0] == n else -1
    if n == 0:
        nchan = values.shape[1] if values.ndim == 2 else 1
    if cell_lat.size != ncell or lat.size != n or nchan < 1:
        raise ValueError("inconsistent shapes")
    if weights is not None:
        weights = np.ascontiguousarray(weights, dtype=np.float32).ravel()
        if weights.size != n:
            raise ValueError("weights must have one entry per sample")
    cube = np.empty((ncell, nchan), dtype=np.float64)
    wmap = np.empty(ncell, dtype=np.float64)
    counts = np.empty(ncell, dtype=np.int64)
    absmap = np.empty((ncell, nchan), dtype=np.float64)
    nb = np.empty(ncell, dtype=np.int64)
    if kernel is not None:
        ktype, ka, kb = kernel
        absw = np.empty(ncell, dtype=np.float64)
        rc = lib.hcgrid_oracle_grid_kernel(int(ktype), float(ka), float(kb), float(sigma_deg), float(radius_deg),
                                           ncell, _ptr(cell_lon), _ptr(cell_lat), n, _ptr(lon), _ptr(lat),
                                           _ptr(values), nchan, _ptr(weights), _ptr(cube), _ptr(wmap),
                                           _ptr(counts), _ptr(absmap), _ptr(absw), _ptr(nb), int(nthreads))
        if rc != 0:
            raise ValueError("hcgrid_oracle_grid_kernel rejected its arguments")
        return OracleResult(cube, wmap, counts, absmap, nb, int(lib.hcgrid_oracle_last_threads()), absw, _vmax(values))
    rc = lib.hcgrid_oracle_grid(float(sigma_deg), float(radius_deg), ncell, _ptr(cell_lon),
                                _ptr(cell_lat), n, _ptr(lon), _ptr(lat), _ptr(values), nchan,
                                _ptr(weights), _ptr(cube), _ptr(wmap), _ptr(counts),
                                _ptr(absmap), _ptr(nb), int(nthreads))
    if rc != 0:
        raise ValueError("hcgrid_oracle_grid rejected its arguments")
    return OracleResult(cube, wmap, counts, absmap, nb, int(lib.hcgrid_oracle_last_threads()), None, _vmax(values))


if __name__ == "__main__":
    print(build(force=True))
