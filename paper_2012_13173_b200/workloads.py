"""Seeded synthetic input generators for the five BASELINE.json configs.

This module serves BOTH the CUDA path's tests/bench and the oracle's tests.  It holds
none of the method's arithmetic (no distances, no kernel weights, no pixelisation): it
only draws sample positions, values and weights and states the kernel / target
parameters of each config.  numpy only; it imports nothing else from this package.

Recipes follow SURVEY.md 8(d) / DESIGN.md "Input recipe".  The paper measured on
simulated data "generated in the similar way as Winkel et al. (2016b)": one Gaussian
random value at each uniformly random position in a field, available
only on request; these seeded generators stand in for it and add FAST's
drift-scan geometry.

rng = numpy.random.default_rng([13173, k]) for config k; draws happen in the order
written below, so a given (k, scale) is reproducible bit for bit.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

ARCMIN = 1.0 / 60.0          # degrees
ARCSEC = 1.0 / 3600.0        # degrees


@dataclass
class CarTarget:
    """Plate-carree target grid: cell (ix, iy) centre = (lon0 + ix*dlon, lat0 + iy*dlat),
    flat index iy*nx + ix (SURVEY.md 8c reading c12/c13)."""
    nx: int
    ny: int
    lon0: float
    lat0: float
    dlon: float
    dlat: float

    @property
    def ncell(self) -> int:
        return self.nx * self.ny

    def cell_centers(self):
        """Per-cell (lon, lat) in degrees, flat [ny*nx]; evaluated as lon0 + ix*dlon with
        one rounding per operation (no FMA), the expression the CUDA path reproduces."""
        ix = np.arange(self.nx, dtype=np.float64)
        iy = np.arange(self.ny, dtype=np.float64)
        lon = self.lon0 + ix * self.dlon
        lat = self.lat0 + iy * self.dlat
        return (np.broadcast_to(lon[None, :], (self.ny, self.nx)).reshape(-1).copy(),
                np.broadcast_to(lat[:, None], (self.ny, self.nx)).reshape(-1).copy())


@dataclass
class Workload:
    name: str
    config: int
    scale: float
    lon: np.ndarray                 # [n] float64 degrees
    lat: np.ndarray                 # [n] float64 degrees
    values: np.ndarray              # [n, nchan] float32
    weights: Optional[np.ndarray]   # [n] float32 or None
    sigma_deg: float
    radius_deg: float
    nside: int
    target: CarTarget
    notes: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.lon.size)

    @property
    def nchan(self) -> int:
        return int(self.values.shape[1])


def _centred_target(lon_c, lat_c, nx, ny, delta) -> CarTarget:
    return CarTarget(nx, ny, lon_c - 0.5 * (nx - 1) * delta, lat_c - 0.5 * (ny - 1) * delta,
                     delta, delta)


def _smooth_field(rng, lon, lat, lon_c, lat_c, half_lon, half_lat, sd_lo, sd_hi, ncomp=50,
                  chunk=1 << 20):
    """Sum of `ncomp` seeded 2-D Gaussian blobs (a synthetic sky brightness, not the
    gridding kernel): centres U over the patch, sd U(sd_lo, sd_hi) degrees on the sky,
    amplitude U(0.5, 2).  Flat-sky offsets scaled by cos(lat_c) are good enough for a
    value field."""
    cx = lon_c + rng.uniform(-half_lon, half_lon, ncomp)
    cy = lat_c + rng.uniform(-half_lat, half_lat, ncomp)
    sd = rng.uniform(sd_lo, sd_hi, ncomp)
    amp = rng.uniform(0.5, 2.0, ncomp)
    cosl = np.cos(np.deg2rad(lat_c))
    out = np.empty(lon.size, dtype=np.float64)
    for a in range(0, lon.size, chunk):
        b = min(a + chunk, lon.size)
        dx = (lon[a:b, None] - cx[None, :]) * cosl
        dy = lat[a:b, None] - cy[None, :]
        out[a:b] = (amp[None, :] * np.exp(-(dx * dx + dy * dy) / (2.0 * sd[None, :] ** 2))).sum(1)
    return out


def _drift_scan(rng, lon_c, lat_c, side_deg, coverages=4):
    """FAST-like drift scan (19 beams, 23.4 deg rotation, 1'09'' declination
    spacing, 1 s sampling).  The 19 beams of the hexagonal lattice rotated by
    atan(sqrt(3)/4) = 23.41 deg have declination offsets (2i+5j)*u, u = 69'', which tile
    the declination axis uniformly when passes step by 19u; `coverages` interleaved
    coverages offset by u/coverages give tracks u/coverages apart.  Each track is a
    constant-declination line sampled every 15'' of RA (1 s at the sidereal rate) with
    a seeded phase.  Track order: coverage-major, then declination, samples in time
    order."""
    u = 69.0 * ARCSEC
    step = u / coverages
    ntrack = int(np.floor(side_deg / step)) + 1
    nsamp = int(round(side_deg / (15.0 * ARCSEC)))
    m = np.arange(ntrack)
    order = np.lexsort((m // coverages, m % coverages))     # coverage-major
    m = m[order]
    dec = lat_c - 0.5 * side_deg + m * step
    phase = rng.uniform(0.0, 1.0, ntrack)
    t = np.arange(nsamp, dtype=np.float64)
    lon = (lon_c - 0.5 * side_deg) + (phase[:, None] + t[None, :]) * (15.0 * ARCSEC)
    lat = np.broadcast_to(dec[:, None], lon.shape)
    return lon.reshape(-1).copy(), lat.reshape(-1).copy(), ntrack, nsamp


def make(config: int, scale: float = 1.0) -> Workload:
    """Build config `config` (1..5).  `scale` in (0, 1] shrinks the patch AREA (and with
    it the sample and cell counts) at fixed density, kernel and nside, so every config
    has a seconds-fast miniature with the same local structure."""
    if config not in (1, 2, 3, 4, 5):
        raise ValueError("config must be 1..5")
    if not (0.0 < scale <= 1.0):
        raise ValueError("scale must be in (0, 1]")
    rng = np.random.default_rng([13173, config])
    s = float(np.sqrt(scale))

    if config == 1:
        n = max(1, int(round(20000 * scale)))
        half = 0.5 * s
        lon = 30.0 + rng.uniform(-half, half, n)
        lat = 20.0 + rng.uniform(-half, half, n)
        val = (np.sin(3.0 * np.deg2rad(lon) * 60.0) + np.cos(2.0 * np.deg2rad(lat) * 60.0)
               + rng.normal(0.0, 0.1, n))
        nc = max(1, int(round(60 * s)))
        return Workload("tiny", 1, scale, lon, lat, val.astype(np.float32)[:, None], None,
                        1.5 * ARCMIN, 4.5 * ARCMIN, 2048,
                        _centred_target(30.0, 20.0, nc, nc, 1.0 * ARCMIN))

    if config in (2, 4):
        side = 5.0 * s
        lon, lat, ntrack, nsamp = _drift_scan(rng, 30.0, 25.0, side)
        notes = {"tracks": ntrack, "samples_per_track": nsamp}
        nc = max(1, int(round(300 * s)))
        tgt = _centred_target(30.0, 25.0, nc, nc, 1.0 * ARCMIN)
        if config == 2:
            val = (_smooth_field(rng, lon, lat, 30.0, 25.0, side / 2, side / 2,
                                 3.0 * ARCMIN, 30.0 * ARCMIN)
                   + rng.normal(0.0, 0.05, lon.size))
            return Workload("drift", 2, scale, lon, lat, val.astype(np.float32)[:, None], None,
                            1.23 * ARCMIN, 3.69 * ARCMIN, 4096, tgt, notes)
        # config 4: seeded subset of exactly round(1e6*scale) samples kept in time order
        n = min(lon.size, max(1, int(round(1_000_000 * scale))))
        keep = np.sort(rng.choice(lon.size, size=n, replace=False))
        lon, lat = lon[keep], lat[keep]
        nchan = 256
        f = []
        for _ in range(3):
            g = _smooth_field(rng, lon, lat, 30.0, 25.0, side / 2, side / 2,
                              3.0 * ARCMIN, 30.0 * ARCMIN)
            lo, hi = g.min(), g.max()
            f.append((g - lo) / (hi - lo) if hi > lo else np.zeros_like(g))
        amp = 2.0 + 8.0 * f[0]
        k0 = 64.0 + 128.0 * f[1]
        wid = 2.0 + 10.0 * f[2]
        k = np.arange(nchan, dtype=np.float64)
        val = np.empty((n, nchan), dtype=np.float32)
        chunk = 1 << 16
        for a in range(0, n, chunk):
            b = min(a + chunk, n)
            line = amp[a:b, None] * np.exp(-(k[None, :] - k0[a:b, None]) ** 2
                                           / (2.0 * wid[a:b, None] ** 2))
            val[a:b] = (rng.standard_normal((b - a, nchan)) + line).astype(np.float32)
        notes["subset_of"] = int(ntrack * nsamp)
        return Workload("cube", 4, scale, lon, lat, val, None,
                        1.23 * ARCMIN, 3.69 * ARCMIN, 4096, tgt, notes)

    if config == 3:
        n = max(1, int(round(10_000_000 * scale)))
        half = 5.0 * s
        lon = 180.0 + rng.uniform(-half, half, n)
        lat = rng.uniform(-half, half, n)
        val = rng.standard_normal(n) + _smooth_field(rng, lon, lat, 180.0, 0.0, half, half,
                                                     3.0 * ARCMIN, 60.0 * ARCMIN)
        nc = max(1, int(round(1200 * s)))
        return Workload("dense", 3, scale, lon, lat, val.astype(np.float32)[:, None], None,
                        0.5 * ARCMIN, 1.5 * ARCMIN, 8192,
                        _centred_target(180.0, 0.0, nc, nc, 0.5 * ARCMIN))

    # config 5: 2-D Gaussian density (sd 1.5 deg in COORDINATE degrees) clipped to +-4 deg
    n = max(1, int(round(20_000_000 * scale)))
    sd, clip = 1.5 * s, 4.0 * s
    lon = np.empty(n)
    lat = np.empty(n)
    have = 0
    while have < n:
        m = int((n - have) * 1.1) + 1024
        x = rng.normal(0.0, sd, m)
        y = rng.normal(0.0, sd, m)
        ok = (np.abs(x) <= clip) & (np.abs(y) <= clip)
        x, y = x[ok][: n - have], y[ok][: n - have]
        lon[have:have + x.size] = 45.0 + x
        lat[have:have + x.size] = 80.0 + y
        have += x.size
    val = (_smooth_field(rng, lon, lat, 45.0, 80.0, clip, clip, 3.0 * ARCMIN, 30.0 * ARCMIN)
           + rng.normal(0.0, 0.05, n))
    wts = rng.uniform(0.5, 1.5, n).astype(np.float32)
    nc = max(1, int(round(480 * s)))
    return Workload("polar", 5, scale, lon, lat, val.astype(np.float32)[:, None], wts,
                    1.0 * ARCMIN, 3.0 * ARCMIN, 4096,
                    _centred_target(45.0, 80.0, nc, nc, 1.0 * ARCMIN))


def random_case(seed: int, n: int, ncell: int, lon_c: float, lat_c: float, half_deg: float,
                nchan: int = 1, with_weights: bool = False):
    """Small unstructured case for property tests: n samples and ncell arbitrary cell
    centres uniform in a (2*half_deg)^2 coordinate box around (lon_c, lat_c); longitudes
    are reduced to [0, 360), latitudes clipped to [-90, 90]."""
    rng = np.random.default_rng([13173, 99, seed])
    lon = np.mod(lon_c + rng.uniform(-half_deg, half_deg, n), 360.0)
    lat = np.clip(lat_c + rng.uniform(-half_deg, half_deg, n), -90.0, 90.0)
    clon = np.mod(lon_c + rng.uniform(-half_deg, half_deg, ncell), 360.0)
    clat = np.clip(lat_c + rng.uniform(-half_deg, half_deg, ncell), -90.0, 90.0)
    val = rng.standard_normal((n, nchan)).astype(np.float32)
    wts = rng.uniform(0.5, 1.5, n).astype(np.float32) if with_weights else None
    return lon, lat, val, wts, clon, clat
