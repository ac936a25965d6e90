"""Roofline model of the convolution kernel (step a6) -- measurement support for bench.py.

Definitions:
  N_hit   pairs (cell, sample) with d <= R: sum of the contributing-sample counts.
  N_cand  the METHOD's candidate pairs: samples lying in a HEALPix pixel that the per-cell
          search of PAPER.md:134-140 (Sect. 3.4 i-iv) visits -- rings
          ring_of(phi_c + R) - 1 .. ring_of(phi_c - R) + 1 and, in ring r, the pixels whose
          centre lies within dl_r + pi / npix_ring(r) of the cell's longitude, dl_r being the
          largest longitude half-width of the support disc over the ring's latitude band.
          Counted here with numpy from the samples' pixel indices, independently of the
          production kernel's loops (whatever windows the kernel really walks, it is
          credited with these pairs only).
  T_roof = max( (N_cand F_d + N_hit F_a) / P_fp32 ,  N_hit / P_mufu ,  B_unique / BW_hbm )
  F_d = 12 FP32-pipe instructions per candidate, F_a = 5 + nchan (+1 with weights, +1 with the
  count output) per hit,
  one MUFU.EX2 per hit; B_unique = the API-level arrays once each.

Nothing here runs on the product path; the pixel indices come from the library's own
host build of step a2 (binding.host_ang2pix_ring).
"""
from __future__ import annotations

import numpy as np

from . import binding

F_D = 12
NUM_SMS = 148
FP32_LANES_PER_SM = 128
MUFU_LANES_PER_SM = 16
SM_MAX_HZ = 1.965e9
# peak DESIGN.md derives from the guide's unit counts and clocks (thread-instructions / s)
P_FP32_NOMINAL = NUM_SMS * FP32_LANES_PER_SM * SM_MAX_HZ
P_MUFU_NOMINAL = NUM_SMS * MUFU_LANES_PER_SM * SM_MAX_HZ


def f_a(nchan: int, has_weights: bool, want_counts: bool = True) -> int:
    """FP32-pipe instructions per accepted pair; the count increment is only charged when the
    count output is requested."""
    return 5 + nchan + (1 if has_weights else 0) + (1 if want_counts else 0)


def _ring_z(nside: int) -> np.ndarray:
    """z of the centre of ring i for i = 0 .. 4 nside (0 and 4 nside are the poles)."""
    i = np.arange(0, 4 * nside + 1, dtype=np.float64)
    n = float(nside)
    z = np.where(i < n, 1.0 - i * i / (3.0 * n * n),
                 np.where(i <= 3 * n, (2.0 * n - i) * 2.0 / (3.0 * n), -(1.0 - (4 * n - i) ** 2 / (3.0 * n * n))))
    return z


def count_candidates(w, max_rows: int | None = None) -> dict:
    """N_cand of workload `w` (plate-carree target) by the definition above.  Returns
    {"n_cand", "rows_counted", "ncell_counted"}; with max_rows the count is taken on an evenly
    spaced subset of rows and scaled (stated in the result)."""
    nside = w.nside
    t = w.target
    R = np.deg2rad(w.radius_deg)
    pix = binding.host_ang2pix_ring(nside, w.lon, w.lat)
    i = np.arange(1, 4 * nside, dtype=np.int64)
    npr_all = 4 * np.minimum(np.minimum(i, 4 * nside - i), nside)
    first = np.concatenate([[0], np.cumsum(npr_all)])          # first[r-1] = first pixel of ring r
    ring = np.searchsorted(first, pix, side="right")           # 1-based ring number
    jpix = pix - first[ring - 1]
    zc = _ring_z(nside)
    latc = np.arcsin(np.clip(zc, -1.0, 1.0))                   # latitude of ring centres, [0..4n]
    rmin, rmax = int(ring.min()), int(ring.max())
    # per-ring cumulative histogram over pixel-in-ring (only the data's rings)
    cum = {}
    order = np.argsort(ring, kind="stable")
    rs, js = ring[order], jpix[order]
    bounds = np.searchsorted(rs, np.arange(rmin, rmax + 2))
    for r in range(rmin, rmax + 1):
        h = np.bincount(js[bounds[r - rmin]:bounds[r - rmin + 1]], minlength=int(npr_all[r - 1]))
        cum[r] = np.concatenate([[0], np.cumsum(h)])
    ix = np.arange(t.nx, dtype=np.float64)
    lonc = np.deg2rad(t.lon0 + ix * t.dlon)
    rows = np.arange(t.ny)
    if max_rows is not None and t.ny > max_rows:
        rows = np.unique(np.linspace(0, t.ny - 1, max_rows).round().astype(int))
    total = 0
    for iy in rows:
        phic = np.deg2rad(t.lat0 + iy * t.dlat)
        # ring_of(lat): the ring whose band holds lat = number of ring centres with z >= sin(lat), clipped
        def ring_of(phi):
            phi = min(max(phi, -np.pi / 2), np.pi / 2)
            z = np.sin(phi)
            k = int(np.searchsorted(-zc, -z, side="left"))     # first ring centre with zc <= z
            return min(max(k, 1), 4 * nside - 1)
        r_lo = max(ring_of(phic + R) - 1, 1)
        r_hi = min(ring_of(phic - R) + 1, 4 * nside - 1)
        for r in range(max(r_lo, rmin), min(r_hi, rmax) + 1):
            band_hi, band_lo = latc[r - 1], latc[r + 1]
            lo, hi = max(band_lo, phic - R), min(band_hi, phic + R)
            if lo > hi:
                continue
            npr = int(npr_all[r - 1])
            whole = abs(phic) + R >= np.pi / 2
            dl = np.pi
            if not whole:
                pstar = np.arcsin(np.clip(np.sin(phic) / np.cos(R), -1.0, 1.0))
                pe = min(hi, max(lo, pstar))
                f = (np.sin(R / 2) ** 2 - np.sin((pe - phic) / 2) ** 2) / (np.cos(pe) * np.cos(phic))
                if f >= 1.0:
                    whole = True
                else:
                    dl = 2.0 * np.arcsin(np.sqrt(max(f, 0.0)))
            c = cum[r]
            if whole or 2.0 * (dl + np.pi / npr) >= 2.0 * np.pi:
                total += int(c[-1]) * t.nx
                continue
            # pixel j of ring r is centred at (j + off) * 2 pi / npr
            belt = nside <= r <= 3 * nside
            off = 0.0 if (belt and ((r - nside + 1) & 1) == 0) else 0.5
            half = dl + np.pi / npr
            g_lo = (lonc - half) * npr / (2 * np.pi) - off     # centres with j >= g_lo
            g_hi = (lonc + half) * npr / (2 * np.pi) - off     # and j <= g_hi
            j0 = np.ceil(g_lo).astype(np.int64)
            j1 = np.floor(g_hi).astype(np.int64)
            cnt = np.zeros(t.nx, dtype=np.int64)
            # unwrap modulo the ring length (a window crossing lon = 0 becomes two ranges)
            for shift in (-npr, 0, npr):
                a = np.clip(j0 + shift, 0, npr)
                b = np.clip(j1 + shift + 1, 0, npr)
                cnt += np.where(b > a, c[b] - c[a], 0)
            total += int(cnt.sum())
    scale = t.ny / len(rows)
    return {"n_cand": int(round(total * scale)), "rows_counted": int(len(rows)),
            "ncell_counted": int(len(rows) * t.nx)}


def model(n: int, ncell: int, nchan: int, has_weights: bool, n_hit: int, n_cand: int, hbm_gbs: float,
          p_fp32: float = P_FP32_NOMINAL, p_mufu: float = P_MUFU_NOMINAL, want_counts: bool = True) -> dict:
    """The three legs of T_roof in seconds and which one binds."""
    inst = n_cand * F_D + n_hit * f_a(nchan, has_weights, want_counts)
    b_unique = n * (16 + 4 * nchan + (4 if has_weights else 0)) + ncell * (4 * nchan + 4 + (4 if want_counts else 0))
    t_fp32 = inst / p_fp32
    t_mufu = n_hit / p_mufu
    t_hbm = b_unique / (hbm_gbs * 1e9)
    legs = {"alu": t_fp32, "mufu": t_mufu, "hbm": t_hbm}
    bound = max(legs, key=legs.get)
    return {"fp32_inst": int(inst), "bytes_unique": int(b_unique), "t_fp32_s": t_fp32, "t_mufu_s": t_mufu,
            "t_hbm_s": t_hbm, "t_roof_s": legs[bound], "bound": bound}
