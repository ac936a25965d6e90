"""The declared stratified cell subset of SURVEY.md 8c for the full-size oracle runs that are too
long to repeat in every test run: all four borders of the target 8 cells deep plus 64 seeded 32 x 32
interior blocks.  Shared by tests/make_golden.py (writes the oracle's results) and the GPU parity test
(reads them); no arithmetic of the method lives here."""
import hashlib

import numpy as np

BORDER = 8
NBLOCKS = 64
BLOCK = 32


def subset_cells(nx: int, ny: int, cfg: int) -> np.ndarray:
    """Sorted flat indices (iy * nx + ix) of the subset."""
    mask = np.zeros((ny, nx), dtype=bool)
    mask[:BORDER, :] = True
    mask[-BORDER:, :] = True
    mask[:, :BORDER] = True
    mask[:, -BORDER:] = True
    rng = np.random.default_rng([13173, 290, cfg])
    for _ in range(NBLOCKS):
        x0 = int(rng.integers(BORDER, max(BORDER + 1, nx - BORDER - BLOCK)))
        y0 = int(rng.integers(BORDER, max(BORDER + 1, ny - BORDER - BLOCK)))
        mask[y0:y0 + BLOCK, x0:x0 + BLOCK] = True
    return np.flatnonzero(mask.ravel()).astype(np.int64)


def workload_key(w) -> str:
    """Hash of everything the oracle's result depends on: kernel, target, and the input arrays themselves."""
    h = hashlib.sha256()
    t = w.target
    h.update(repr((w.sigma_deg, w.radius_deg, t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat, w.n, w.nchan)).encode())
    for a in (w.lon, w.lat, w.values, w.weights):
        if a is not None:
            h.update(np.ascontiguousarray(a).tobytes())
    return h.hexdigest()[:32]


def golden_path(cfg: int) -> str:
    import os
    return os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", f"config{cfg}_subset_oracle.npz")
