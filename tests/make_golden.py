"""Writes the oracle's results on the stratified cell subset (tests/golden_subset.py) of the full-size
BASELINE configs 3 and 5 to tests/golden/config{3,5}_subset_oracle.npz.

    python tests/make_golden.py [3] [5]

Calls only oracle/ and the seeded input generators (paper_2012_13173_b200/workloads.py holds no arithmetic of
the method); nothing here touches the CUDA path.  About 5 + 8 minutes on 8 cores.  Each file carries the hash
of the kernel parameters, the target and the input arrays it was computed from; the parity test refuses a
file whose hash does not match the workload it regenerates."""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

from golden_subset import golden_path, subset_cells, workload_key  # noqa: E402
from oracle import oracle  # noqa: E402
from paper_2012_13173_b200 import workloads  # noqa: E402


def main():
    cfgs = [int(a) for a in sys.argv[1:]] or [3, 5]
    oracle.build()
    for cfg in cfgs:
        w = workloads.make(cfg, 1.0)
        t = w.target
        cells = subset_cells(t.nx, t.ny, cfg)
        cl, cb = t.cell_centers()
        t0 = time.time()
        ref = oracle.grid(w.sigma_deg, w.radius_deg, cl[cells], cb[cells], w.lon, w.lat, w.values, w.weights)
        print(f"config {cfg}: {cells.size} cells x {w.n} samples in {time.time() - t0:.0f} s on {ref.threads} threads",
              flush=True)
        np.savez_compressed(golden_path(cfg), key=workload_key(w), cells=cells, datacube=ref.datacube.astype(np.float64),
                            weightmap=ref.weightmap, counts=ref.counts.astype(np.int32),
                            absmap=ref.absmap, near_boundary=ref.near_boundary.astype(np.int16), vmax=ref.vmax)


if __name__ == "__main__":
    main()
