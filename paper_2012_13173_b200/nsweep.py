"""Time versus input size: the SHAPE of the paper's Exp. 3 (Fig. 9) on synthetic data.

    python -m paper_2012_13173_b200.nsweep [--nmax 3.6e8] [--steps 5] [--json out.json]

Workload as the paper states it: a 5 deg x 5 deg field gridded to 90 x 90 cells of 200 arcsec,
kernel FWHM 300 arcsec (sigma = FWHM / sqrt(8 ln 2), support 3 sigma), N from
1e3 to 3.6e8 samples, here uniformly random positions with one Gaussian random value each
(PAPER.md:195).  nside 2048 (pixel side ~ sigma / 1.2; the paper's rule of thumb).
The paper's own curves are only in Fig. 9, whose image is not available; what can be checked is
its statement of the shape: flat below ~1e5 samples, ~O(n) above, and the convolution's share of
the whole call.  Inputs are resident on the device; per N the whole hcgrid_grid call and its
stages are timed with the library's CUDA events (median of `steps` calls after 2 warm-ups).
"""
from __future__ import annotations

import argparse
import json
import math

import numpy as np

FIELD_DEG = 5.0
CELL_DEG = 200.0 / 3600.0
NCELL_SIDE = 90
SIGMA_DEG = 300.0 / 3600.0 / math.sqrt(8.0 * math.log(2.0))
RADIUS_DEG = 3.0 * SIGMA_DEG
NSIDE = 2048
LON_C, LAT_C = 30.0, 25.0


def sizes(nmax: float):
    out, n = [], 1.0e3
    while n < nmax * 0.999:
        out.append(int(n))
        n *= math.sqrt(10.0)
    out.append(int(nmax))
    return out


def main():
    import torch
    from . import binding
    ap = argparse.ArgumentParser()
    ap.add_argument("--nmax", type=float, default=3.6e8)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--json", default=None)
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("nsweep needs a CUDA device: the product path has no CPU fallback")
    dev = torch.device("cuda", 0)
    g = binding.HCGrid(SIGMA_DEG, RADIUS_DEG, NSIDE, device=0)
    half = 0.5 * (NCELL_SIDE - 1) * CELL_DEG
    g.set_target_car(NCELL_SIDE, NCELL_SIDE, LON_C - half, LAT_C - half, CELL_DEG, CELL_DEG)
    g.set_option(binding.OPT_PROFILE, 1)
    ncell = NCELL_SIDE * NCELL_SIDE
    out = (torch.empty((ncell, 1), dtype=torch.float32, device=dev), torch.empty(ncell, dtype=torch.float32, device=dev),
           None)
    gen = torch.Generator(device=dev)
    rows = []
    for n in sizes(args.nmax):
        # a fresh target per size: the lookup-bin refinement a dense size triggers is not inherited by the next
        g.set_target_car(NCELL_SIDE, NCELL_SIDE, LON_C - half, LAT_C - half, CELL_DEG, CELL_DEG)
        gen.manual_seed(13173 + n % 1000003)
        # positions uniform over the field (in coordinate degrees), generated on the device
        lon = LON_C + (torch.rand(n, dtype=torch.float64, device=dev, generator=gen) - 0.5) * FIELD_DEG
        lat = LAT_C + (torch.rand(n, dtype=torch.float64, device=dev, generator=gen) - 0.5) * FIELD_DEG
        val = torch.randn((n, 1), dtype=torch.float32, device=dev, generator=gen)
        keys = ("us_pixelise", "us_sort", "us_tables", "us_pack", "us_convolve", "us_total")
        acc = {k: [] for k in keys}
        for i in range(2 + args.steps):
            g.grid(lon, lat, val, None, want_counts=False, out=out)
            torch.cuda.synchronize()
            s = g.stats()
            if i >= 2:
                for k in keys:
                    acc[k].append(s[k])
        med = {k: float(np.median(v)) for k, v in acc.items()}
        # the call as a caller sees it (no per-stage events): back-to-back calls between two CUDA events, once with the
        # graph replay of repeated calls (the default up to 2^21 samples) and once with eager launches
        call = {}
        reps = 50 if n <= 10 ** 6 else 5
        for name, mode in (("us_call", -1), ("us_call_eager", 0)):
            g.set_option(binding.OPT_PROFILE, 0)
            g.set_option(binding.OPT_GRAPH, mode)
            for _ in range(3):
                g.grid(lon, lat, val, None, want_counts=False, out=out)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            for _ in range(reps):
                g.grid(lon, lat, val, None, want_counts=False, out=out)
            e1.record()
            torch.cuda.synchronize()
            call[name] = 1e3 * e0.elapsed_time(e1) / reps
            call[name + "_graph"] = g.stats()["graph"]
        g.set_option(binding.OPT_GRAPH, -1)
        g.set_option(binding.OPT_PROFILE, 1)
        row = {"n": n, "us_call": call["us_call"], "graph": call["us_call_graph"], "us_call_eager": call["us_call_eager"],
               "subpix_bits": s["subpix_bits"], "preorder": s["preorder"],
               "us_total": med["us_total"], "us_convolve": med["us_convolve"],
               "us_preorder": med["us_pixelise"] + med["us_sort"] + med["us_tables"] + med["us_pack"],
               "conv_share": med["us_convolve"] / med["us_total"], "samples_per_s": n / (med["us_total"] * 1e-6),
               "tile": f"{s['coarsen']}x{s['coarsen_y']}"}
        rows.append(row)
        print(json.dumps(row), flush=True)
        del lon, lat, val
    if args.json:
        with open(args.json, "w") as f:
            json.dump({"workload": "5x5 deg, 90x90 cells of 200 arcsec, FWHM 300 arcsec, nside 2048", "rows": rows}, f,
                      indent=1)
    g.close()


if __name__ == "__main__":
    main()
