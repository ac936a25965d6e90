#!/usr/bin/env python
"""bench.py -- throughput of the HCGrid hot path on B200 (BASELINE.json metric:
"gridded cell-channels/s and kernel evals/s at 1 B200; % of roofline").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl reference]

With --gpus N > 1 and no torchrun environment the script starts the N ranks itself (one process
per GPU, rendezvous on 127.0.0.1); under torchrun it uses the ranks it was given and fails if
their number differs from --gpus.

A step is one pass of the whole hot path (a2 pixelise, a3 sort, a4 tables, a5 pack, a6
convolve: one hcgrid_grid call) over one batch of seeded synthetic input, by default
BASELINE config 3 ("dense scan", 10 M samples, 1200 x 1200 cells) -- the configuration the
north_star's roofline target is quoted on.  `value` is measured with the inputs resident
in HBM; `e2e` goes through hcgrid_grid_host with pinned HOST buffers (H2D + path + D2H
inside the timed region).  `roofline` is for the dominant kernel, the convolution, timed
with CUDA events on its own stream (the library's per-stage events).  `cpu_baseline` is
the brute-force oracle timed on this box's host cores on a bounded sample of the cells.

--impl reference times the oracle itself (there is no reference implementation to
install: /root/reference holds the paper only).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "gridded cell-channels/s (whole hcgrid_grid call, inputs resident in HBM)"
UNIT = "cell-channels/s"
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed
# `ncu --set full` captures (profiles/): (config, stats kernel id) -> (bytes, source)
NCU_TRAFFIC = {
    (3, 6): (191993856 + 12059648, "profiles/r02_conv1_tile_ncu_full.md"),
    (4, 7): (3714980000 + 98979072, "profiles/r01c_conv_mc_ncu_full.md"),
    (4, 8): (1360306000 + 82240256, "profiles/r02_conv_mc_tc_ncu_full.md"),
}
WORKLOAD_NAMES = {1: "config1_tiny_20k", 2: "config2_drift_scan_1.25M", 3: "config3_dense_10M",
                  4: "config4_spectral_cube_1M_x256", 5: "config5_polar_20M"}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(w, cells, nthreads=0):
    """Run the oracle on the flat cell indices `cells`; returns (result, seconds)."""
    from oracle import oracle
    oracle.build()
    cl, cb = w.target.cell_centers()
    t0 = time.perf_counter()
    ref = oracle.grid(w.sigma_deg, w.radius_deg, cl[cells], cb[cells], w.lon, w.lat, w.values, w.weights,
                      nthreads=nthreads)
    return ref, time.perf_counter() - t0


def evenly_spaced_cells(ncell, k):
    return np.unique(np.linspace(0, ncell - 1, min(k, ncell)).round().astype(np.int64))


def cpu_cells_per_step(w, budget_s):
    """Cells of a bounded oracle sample sized for about `budget_s` seconds of CPU work."""
    probe = evenly_spaced_cells(w.target.ncell, 64)
    _, t = oracle_sample(w, probe)
    rate = probe.size / max(t, 1e-6)
    return int(max(64, min(w.target.ncell, rate * budget_s)))


# ------------------------------------------------------------------------------- reference arm
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_2012_13173_b200 import workloads
    w = workloads.make(args.config, args.scale)
    total = max(1, args.steps + args.warmup)
    k = cpu_cells_per_step(w, min(20.0, 150.0 / total))
    cells = evenly_spaced_cells(w.target.ncell, k)
    threads = 0
    for _ in range(args.warmup):
        threads = oracle_sample(w, cells)[0].threads
    ts, nhit = [], 0
    for _ in range(args.steps):
        ref, t = oracle_sample(w, cells)
        ts.append(t); nhit = int(ref.counts.sum()); threads = ref.threads
    tot = sum(ts)
    value = cells.size * w.nchan * args.steps / tot
    sample = (f"{cells.size} evenly spaced cells of {w.target.ncell} per step, all {w.n} samples, fp64 brute force "
              f"(oracle/hcgrid_oracle.c as it stands)")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD_NAMES[args.config], "scale": args.scale, "n_samples": w.n,
                       "ncell": w.target.ncell, "nchan": w.nchan, "cells_per_step": int(cells.size)},
            "kernel_evals_per_s": nhit * args.steps / tot,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------- product arm
def run_product(args):
    import torch
    import torch.distributed as dist
    from paper_2012_13173_b200 import binding, roofline, workloads
    from paper_2012_13173_b200 import dist as hdist

    world, rank, local = hdist.env_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    # every rank grids one independent, identically shaped problem (weak scaling; the path has no
    # data-path collective: DESIGN.md "Multi-GPU")
    w = workloads.make(args.config, args.scale)
    units_total = None
    if args.shard == "rows" and world > 1:
        # strong scaling: ONE problem, every rank owns a band of target rows and the samples within the
        # support radius of it (paper_2012_13173_b200/dist.py); outputs are disjoint, no collective
        full = w.target
        units_total = full.ncell * w.nchan
        iy0, iy1 = hdist.row_band(full.ny, world, rank, align=4)
        m = hdist.band_sample_mask(w.lat, full, iy0, iy1, w.radius_deg)
        w.target = hdist.band_target(full, iy0, iy1)
        w.lon, w.lat, w.values = w.lon[m], w.lat[m], np.ascontiguousarray(w.values[m])
        w.weights = None if w.weights is None else w.weights[m]
    t = w.target
    g = binding.HCGrid(w.sigma_deg, w.radius_deg, w.nside, precision="f32", device=local)
    if args.kernel_function == "sinc":                 # variants, not the headline: DESIGN.md "Kernel functions"
        g.set_kernel(binding.KERNEL_TAPERED_SINC, 2.52, 1.55)
    elif args.kernel_function == "elliptical":
        g.set_kernel(binding.KERNEL_ELLIPTICAL_GAUSS, 0.5, 30.0)
    if args.explicit_cells:                            # the same cells handed over one by one (hcgrid_set_target_cells)
        if args.per_cell_path:
            g.set_option(binding.OPT_CELLS_AS_GRID, 0)     # do not recognise the grid: time the per-cell path itself
        cl, cb = t.cell_centers()
        g.set_target_cells(torch.from_numpy(cl).to(dev), torch.from_numpy(cb).to(dev))
    else:
        g.set_target_car(t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat)
    lon, lat = torch.from_numpy(w.lon).to(dev), torch.from_numpy(w.lat).to(dev)
    val = torch.from_numpy(w.values).to(dev)
    wts = None if w.weights is None else torch.from_numpy(w.weights).to(dev)
    ncell, nchan = t.ncell, w.nchan
    # the timed call returns what the north_star names: datacube and weight map.  The optional
    # contributing-sample counts (a parity output) are fetched by one extra, untimed call.
    cnt_t = torch.empty(ncell, dtype=torch.int32, device=dev)
    out = (torch.empty((ncell, nchan), dtype=torch.float32, device=dev),
           torch.empty(ncell, dtype=torch.float32, device=dev), None)

    def barrier():
        hdist.barrier(world, torch.cuda.synchronize)

    def step():
        g.grid(lon, lat, val, wts, want_counts=False, out=out)

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()

    # ---- timed region 1: K steps, device-resident inputs
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    launches = g.stats()["gpu_launches"] * args.steps

    # ---- timed region 2: the same K steps with the library's per-stage events (convolution kernel alone)
    g.set_option(binding.OPT_PROFILE, 1)
    stage = {k: [] for k in ("us_pixelise", "us_sort", "us_tables", "us_pack", "us_convolve", "us_total")}
    step(); torch.cuda.synchronize()
    # the stage events are read (a host synchronisation) after every fourth call only, so that the calls that are
    # measured run back to back like those of the timed region: after an idle gap the same kernels run 5-7 % slower
    for i in range(args.steps):
        step()
        if i % 4 == 3 or args.steps < 4:
            s = g.stats()
            for k in stage:
                stage[k].append(s[k])
    st = g.stats()
    # the same call with the count output (untimed for `value`; its convolution time is reported)
    us_conv_counts = []
    for _ in range(3):
        g.grid(lon, lat, val, wts, want_counts=True, out=(out[0], out[1], cnt_t))
        us_conv_counts.append(g.stats()["us_convolve"])
    g.set_option(binding.OPT_PROFILE, 0)

    # ---- timed region 3: end to end through hcgrid_grid_host, pinned host buffers
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_lon, h_lat, h_val = pin(w.lon), pin(w.lat), pin(w.values)
    h_wts = None if w.weights is None else pin(w.weights)
    h_out = (torch.empty((ncell, nchan), dtype=torch.float32).pin_memory(),
             torch.empty(ncell, dtype=torch.float32).pin_memory())
    h_out_np = tuple(x.numpy() for x in h_out) + (None,)

    def step_host():
        g.grid_host(h_lon.numpy(), h_lat.numpy(), h_val.numpy(), None if h_wts is None else h_wts.numpy(),
                    want_counts=False, out=h_out_np)

    for _ in range(2):
        step_host()
    barrier()
    e0.record()
    for _ in range(args.steps):
        step_host()
    e1.record()
    barrier()
    ms_e2e = e0.elapsed_time(e1)
    clocks = sampler.stop() if rank == 0 else None
    h2d = w.n * (16 + 4 * nchan + (4 if w.weights is not None else 0))
    d2h = ncell * (4 * nchan + 4)

    # ---- max over ranks
    ms_total, ms_e2e = hdist.max_over_ranks([ms_total, ms_e2e], world, dev)
    cnt = cnt_t.cpu().numpy().astype(np.int64)
    n_hit = int(cnt.sum())
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    if units_total is None:
        units = ncell * nchan * world
        value = hdist.whole_job_rate(ncell * nchan, world, args.steps, ms_total)
    else:
        units = units_total
        value = units_total * args.steps / (ms_total * 1e-3)
    hbm_gbs, hbm_src = load_peaks()
    t_conv = float(np.mean(stage["us_convolve"])) * 1e-6
    cand = roofline.count_candidates(w, max_rows=args.cand_rows)
    p_fp32_meas, p_mufu_meas = binding.measure_peaks(local)
    mdl = roofline.model(w.n, ncell, nchan, w.weights is not None, n_hit, cand["n_cand"], hbm_gbs,
                         want_counts=False)
    if mdl["bound"] == "hbm":
        rl = {"bound": "hbm", "achieved": mdl["bytes_unique"] / t_conv / 1e9, "peak": hbm_gbs, "unit": "GB/s"}
    elif mdl["bound"] == "mufu":
        rl = {"bound": "alu", "achieved": n_hit / t_conv / 1e9, "peak": roofline.P_MUFU_NOMINAL / 1e9,
              "unit": "G MUFU.EX2 thread-inst/s"}
    else:
        rl = {"bound": "alu", "achieved": mdl["fp32_inst"] / t_conv / 1e9, "peak": roofline.P_FP32_NOMINAL / 1e9,
              "unit": "G FP32-pipe thread-inst/s"}
    rl["frac"] = rl["achieved"] / rl["peak"]
    rl.update({
        "traffic": args.traffic if args.traffic is not None else (
            NCU_TRAFFIC[(args.config, st["kernel"])][0]
            if args.scale == 1.0 and (args.config, st["kernel"]) in NCU_TRAFFIC else None),
        "traffic_source": NCU_TRAFFIC.get((args.config, st["kernel"]), (None, None))[1] if args.traffic is None else "--traffic",
        "kernel": {1: "conv1_simple_f32", 2: "conv1_staged_f32", 3: "conv_general<f32>", 4: "conv_general<f64 pair>",
                   5: "conv_general<f64>", 6: "conv1_tile_f32", 7: "conv_mc_f32", 8: "conv_mc_tc_f32"}.get(st["kernel"], str(st["kernel"])),
        "kernel_us": t_conv * 1e6, "t_roof_us": mdl["t_roof_s"] * 1e6,
        "legs_us": {"fp32": mdl["t_fp32_s"] * 1e6, "mufu": mdl["t_mufu_s"] * 1e6, "hbm": mdl["t_hbm_s"] * 1e6},
        "n_hit": n_hit, "n_cand": cand["n_cand"], "n_cand_rows_counted": cand["rows_counted"],
        "algorithmic_fp32_inst_per_launch": mdl["fp32_inst"], "algorithmic_bytes_per_launch": mdl["bytes_unique"],
        "peak_source": "derived: 148 SMs x 128 FP32 lanes x 1.965 GHz (DESIGN.md); HBM " + hbm_src,
        "peak_measured_issue_rate": {"fp32_ginst_s": p_fp32_meas / 1e9, "mufu_ginst_s": p_mufu_meas / 1e9},
        "frac_of_measured_issue_rate": (mdl["fp32_inst"] / t_conv) / p_fp32_meas if p_fp32_meas > 0 else None,
        "hbm_gbs_achieved_unique_bytes": mdl["bytes_unique"] / t_conv / 1e9,
    })
    # the contract exactly as SURVEY.md 8d wrote it: F_a = 6 + nchan per accepted pair (the count increment always
    # charged) against the kernel that does write the count output
    if mdl["bound"] == "alu":
        t_cnt = float(np.median(us_conv_counts)) * 1e-6
        inst_s = cand["n_cand"] * roofline.F_D + n_hit * (6 + nchan + (1 if w.weights is not None else 0))
        rl["survey_contract"] = {"f_a": 6 + nchan, "fp32_inst": inst_s, "kernel_us_with_count_output": t_cnt * 1e6,
                                 "frac": inst_s / t_cnt / roofline.P_FP32_NOMINAL}

    # ---- oracle on this box's host cores, bounded sample
    cpu = None
    if world == 1 and not args.no_cpu_baseline and args.kernel_function == "gauss":
        k = cpu_cells_per_step(w, args.cpu_seconds)
        cells = evenly_spaced_cells(ncell, k)
        ref, tcpu = oracle_sample(w, cells)
        cpu = {"value": cells.size * nchan / tcpu, "unit": UNIT, "cores": ref.threads, "kind": "oracle",
               "sample": f"{cells.size} evenly spaced cells of {ncell}, all {w.n} samples, {tcpu:.1f} s",
               "kernel_evals_per_s": int(ref.counts.sum()) / tcpu}
        # the sample doubles as a parity spot check of the run that was just timed
        sys.path.insert(0, os.path.join(ROOT, "tests"))
        from parity import TOL_F32, compare
        chk = compare(out[0].cpu().numpy(), out[1].cpu().numpy(), cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32,
                      1.0 if w.weights is None else float(w.weights.max()), cells=cells)
        # max_rel_*: over the cells no pair within 1e-9 rad of the support radius can move (reading c4);
        # the few cells that hold such a pair are checked by compare() with that pair's weight as slack
        cpu["parity_on_sample"] = {"max_rel_w": chk["max_rel_w_clear"], "max_rel_v": chk["max_rel_v_clear"],
                                   "counts": "exact", "cells_with_boundary_pairs": chk["cells_with_boundary_pairs"],
                                   "max_rel_w_all_cells": chk["max_rel_w"], "max_rel_v_all_cells": chk["max_rel_v"]}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_total / args.steps, "higher_is_better": True,
        "scaling": "weak" if units_total is None else "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": WORKLOAD_NAMES[args.config], "scale": args.scale, "n_samples": w.n, "ncell": ncell,
                   "nchan": nchan, "nside": w.nside, "sigma_arcmin": w.sigma_deg * 60, "radius_arcmin": w.radius_deg * 60,
                   "l2": "inputs larger than L2 (no flush): lon/lat/values %.0f MB + packed records %.0f MB per step"
                         % (h2d / 1e6, st["n_kept"] * 16 / 1e6),
                   "coarsen": st["coarsen"], "coarsen_y": st["coarsen_y"], "subpix_bits": st["subpix_bits"],
                   "preorder": {1: "radix sort", 2: "counting sort"}.get(st["preorder"], "?"),
                   "e2e_path": "hcgrid_grid_host, pinned buffers; inputs of 64 MB or more are copied in 4 pieces and gridded as they arrive", "per_rank": "one independent problem" if units_total is None else "a band of target rows + its samples (rank 0's figures in roofline / stages)",
                   "outputs": "datacube + weight map (count output off in the timed calls)",
                   "kernel_function": args.kernel_function,
                   "target": ("per-cell lon/lat (hcgrid_set_target_cells), grid recognition " + ("off" if args.per_cell_path else "on"))
                             if args.explicit_cells else "CAR parameters"},
        "kernel_evals_per_s": n_hit * world * args.steps / (ms_total * 1e-3),
        "conv_kernel": {"us": t_conv * 1e6, "cell_channels_per_s": ncell * nchan / t_conv,
                        "kernel_evals_per_s": n_hit / t_conv,
                        "us_with_count_output": float(np.median(us_conv_counts))},
        "stages_us": {k[3:]: float(np.mean(v)) for k, v in stage.items()},
        "roofline": rl,
        "cpu_baseline": cpu,
        "e2e": {"value": units * args.steps / (ms_e2e * 1e-3), "unit": UNIT, "ms_per_step": ms_e2e / args.steps,
                "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
        "gpu_launches": launches,
        "clocks": clocks,
    }
    print(json.dumps(line), flush=True)
    g.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


# ------------------------------------------------------------------------------- N ranks on one node
def free_port() -> int:
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def child_envs(n: int, port: int, base=None) -> list:
    """Environment of each of the N ranks `python bench.py --gpus N` starts when it is not already
    running under torchrun: one process per GPU, rendezvous on 127.0.0.1 (the container hostname
    may not resolve)."""
    base = dict(os.environ if base is None else base)
    return [dict(base, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(n), LOCAL_WORLD_SIZE=str(n),
                 MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port)) for r in range(n)]


def launch_ranks(n: int, argv: list) -> int:
    """Start N copies of this script, one per GPU; rank 0 prints the JSON line.  NCCL's own log
    (NCCL_DEBUG) is passed through untouched."""
    procs = [subprocess.Popen([sys.executable, os.path.abspath(__file__), *argv], env=env)
             for env in child_envs(n, free_port())]
    rcs = [p.wait() for p in procs]
    bad = [(r, rc) for r, rc in enumerate(rcs) if rc != 0]
    if bad:
        sys.stderr.write(f"bench.py: ranks failed (rank, exit code): {bad}\n")
    return max(abs(rc) for rc in rcs)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="product", choices=["product", "reference"])
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--scale", type=float, default=1.0)
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cand-rows", type=int, default=None, help="count N_cand on this many rows and scale")
    ap.add_argument("--shard", default="replicas", choices=["replicas", "rows"],
                    help="N > 1: independent replicas (weak scaling, default) or one problem cut into row bands (strong)")
    ap.add_argument("--kernel-function", default="gauss", choices=["gauss", "sinc", "elliptical"],
                    help="kernel function of Eq. 1: the paper's Gaussian (default), the tapered sinc (a 2.52, b 1.55) or "
                         "the elliptical Gaussian (ratio 0.5, position angle 30 deg)")
    ap.add_argument("--explicit-cells", action="store_true",
                    help="hand the target over as per-cell lon/lat (hcgrid_set_target_cells) instead of CAR parameters")
    ap.add_argument("--per-cell-path", action="store_true",
                    help="with --explicit-cells: switch the grid recognition off (HCGRID_OPT_CELLS_AS_GRID 0)")
    ap.add_argument("--traffic", type=float, default=None,
                    help="dram bytes per launch of the convolution kernel from the committed ncu capture")
    args = ap.parse_args()
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    world = os.environ.get("WORLD_SIZE")
    if world is None and args.gpus > 1:
        return launch_ranks(args.gpus, sys.argv[1:])       # not under torchrun: start the N ranks here
    if world is not None and int(world) != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but the launcher started WORLD_SIZE={world} ranks")
    if args.impl == "reference":
        return run_reference(args)
    return run_product(args)


if __name__ == "__main__":
    sys.exit(main())
