"""Comparison of a CUDA-path result with the oracle's, at the bar BASELINE.json's north_star
states: counts bit-exact up to the pairs within 1e-9 rad of the
support boundary, weight map and datacube within `tol` relative, NaN where W == 0."""
import math

import numpy as np

TOL_F32 = 1e-5     # north_star: "within 1e-5 relative (fp32 accumulation)"
TOL_F64 = 1e-12    # north_star: "or 1e-12 (fp64 mode)"


def compare(cube, wmap, counts, ref, sigma_deg, radius_deg, tol, qmax=1.0, cells=None):
    """ref: oracle.OracleResult (optionally of the subset `cells` of the flat cell index).
    Returns a dict of the worst normalised errors; raises AssertionError on a violation."""
    cube = np.asarray(cube, dtype=np.float64)
    wmap = np.asarray(wmap, dtype=np.float64)
    if cube.ndim == 1:
        cube = cube[:, None]
    if cells is not None:
        cube, wmap = cube[cells], wmap[cells]
        counts = None if counts is None else np.asarray(counts)[cells]
    nb = ref.near_boundary
    # a pair within 1e-9 rad of the boundary may fall on either side: it moves the count by
    # one and W by at most q * exp(-R^2 / 2 sigma^2)
    w_edge = qmax * math.exp(-0.5 * (radius_deg / sigma_deg) ** 2) * 1.001
    if counts is not None:
        dc = np.abs(np.asarray(counts, dtype=np.int64) - ref.counts)
        bad = np.flatnonzero(dc > nb)
        assert bad.size == 0, (f"{bad.size} cells with wrong contributing-sample count; first: cell {bad[0]} "
                               f"gpu {int(np.asarray(counts)[bad[0]])} oracle {int(ref.counts[bad[0]])} "
                               f"near-boundary {int(nb[bad[0]])}")
    empty = ref.weightmap == 0
    # weight map
    errw = np.abs(wmap - ref.weightmap)
    alloww = tol * ref.weightmap + nb * w_edge
    badw = np.flatnonzero(errw > alloww)
    assert badw.size == 0, (f"{badw.size} weight-map cells out of tolerance; first: cell {badw[0]} gpu "
                            f"{wmap[badw[0]]!r} oracle {ref.weightmap[badw[0]]!r}")
    # datacube
    assert np.array_equal(np.isnan(cube), np.isnan(ref.datacube)), "NaN pattern (empty cells) differs"
    ok = ~empty
    scale = np.maximum(np.abs(ref.datacube[ok]), ref.absmap[ok])
    errv = np.abs(cube[ok] - ref.datacube[ok])
    # a pair within 1e-9 rad of the boundary (reading c4) may fall on either side: it changes V by at most
    # w_edge (|v_s| + |V|) / W <= 2 w_edge max|v| / W; only cells that hold such a pair (nb > 0) get this slack
    slack = (nb[ok] * w_edge / np.maximum(ref.weightmap[ok], 1e-300))[:, None] * 2.0 * ref.vmax
    allowv = tol * scale + slack
    badv = np.argwhere(errv > allowv)
    assert badv.shape[0] == 0, (f"{badv.shape[0]} datacube entries out of tolerance; first: {badv[0]} gpu "
                                f"{cube[ok][tuple(badv[0])]!r} oracle {ref.datacube[ok][tuple(badv[0])]!r}")
    nz = ref.weightmap > 0
    clear = nz & (nb == 0)          # cells no boundary pair (reading c4) can move
    relv = errv / np.maximum(scale, 1e-300)
    return {
        "max_rel_w": float(np.max(errw[nz] / ref.weightmap[nz])) if nz.any() else 0.0,
        "max_rel_v": float(np.max(relv)) if ok.any() else 0.0,
        "max_rel_w_clear": float(np.max(errw[clear] / ref.weightmap[clear])) if clear.any() else 0.0,
        "max_rel_v_clear": float(np.max(relv[(nb == 0)[ok]])) if clear.any() else 0.0,
        "cells_with_boundary_pairs": int(np.count_nonzero(nb)),
        "near_boundary_pairs": int(nb.sum()),
        "n_hit": int(ref.counts.sum()),
    }


KFLOOR_F32 = 5e-7   # absolute accuracy of one fp32 kernel evaluation where the kernel has zeros (see compare_signed)
KFLOOR_F64 = 1e-15


def compare_signed(cube, wmap, counts, ref, w_edge, tol, kfloor, qmax=1.0, vmax=None, cond=0.05):
    """The same bar for kernel functions with negative lobes (ref from oracle.grid(kernel=...)).
    W is a sum of signed terms, so its error is measured against sum |q w| (ref.abswmap), plus a
    floor per contributing pair: the fp32 pair arithmetic delivers d to ~1.5e-7 relative, which keeps
    a Gaussian weight accurate RELATIVE to itself, but at a zero of the sinc the weight's error is
    |omega'(d)| d 1.5e-7 <= ~2e-7 ABSOLUTE (|y cos y / y| <= 1) however small omega is there; hence
    dW <= tol * sum |q w| + kfloor * count * qmax and dS likewise with |v| <= vmax.
    V = S / W inherits dS / |W| + |V| dW / |W| and is compared only where |W| >= cond * sum |q w|
    (below that V is ill-conditioned by construction: the oracle's own V moves with the last bits of
    W).  w_edge bounds |q omega(R)| for the pairs within 1e-9 rad of the support boundary."""
    cube = np.asarray(cube, dtype=np.float64)
    wmap = np.asarray(wmap, dtype=np.float64)
    if cube.ndim == 1:
        cube = cube[:, None]
    nb = ref.near_boundary
    if counts is not None:
        dc = np.abs(np.asarray(counts, dtype=np.int64) - ref.counts)
        assert np.all(dc <= nb), f"{int(np.sum(dc > nb))} cells with wrong contributing-sample count"
    if vmax is None:
        vmax = 1.0
    errw = np.abs(wmap - ref.weightmap)
    alloww = tol * ref.abswmap + kfloor * ref.counts * qmax + nb * w_edge
    badw = np.flatnonzero(errw > alloww)
    assert badw.size == 0, (f"{badw.size} weight-map cells out of tolerance; first: cell {badw[0]} gpu "
                            f"{wmap[badw[0]]!r} oracle {ref.weightmap[badw[0]]!r} scale {ref.abswmap[badw[0]]!r}")
    empty = ref.counts == 0
    assert np.all(np.isnan(cube[empty])), "cells without contributors must be NaN"
    ok = (~empty) & (np.abs(ref.weightmap) >= cond * ref.abswmap) & (ref.abswmap > 0)
    aw = np.abs(ref.weightmap[ok])
    a_un = ref.absmap[ok] * aw[:, None]                                   # sum |q w||v|
    e_s = tol * a_un + (kfloor * ref.counts[ok] * qmax * vmax + nb[ok] * w_edge * vmax)[:, None]
    e_w = alloww[ok]
    allowv = e_s / aw[:, None] + np.abs(ref.datacube[ok]) * (e_w / aw)[:, None]
    errv = np.abs(cube[ok] - ref.datacube[ok])
    badv = np.argwhere(errv > allowv)
    assert badv.shape[0] == 0, (f"{badv.shape[0]} datacube entries out of tolerance; first: {badv[0]} gpu "
                                f"{cube[ok][tuple(badv[0])]!r} oracle {ref.datacube[ok][tuple(badv[0])]!r}")
    return {"max_rel_w": float(np.max(errw / np.maximum(alloww, 1e-300))),
            "max_rel_v": float(np.max(errv / np.maximum(allowv, 1e-300))) if ok.any() else 0.0,
            "cells_compared": int(ok.sum()), "negative_w_cells": int(np.sum(ref.weightmap < 0))}
