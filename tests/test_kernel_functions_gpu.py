"""GPU parity for kernel functions other than the paper's Gaussian (PAPER.md:186
names the sinc): hcgrid_set_kernel(TAPERED_SINC) against oracle.grid(kernel=...), element by element.

Bar for signed weights (tests/parity.py compare_signed): counts exact up to boundary pairs; W within
tol * sum |q w| + the per-pair evaluation floor; V = S / W with both errors propagated, where |W| >= 5 % of sum |q w|.
"""
import math

import numpy as np
import pytest

from paper_2012_13173_b200 import workloads

from parity import KFLOOR_F32, KFLOOR_F64, TOL_F32, TOL_F64, compare, compare_signed

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

A, B = 2.52, 1.55


def _dev(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


def _w_edge(w, a=A):
    q = 1.0 if w.weights is None else float(w.weights.max())
    return q * math.exp(-(w.radius_deg / (a * w.sigma_deg)) ** 2) * 1.001


def _gpu(w, precision, kernel, explicit_cells=False, options=None, batches=None):
    from paper_2012_13173_b200 import binding
    g = binding.HCGrid(w.sigma_deg, w.radius_deg, w.nside, precision=precision)
    for k, v in (options or {}).items():
        g.set_option(k, v)
    g.set_kernel(*kernel)
    t = w.target
    if explicit_cells:
        cl, cb = t.cell_centers()
        g.set_target_cells(_dev(cl), _dev(cb))
    else:
        g.set_target_car(t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat)
    wts = None if w.weights is None else _dev(w.weights)
    if batches is None:
        cube, wmap, cnt = g.grid(_dev(w.lon), _dev(w.lat), _dev(w.values), wts)
    else:
        edges = np.linspace(0, w.n, batches + 1).astype(int)
        for lo, hi in zip(edges[:-1], edges[1:]):
            g.accumulate(_dev(w.lon[lo:hi]), _dev(w.lat[lo:hi]), _dev(w.values[lo:hi]),
                         None if w.weights is None else _dev(w.weights[lo:hi]))
        cube, wmap, cnt = g.finalize()
    torch.cuda.synchronize()
    st = g.stats()
    g.close()
    return cube.cpu().numpy(), wmap.cpu().numpy(), cnt.cpu().numpy(), st


def _cmp(cube, wmap, cnt, ref, w, precision):
    f64 = precision == "f64"
    qmax = 1.0 if w.weights is None else float(w.weights.max())
    return compare_signed(cube, wmap, cnt, ref, _w_edge(w), TOL_F64 if f64 else TOL_F32,
                          KFLOOR_F64 if f64 else KFLOOR_F32, qmax=qmax, vmax=float(np.abs(w.values).max()))


def _oracle(oracle, w, kernel):
    cl, cb = w.target.cell_centers()
    return oracle.grid(w.sigma_deg, w.radius_deg, cl, cb, w.lon, w.lat, w.values, w.weights, kernel=kernel)


MINI = {1: 1.0, 2: 0.03, 3: 0.006, 4: 0.012, 5: 0.004}


@pytest.mark.parametrize("precision", ["f32", "f64"])
@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_tapered_sinc_config_miniatures(oracle, cfg, precision):
    w = workloads.make(cfg, MINI[cfg])
    ref = _oracle(oracle, w, (oracle.TAPERED_SINC, A, B))
    cube, wmap, cnt, st = _gpu(w, precision, (1, A, B))
    # fp32, one channel, plate-carree: the tile kernel; otherwise the general kernels
    assert st["kernel"] == (6 if precision == "f32" and w.nchan == 1 else (3 if precision == "f32" else 5))
    r = _cmp(cube, wmap, cnt, ref, w, precision)
    assert r["cells_compared"] > 0.5 * w.target.ncell


@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_tapered_sinc_negative_weight_cells_and_arbitrary_cells(oracle, precision):
    """Sparse samples and R = 3 sigma > b sigma: some cells see only the negative lobe (W < 0) and V is
    still S / W there; per-cell lon/lat target."""
    rng = np.random.default_rng(11)
    n = 80
    w0 = workloads.make(1, 1.0)
    t = w0.target
    lon = t.lon0 + rng.uniform(0, t.nx * t.dlon, n)
    lat = t.lat0 + rng.uniform(0, t.ny * t.dlat, n)
    val = rng.normal(1.0, 0.3, (n, 2)).astype(np.float32)
    w = workloads.Workload("sparse", 1, 1.0, lon, lat, val, None, w0.sigma_deg, 3 * w0.sigma_deg, w0.nside, t)
    ref = _oracle(oracle, w, (oracle.TAPERED_SINC, A, B))
    assert np.sum(ref.weightmap < 0) > 0
    from paper_2012_13173_b200 import binding
    cube, wmap, cnt, st = _gpu(w, precision, (1, A, B), explicit_cells=True, options={binding.OPT_CELLS_AS_GRID: 0})
    assert st["kernel"] in (3, 5)                      # the per-cell path: general kernels
    r = _cmp(cube, wmap, cnt, ref, w, precision)
    assert r["negative_w_cells"] > 0
    neg = (ref.weightmap < 0) & (np.abs(ref.weightmap) >= 0.05 * ref.abswmap)
    assert np.all(np.isfinite(cube[neg]))


@pytest.mark.parametrize("cfg", [1, 3, 5])
@pytest.mark.parametrize("variant", ["general", "tile1x1", "tile2x2", "tile4x2", "tile4x2split2"])
def test_tapered_sinc_kernel_variants(oracle, cfg, variant):
    from paper_2012_13173_b200 import binding
    w = workloads.make(cfg, MINI[cfg])
    ref = _oracle(oracle, w, (oracle.TAPERED_SINC, A, B))
    if variant == "general":
        opts, want = {binding.OPT_KERNEL: binding.KERNEL_GENERAL}, 3
    else:
        gx, gy = int(variant[4]), int(variant[6])
        opts, want = {binding.OPT_KERNEL: binding.KERNEL_TILE, binding.OPT_COARSEN: gx, binding.OPT_COARSEN_Y: gy}, 6
        if variant.endswith("split2"):
            opts[binding.OPT_SPLIT] = 2
    cube, wmap, cnt, st = _gpu(w, "f32", (1, A, B), options=opts)
    assert st["kernel"] == want
    _cmp(cube, wmap, cnt, ref, w, "f32")


def test_tapered_sinc_with_huge_b_is_the_gaussian_path(oracle):
    """b -> infinity leaves exp(-(d / (a sigma))^2): the general kernel's tapered-sinc branch must then
    agree with the Gaussian oracle of width a sigma / sqrt 2 at the ordinary 1e-5 bar."""
    w = workloads.make(3, 0.006)
    cl, cb = w.target.cell_centers()
    ref = oracle.grid(A * w.sigma_deg / math.sqrt(2.0), w.radius_deg, cl, cb, w.lon, w.lat, w.values, w.weights)
    cube, wmap, cnt, _ = _gpu(w, "f32", (1, A, 1e9))
    compare(cube, wmap, cnt, ref, A * w.sigma_deg / math.sqrt(2.0), w.radius_deg, TOL_F32)


def test_set_kernel_switches_back_and_validates(oracle):
    from paper_2012_13173_b200 import binding
    w = workloads.make(1, 1.0)
    g = binding.HCGrid(w.sigma_deg, w.radius_deg, w.nside)
    t = w.target
    g.set_target_car(t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat)
    for bad in ((1, 0.0, 1.0), (1, 2.0, -1.0), (5, 1.0, 1.0), (1, float("nan"), 1.0)):
        with pytest.raises(binding.HCGridError):
            g.set_kernel(*bad)
    lon, lat, val = _dev(w.lon), _dev(w.lat), _dev(w.values)
    g.set_kernel(binding.KERNEL_TAPERED_SINC, A, B)
    g.set_option(binding.OPT_KERNEL, binding.KERNEL_STAGED)
    with pytest.raises(binding.HCGridError):            # the staged kernel evaluates the Gaussian only
        g.grid(lon, lat, val)
    g.set_option(binding.OPT_KERNEL, binding.KERNEL_AUTO)
    c1, w1, n1 = g.grid(lon, lat, val)
    assert g.stats()["kernel"] == 6
    g.set_kernel(binding.KERNEL_GAUSS)
    c0, w0, n0 = g.grid(lon, lat, val)
    torch.cuda.synchronize()
    assert g.stats()["kernel"] == 6                      # back on the tile kernel
    cl, cb = t.cell_centers()
    ref = oracle.grid(w.sigma_deg, w.radius_deg, cl, cb, w.lon, w.lat, w.values)
    compare(c0.cpu().numpy(), w0.cpu().numpy(), n0.cpu().numpy(), ref, w.sigma_deg, w.radius_deg, TOL_F32)
    assert torch.equal(n0, n1) and not torch.equal(w0, w1)
    g.accumulate(lon, lat, val)
    with pytest.raises(binding.HCGridError):            # not while an accumulation is open
        g.set_kernel(binding.KERNEL_TAPERED_SINC, A, B)
    g.finalize()
    g.close()


@pytest.mark.parametrize("cfg,precision", [(3, "f32"), (4, "f32"), (2, "f64")])
def test_tapered_sinc_accumulated_batches(oracle, cfg, precision):
    w = workloads.make(cfg, MINI[cfg])
    ref = _oracle(oracle, w, (oracle.TAPERED_SINC, A, B))
    cube, wmap, cnt, _ = _gpu(w, precision, (1, A, B), batches=3)
    _cmp(cube, wmap, cnt, ref, w, precision)
