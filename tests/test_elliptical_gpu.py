"""GPU parity for the elliptical Gaussian kernel (reading c21):
hcgrid_set_kernel(ELLIPTICAL_GAUSS, ratio, PA) against oracle.grid(kernel=(2, ratio, PA)), element by element, at the
ordinary bar of tests/parity.py (weights are positive: 1e-5 in fp32 mode, 1e-12 in fp64 mode).
"""
import numpy as np
import pytest

from paper_2012_13173_b200 import workloads

from parity import TOL_F32, TOL_F64, compare

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

RATIO, PA = 0.5, 30.0
MINI = {1: 1.0, 2: 0.03, 3: 0.006, 4: 0.012, 5: 0.004}


def _dev(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


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


def _oracle(oracle, w, ratio=RATIO, pa=PA):
    cl, cb = w.target.cell_centers()
    return oracle.grid(w.sigma_deg, w.radius_deg, cl, cb, w.lon, w.lat, w.values, w.weights,
                       kernel=(oracle.ELLIPTICAL_GAUSS, ratio, pa))


def _cmp(cube, wmap, cnt, ref, w, precision, ratio=RATIO):
    qmax = 1.0 if w.weights is None else float(w.weights.max())
    # the largest weight a pair on the support boundary can have is that of the wider axis
    return compare(cube, wmap, cnt, ref, w.sigma_deg * max(1.0, ratio), w.radius_deg,
                   TOL_F64 if precision == "f64" else TOL_F32, qmax)


@pytest.mark.parametrize("precision", ["f32", "f64"])
@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_elliptical_config_miniatures(oracle, cfg, precision):
    w = workloads.make(cfg, MINI[cfg])
    ref = _oracle(oracle, w)
    cube, wmap, cnt, st = _gpu(w, precision, (2, RATIO, PA))
    # fp32, one channel, plate-carree: the tile kernel; otherwise the general kernels
    assert st["kernel"] == (6 if precision == "f32" and w.nchan == 1 else (3 if precision == "f32" else 5))
    r = _cmp(cube, wmap, cnt, ref, w, precision)
    assert r["n_hit"] > 0
    # and the kernel is not the circular one: the weight map differs visibly from the Gaussian oracle's
    cl, cb = w.target.cell_centers()
    g = oracle.grid(w.sigma_deg, w.radius_deg, cl, cb, w.lon, w.lat, w.values, w.weights)
    assert np.abs(g.weightmap - ref.weightmap).max() > 1e-2 * g.weightmap.max()


@pytest.mark.parametrize("cfg", [1, 3, 5])
@pytest.mark.parametrize("variant", ["general", "tile1x1", "tile2x2", "tile4x2", "tile4x2split2"])
def test_elliptical_kernel_variants(oracle, cfg, variant):
    from paper_2012_13173_b200 import binding
    w = workloads.make(cfg, MINI[cfg])
    ref = _oracle(oracle, w)
    if variant == "general":
        opts, want = {binding.OPT_KERNEL: binding.KERNEL_GENERAL}, 3
    else:
        gx, gy = int(variant[4]), int(variant[6])
        opts, want = {binding.OPT_KERNEL: binding.KERNEL_TILE, binding.OPT_COARSEN: gx, binding.OPT_COARSEN_Y: gy}, 6
        if variant.endswith("split2"):
            opts[binding.OPT_SPLIT] = 2
    cube, wmap, cnt, st = _gpu(w, "f32", (2, RATIO, PA), options=opts)
    assert st["kernel"] == want
    _cmp(cube, wmap, cnt, ref, w, "f32")


@pytest.mark.parametrize("ratio,pa", [(0.4, 0.0), (0.4, 90.0), (0.7, -45.0), (0.6, 200.0), (1.6, 75.0), (1.0, 12.0)])
@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_elliptical_axis_ratios_and_position_angles(oracle, ratio, pa, precision):
    """Axis along the meridian, along the parallel, in every quadrant; ratio above 1 (the axis at the position angle
    is then the minor one) and ratio 1 (the circular kernel through the elliptical code)."""
    w = workloads.make(3, MINI[3])
    ref = _oracle(oracle, w, ratio, pa)
    cube, wmap, cnt, _ = _gpu(w, precision, (2, ratio, pa))
    _cmp(cube, wmap, cnt, ref, w, precision, ratio)
    if ratio == 1.0:
        cl, cb = w.target.cell_centers()
        g = oracle.grid(w.sigma_deg, w.radius_deg, cl, cb, w.lon, w.lat, w.values, w.weights)
        compare(cube, wmap, cnt, g, w.sigma_deg, w.radius_deg, TOL_F64 if precision == "f64" else TOL_F32)


def test_elliptical_quarter_turn_swaps_the_axes_on_the_device(oracle):
    """(s1, ratio, PA) and (ratio s1, 1 / ratio, PA + 90) are one ellipse: two device runs with different constants
    agree with each other as closely as each agrees with the oracle."""
    w = workloads.make(1, 1.0)
    ref = _oracle(oracle, w, 0.5, 20.0)
    c1, w1, n1, _ = _gpu(w, "f32", (2, 0.5, 20.0))
    w2l = workloads.Workload(w.name, w.config, w.scale, w.lon, w.lat, w.values, w.weights, w.sigma_deg * 0.5,
                             w.radius_deg, w.nside, w.target)
    c2, w2, n2, _ = _gpu(w2l, "f32", (2, 2.0, 110.0))
    _cmp(c1, w1, n1, ref, w, "f32", 0.5)
    compare(c2, w2, n2, ref, w.sigma_deg, w.radius_deg, TOL_F32)
    assert np.array_equal(n1, n2)


@pytest.mark.parametrize("precision", ["f32", "f64"])
@pytest.mark.parametrize("lat_c,sigma_arcmin", [(88.6, 6.0), (-89.2, 4.0), (40.0, 40.0)])
def test_elliptical_polar_caps_and_wide_kernels(oracle, lat_c, sigma_arcmin, precision):
    """Where the small-angle series is not valid (a pole in reach, or R > 0.05 rad) the fp64 pair arithmetic with the
    full functions runs in both modes; per-cell target, so the general kernel."""
    rng = np.random.default_rng([13173, 909, int(abs(lat_c) * 10)])
    sigma = sigma_arcmin / 60.0
    radius = 3.0 * sigma
    n = 6000
    half = 6 * sigma
    lat = np.clip(lat_c + rng.uniform(-half, half, n), -90.0, 90.0)
    if abs(lat_c) > 80:
        lon = rng.uniform(0.0, 360.0, n)
    else:
        lon = np.mod(359.0 + rng.uniform(-half, half, n) / np.cos(np.deg2rad(lat_c)), 360.0)
    val = rng.standard_normal((n, 3)).astype(np.float32)
    wts = rng.uniform(0.5, 1.5, n).astype(np.float32)
    m = 120
    cb = np.clip(lat_c + rng.uniform(-0.7 * half, 0.7 * half, m), -89.999, 89.999)
    cl = rng.uniform(0.0, 360.0, m) if abs(lat_c) > 80 else np.mod(359.0 + rng.uniform(-half, half, m), 360.0)
    ref = oracle.grid(sigma, radius, cl, cb, lon, lat, val, wts, kernel=(oracle.ELLIPTICAL_GAUSS, 0.5, 65.0))
    assert ref.counts.sum() > 0
    from paper_2012_13173_b200 import binding
    g = binding.HCGrid(sigma, radius, 256, precision=precision)
    g.set_kernel(binding.KERNEL_ELLIPTICAL_GAUSS, 0.5, 65.0)
    g.set_target_cells(_dev(cl), _dev(cb))
    cube, wmap, cnt = g.grid(_dev(lon), _dev(lat), _dev(val), _dev(wts))
    torch.cuda.synchronize()
    g.close()
    compare(cube.cpu().numpy(), wmap.cpu().numpy(), cnt.cpu().numpy(), ref, sigma, radius,
            TOL_F64 if precision == "f64" else TOL_F32, 1.5)


@pytest.mark.parametrize("cfg,precision", [(3, "f32"), (4, "f32"), (2, "f64")])
def test_elliptical_accumulated_batches(oracle, cfg, precision):
    w = workloads.make(cfg, MINI[cfg])
    ref = _oracle(oracle, w)
    cube, wmap, cnt, _ = _gpu(w, precision, (2, RATIO, PA), batches=3)
    _cmp(cube, wmap, cnt, ref, w, precision)


def test_elliptical_validates_and_switches_back(oracle):
    from paper_2012_13173_b200 import binding
    w = workloads.make(1, 1.0)
    g = binding.HCGrid(w.sigma_deg, w.radius_deg, w.nside)
    t = w.target
    g.set_target_car(t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat)
    for bad in ((2, 0.0, 10.0), (2, -0.5, 10.0), (2, float("nan"), 1.0), (2, 0.5, float("inf"))):
        with pytest.raises(binding.HCGridError):
            g.set_kernel(*bad)
    lon, lat, val = _dev(w.lon), _dev(w.lat), _dev(w.values)
    g.set_kernel(binding.KERNEL_ELLIPTICAL_GAUSS, RATIO, PA)
    g.set_option(binding.OPT_KERNEL, binding.KERNEL_SIMPLE)
    with pytest.raises(binding.HCGridError):            # the simple kernel evaluates the circular Gaussian only
        g.grid(lon, lat, val)
    g.set_option(binding.OPT_KERNEL, binding.KERNEL_AUTO)
    c1, w1, n1 = g.grid(lon, lat, val)
    g.set_kernel(binding.KERNEL_GAUSS)
    c0, w0, n0 = g.grid(lon, lat, val)
    torch.cuda.synchronize()
    cl, cb = t.cell_centers()
    ref = oracle.grid(w.sigma_deg, w.radius_deg, cl, cb, w.lon, w.lat, w.values)
    compare(c0.cpu().numpy(), w0.cpu().numpy(), n0.cpu().numpy(), ref, w.sigma_deg, w.radius_deg, TOL_F32)
    assert torch.equal(n0, n1) and not torch.equal(w0, w1)
    g.close()
