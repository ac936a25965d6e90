"""GPU parity: the CUDA path (through the C-ABI, via the thin binding) against the brute-force
fp64 oracle, element by element on the same seeded inputs.

Bar (BASELINE.json north_star; tests/parity.py): contributing-sample
counts bit-exact up to the pairs within 1e-9 rad of the support boundary, weight map and
datacube within 1e-5 relative (fp32 mode) or 1e-12 (fp64 mode), NaN where W == 0.

Sizes: miniatures of every BASELINE config (same density / kernel / nside, smaller patch;
several warp tasks, several staging chunks and a ragged tail each) in full, and the
full-size configs in the launch configuration bench.py times, on sampled cells the oracle
computes one by one.
"""
import numpy as np
import pytest

from paper_2012_13173_b200 import workloads

from parity import TOL_F32, TOL_F64, compare

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _dev(a, dtype=None):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype).cuda()


def run_gpu(w, precision="f32", options=None, explicit_cells=False, nside=None, want_counts=True):
    from paper_2012_13173_b200 import binding
    g = binding.HCGrid(w.sigma_deg, w.radius_deg, nside or w.nside, precision=precision)
    for k, v in (options or {}).items():
        g.set_option(k, v)
    t = w.target
    if explicit_cells:
        cl, cb = t.cell_centers()
        g.set_target_cells(_dev(cl), _dev(cb))
    else:
        g.set_target_car(t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat)
    cube, wmap, cnt = g.grid(_dev(w.lon), _dev(w.lat), _dev(w.values),
                             None if w.weights is None else _dev(w.weights), want_counts=want_counts)
    torch.cuda.synchronize()
    st = g.stats()
    g.close()
    return cube.cpu().numpy(), wmap.cpu().numpy(), None if cnt is None else cnt.cpu().numpy(), st


def run_oracle(oracle, w, cells=None):
    cl, cb = w.target.cell_centers()
    if cells is not None:
        cl, cb = cl[cells], cb[cells]
    return oracle.grid(w.sigma_deg, w.radius_deg, cl, cb, w.lon, w.lat, w.values, w.weights)


def qmax(w):
    return 1.0 if w.weights is None else float(w.weights.max())


MINI = {1: 1.0, 2: 0.03, 3: 0.006, 4: 0.012, 5: 0.004}
_cache = {}


def mini(oracle, cfg):
    if cfg not in _cache:
        w = workloads.make(cfg, MINI[cfg])
        _cache[cfg] = (w, run_oracle(oracle, w))
    return _cache[cfg]


# ------------------------------------------------------------ every config, both precisions
@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_config_miniature_f32(oracle, cfg):
    w, ref = mini(oracle, cfg)
    cube, wmap, cnt, st = run_gpu(w, "f32")
    r = compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32, qmax(w))
    assert r["n_hit"] > 0
    assert st["gpu_launches"] >= 4


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_config_miniature_f64(oracle, cfg):
    w, ref = mini(oracle, cfg)
    # fp64 mode compares on the explicit cell arrays the oracle used (SURVEY 8c fp64 pin 2)
    cube, wmap, cnt, _ = run_gpu(w, "f64", explicit_cells=(cfg % 2 == 0))
    assert cube.dtype == np.float64 and wmap.dtype == np.float64
    compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F64, qmax(w))


# ------------------------------------------------------------ every kernel variant / coarsening
# stats()["kernel"] of each forced variant: simple 1, fp64 pair 4, general 3, staged 2, tile 6
KERNEL_IDS = {1: 1, 2: 4, 3: 3, 4: 2, 5: 6}


@pytest.mark.parametrize("cfg", [1, 3, 5])
@pytest.mark.parametrize("kernel", [1, 2, 3, 4, 5])
def test_kernel_variants(oracle, cfg, kernel):
    from paper_2012_13173_b200 import binding
    w, ref = mini(oracle, cfg)
    cube, wmap, cnt, st = run_gpu(w, "f32", {binding.OPT_KERNEL: kernel})
    assert st["kernel"] == KERNEL_IDS[kernel]
    compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32, qmax(w))


def test_auto_kernel_is_the_tile_kernel_on_car_targets(oracle):
    w, ref = mini(oracle, 3)
    _, _, _, st = run_gpu(w, "f32")
    assert st["kernel"] == 6 and st["coarsen"] * st["coarsen_y"] >= 2


@pytest.mark.parametrize("coarsen", [1, 2, 4, 8])
@pytest.mark.parametrize("cfg", [1, 5])
def test_coarsening_simple_and_staged(oracle, cfg, coarsen):
    from paper_2012_13173_b200 import binding
    w, ref = mini(oracle, cfg)
    for kernel in (binding.KERNEL_SIMPLE, binding.KERNEL_STAGED):
        cube, wmap, cnt, st = run_gpu(w, "f32", {binding.OPT_COARSEN: coarsen, binding.OPT_KERNEL: kernel})
        assert st["coarsen"] == coarsen
        compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32, qmax(w))


TILE_SHAPES = [(1, 1), (2, 1), (4, 1), (8, 1), (2, 2), (4, 2), (8, 2), (4, 4)]


@pytest.mark.parametrize("shape", TILE_SHAPES, ids=lambda s: f"{s[0]}x{s[1]}")
@pytest.mark.parametrize("cfg", [1, 2, 3, 5])
def test_tile_shapes(oracle, cfg, shape):
    """Every built tile shape of the tile kernel, with and without the count output; the
    miniature targets are not multiples of the tile, so ragged right / bottom tiles run too."""
    from paper_2012_13173_b200 import binding
    w, ref = mini(oracle, cfg)
    opts = {binding.OPT_KERNEL: binding.KERNEL_TILE, binding.OPT_COARSEN: shape[0], binding.OPT_COARSEN_Y: shape[1]}
    cube, wmap, cnt, st = run_gpu(w, "f32", opts)
    assert (st["kernel"], st["coarsen"], st["coarsen_y"]) == (6, shape[0], shape[1])
    compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32, qmax(w))
    cube2, wmap2, cnt2, _ = run_gpu(w, "f32", opts, want_counts=False)
    assert cnt2 is None
    compare(cube2, wmap2, None, ref, w.sigma_deg, w.radius_deg, TOL_F32, qmax(w))


@pytest.mark.parametrize("nchan", [4, 12, 64, 256, 300])
def test_cube_kernel_channel_counts(oracle, nchan):
    """conv_mc_f32 (stats kernel 7): partial lanes, exactly one and more than one 256-channel
    block, weights, ragged 8 x 8 CTA tiles (the target is 23 x 19), with and without counts;
    the general kernel on the same input as a second opinion."""
    from paper_2012_13173_b200 import binding
    rng = np.random.default_rng([5, nchan])
    n = 5000
    w = workloads.make(1, 1.0)
    w.lon = 30.0 + rng.uniform(-0.3, 0.3, n)
    w.lat = 20.0 + rng.uniform(-0.3, 0.3, n)
    w.values = rng.normal(size=(n, nchan)).astype(np.float32)
    w.weights = rng.uniform(0.5, 1.5, n).astype(np.float32)
    w.target = workloads.CarTarget(23, 19, 29.8, 19.85, 1.0 / 60.0, 1.0 / 60.0)
    ref = run_oracle(oracle, w)
    cube, wmap, cnt, st = run_gpu(w, "f32", {binding.OPT_KERNEL: 6})
    assert st["kernel"] == 7
    compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32, qmax(w))
    cube, wmap, cnt, st = run_gpu(w, "f32", {binding.OPT_KERNEL: 6}, want_counts=False)
    compare(cube, wmap, None, ref, w.sigma_deg, w.radius_deg, TOL_F32, qmax(w))
    cube, wmap, cnt, st = run_gpu(w, "f32", {binding.OPT_KERNEL: binding.KERNEL_GENERAL})
    assert st["kernel"] == 3
    compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32, qmax(w))


def test_cube_kernel_falls_back_for_odd_channel_counts(oracle):
    w, ref = mini(oracle, 4)
    w2 = workloads.make(4, MINI[4])
    w2.values = np.ascontiguousarray(w2.values[:, :7])
    ref2 = run_oracle(oracle, w2)
    cube, wmap, cnt, st = run_gpu(w2, "f32")
    assert st["kernel"] == 3
    compare(cube, wmap, cnt, ref2, w2.sigma_deg, w2.radius_deg, TOL_F32)
    _, _, _, st = run_gpu(w, "f32")
    assert st["kernel"] == 8                     # 256 channels: the tensor-core cube kernel


def test_wide_kernels_take_the_fp64_pair_arithmetic(oracle):
    """R > 0.004 rad: fp32 arithmetic can no longer settle d <= R to the 1e-9 rad of the count bar (d to 1.2e-7
    relative), so the fp32 mode keeps its fp32 sums but tests and weighs the pairs in fp64; forcing an fp32-pair
    kernel there is refused."""
    from paper_2012_13173_b200 import binding
    rng = np.random.default_rng(771)
    n = 6000
    w = workloads.make(1, 1.0)
    w.lon = 200.0 + rng.uniform(-2.0, 2.0, n)
    w.lat = 40.0 + rng.uniform(-2.0, 2.0, n)
    w.sigma_deg, w.radius_deg, w.nside = 0.5, 1.5, 256
    w.target = workloads.CarTarget(23, 19, 199.0, 39.1, 0.09, 0.1)
    for nchan in (1, 8):
        w.values = rng.normal(size=(n, nchan)).astype(np.float32)
        ref = run_oracle(oracle, w)
        cube, wmap, cnt, st = run_gpu(w, "f32")
        assert st["kernel"] == 4
        compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32)
    for forced in (binding.KERNEL_TILE, binding.KERNEL_CUBE, binding.KERNEL_CUBE_TC):
        with pytest.raises(binding.HCGridError):
            run_gpu(w, "f32", {binding.OPT_KERNEL: forced})
    # just below the limit (0.229 deg) the tile kernel still runs
    w.sigma_deg, w.radius_deg = 0.06, 0.229
    w.values = rng.normal(size=(n, 1)).astype(np.float32)
    ref = run_oracle(oracle, w)
    cube, wmap, cnt, st = run_gpu(w, "f32")
    assert st["kernel"] == 6
    compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32)


@pytest.mark.parametrize("radius_deg,sigma_deg", [(0.1, 0.04), (0.2, 0.08), (0.225, 0.05)])
def test_tile_series_modes(oracle, radius_deg, sigma_deg):
    """Wider kernels switch the tile kernel's pair arithmetic to the series / full modes."""
    rng = np.random.default_rng(77)
    n = 6000
    w = workloads.make(1, 1.0)
    w.lon = 200.0 + rng.uniform(-2.0, 2.0, n)
    w.lat = 40.0 + rng.uniform(-2.0, 2.0, n)
    w.values = rng.normal(size=(n, 1)).astype(np.float32)
    w.sigma_deg, w.radius_deg, w.nside = sigma_deg, radius_deg, 256
    w.target = workloads.CarTarget(23, 19, 199.0, 39.1, 0.09, 0.1)
    ref = run_oracle(oracle, w)
    cube, wmap, cnt, st = run_gpu(w, "f32")
    assert st["kernel"] == 6
    compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32)
    # the cube kernel shares the pair arithmetic: same modes with 8 channels
    w.values = np.ascontiguousarray(np.repeat(w.values, 8, axis=1) * np.arange(1, 9, dtype=np.float32))
    ref8 = run_oracle(oracle, w)
    cube, wmap, cnt, st = run_gpu(w, "f32")
    assert st["kernel"] == 7
    compare(cube, wmap, cnt, ref8, w.sigma_deg, w.radius_deg, TOL_F32)


@pytest.mark.parametrize("subpix", [0, 1, 3])
def test_lookup_bin_refinement(oracle, subpix):
    from paper_2012_13173_b200 import binding
    w, ref = mini(oracle, 3)
    cube, wmap, cnt, st = run_gpu(w, "f32", {binding.OPT_SUBPIX_BITS: subpix})
    assert st["subpix_bits"] == subpix
    compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32)


# ------------------------------------------------------------ nside is only an index (c11)
@pytest.mark.parametrize("nside", [64, 256, 1024, 8192])
def test_nside_invariance(oracle, nside):
    w, ref = mini(oracle, 1)
    cube, wmap, cnt, _ = run_gpu(w, "f32", nside=nside)
    compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32)


def test_explicit_cells_equal_car(oracle):
    """A plate-carree grid handed over cell by cell is recognised and takes the plate-carree path (same kernel, same
    bits); with the recognition off, or as soon as one centre is off the grid, the per-cell path runs."""
    from paper_2012_13173_b200 import binding
    w, ref = mini(oracle, 2)
    car = run_gpu(w, "f32")
    a = run_gpu(w, "f32", explicit_cells=True)
    assert a[3]["kernel"] == car[3]["kernel"] == 6
    for x, y in zip(a[:3], car[:3]):
        assert np.array_equal(x, y, equal_nan=True)
    compare(a[0], a[1], a[2], ref, w.sigma_deg, w.radius_deg, TOL_F32)
    b = run_gpu(w, "f32", {binding.OPT_CELLS_AS_GRID: 0}, explicit_cells=True)
    assert b[3]["kernel"] in (1, 2, 3)
    compare(b[0], b[1], b[2], ref, w.sigma_deg, w.radius_deg, TOL_F32)
    # fp64 mode: recognised only because lon0 + ix * dlon reproduces every centre bit for bit -> same bits as the CAR call
    car64 = run_gpu(w, "f64")
    a64 = run_gpu(w, "f64", explicit_cells=True)
    for x, y in zip(a64[:3], car64[:3]):
        assert np.array_equal(x, y, equal_nan=True)
    compare(a64[0], a64[1], a64[2], ref, w.sigma_deg, w.radius_deg, TOL_F64)


@pytest.mark.parametrize("precision", ["f32", "f64"])
@pytest.mark.parametrize("case", ["one_cell_moved", "jitter_1e-12_deg", "rows_swapped", "single_row", "descending"])
def test_explicit_cells_near_grids(oracle, case, precision):
    """Cell lists that are almost, or in another sense, a plate-carree grid: whatever path is chosen, the result is the
    oracle's on the centres as given."""
    from paper_2012_13173_b200 import binding
    w = workloads.make(1, 1.0)
    t = w.target
    cl, cb = t.cell_centers()
    rng = np.random.default_rng(5)
    grid_like = None                                     # None: either path may run
    if case == "one_cell_moved":
        cl = cl.copy(); cl[t.nx * 7 + 3] += 3e-4
        grid_like = False
    elif case == "jitter_1e-12_deg":
        cl = cl + rng.uniform(-1e-12, 1e-12, cl.size)
        cb = cb + np.repeat(rng.uniform(-1e-12, 1e-12, t.ny), t.nx)
        grid_like = precision == "f32"                   # fp64 mode wants the centres bit for bit
    elif case == "rows_swapped":
        idx = np.arange(t.ncell).reshape(t.ny, t.nx)
        idx[[2, 9]] = idx[[9, 2]]
        cl, cb = cl[idx.ravel()], cb[idx.ravel()]
        grid_like = False
    elif case == "single_row":
        cl, cb = cl[5 * t.nx:6 * t.nx], cb[5 * t.nx:6 * t.nx]
        grid_like = True
    elif case == "descending":
        cl, cb = cl[::-1].copy(), cb[::-1].copy()        # a grid with negative steps: not bit-exact in general
    ref = oracle.grid(w.sigma_deg, w.radius_deg, cl, cb, w.lon, w.lat, w.values, w.weights)
    g = binding.HCGrid(w.sigma_deg, w.radius_deg, w.nside, precision=precision)
    g.set_target_cells(_dev(cl), _dev(cb))
    cube, wmap, cnt = g.grid(_dev(w.lon), _dev(w.lat), _dev(w.values))
    torch.cuda.synchronize()
    st = g.stats()
    g.close()
    if grid_like is not None and precision == "f32":
        assert (st["kernel"] == 6) == grid_like
    if grid_like is not None and precision == "f64" and not grid_like:
        assert st["kernel"] == 5
    compare(cube.cpu().numpy(), wmap.cpu().numpy(), cnt.cpu().numpy(), ref, w.sigma_deg, w.radius_deg,
            TOL_F32 if precision == "f32" else TOL_F64)


def test_deterministic_bitwise():
    w = workloads.make(3, MINI[3])
    a = run_gpu(w, "f32")
    b = run_gpu(w, "f32")
    assert np.array_equal(a[0], b[0], equal_nan=True) and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])


# ------------------------------------------------------------ arbitrary cells: seam, poles, odd nchan
CASES = [
    # seed, lon_c, lat_c, half_deg, sigma', nside, nchan, weights
    (1, 0.0, 0.0, 0.5, 2.0, 1024, 1, False),       # lon = 0/360 seam on the equator
    (2, 359.9, 41.8, 0.4, 1.5, 2048, 3, True),     # seam at the belt / cap transition latitude
    (3, 200.0, 89.7, 0.5, 3.0, 512, 1, True),      # north pole inside the discs (whole rings)
    (4, 10.0, -89.8, 0.4, 2.0, 256, 5, False),     # south pole
    (5, 120.0, -60.0, 0.6, 2.0, 4096, 7, False),   # south cap, nchan not a multiple of 4
    (6, 77.0, 10.0, 1.0, 4.0, 128, 300, True),     # more than one 256-channel tile
]


@pytest.mark.parametrize("case", CASES, ids=lambda c: f"seed{c[0]}")
@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_arbitrary_cells(oracle, case, precision):
    from paper_2012_13173_b200 import binding
    seed, lon_c, lat_c, half, sig_am, nside, nchan, use_w = case
    lon, lat, val, wts, clon, clat = workloads.random_case(seed, 6000, 700, lon_c, lat_c, half, nchan, use_w)
    sigma, radius = sig_am / 60.0, 3.0 * sig_am / 60.0
    ref = oracle.grid(sigma, radius, clon, clat, lon, lat, val, wts)
    assert ref.counts.sum() > 0
    g = binding.HCGrid(sigma, radius, nside, precision=precision)
    g.set_target_cells(_dev(clon), _dev(clat))
    cube, wmap, cnt = g.grid(_dev(lon), _dev(lat), _dev(val), None if wts is None else _dev(wts))
    torch.cuda.synchronize()
    tol = TOL_F32 if precision == "f32" else TOL_F64
    compare(cube.cpu().numpy(), wmap.cpu().numpy(), cnt.cpu().numpy(), ref, sigma, radius, tol,
            1.5 if use_w else 1.0)
    g.close()


def test_car_target_across_seam_and_negative_steps(oracle):
    from paper_2012_13173_b200 import binding
    lon, lat, val, _, _, _ = workloads.random_case(11, 8000, 1, 0.0, 30.0, 0.6)
    tgt = workloads.CarTarget(50, 40, 0.4, 30.35, -1.0 / 60.0, -1.0 / 60.0)   # runs westwards over lon = 0
    cl, cb = tgt.cell_centers()
    sigma, radius = 1.5 / 60.0, 4.5 / 60.0
    ref = oracle.grid(sigma, radius, cl, cb, lon, lat, val)
    for precision, tol in (("f32", TOL_F32), ("f64", TOL_F64)):
        g = binding.HCGrid(sigma, radius, 2048, precision=precision)
        g.set_target_car(tgt.nx, tgt.ny, tgt.lon0, tgt.lat0, tgt.dlon, tgt.dlat)
        cube, wmap, cnt = g.grid(_dev(lon), _dev(lat), _dev(val))
        torch.cuda.synchronize()
        compare(cube.cpu().numpy(), wmap.cpu().numpy(), cnt.cpu().numpy(), ref, sigma, radius, tol)
        g.close()


# ------------------------------------------------------------ degenerate inputs
def test_empty_input_and_unreachable_samples():
    from paper_2012_13173_b200 import binding
    g = binding.HCGrid(1.5 / 60, 4.5 / 60, 2048)
    g.set_target_car(20, 10, 30.0, 20.0, 1 / 60, 1 / 60)
    e64 = torch.empty(0, dtype=torch.float64, device="cuda")
    cube, wmap, cnt = g.grid(e64, e64, torch.empty((0, 1), dtype=torch.float32, device="cuda"))
    torch.cuda.synchronize()
    assert torch.isnan(cube).all() and (wmap == 0).all() and (cnt == 0).all()
    # samples that exist but lie far from every cell (other rings / other longitudes), NaN coordinates ignored
    lon = _dev(np.array([100.0, 31.0, 30.1, np.nan, 30.1]))
    lat = _dev(np.array([20.0, -40.0, 20.05, 20.0, 95.0]))
    val = _dev(np.array([[1.0], [2.0], [7.0], [3.0], [4.0]], dtype=np.float32))
    cube, wmap, cnt = g.grid(lon, lat, val)
    torch.cuda.synchronize()
    assert int(cnt.max()) == 1 and int((cnt > 0).sum()) > 0
    hit = cnt > 0
    assert torch.allclose(cube[hit], torch.full_like(cube[hit], 7.0), rtol=1e-6)
    assert torch.isnan(cube[~hit]).all()
    assert g.stats()["n_kept"] == 1
    g.close()


def test_single_cell_single_sample():
    from paper_2012_13173_b200 import binding
    for precision in ("f32", "f64"):
        g = binding.HCGrid(1.0 / 60, 3.0 / 60, 4096, precision=precision)
        g.set_target_car(1, 1, 10.0, -5.0, 1 / 60, 1 / 60)
        cube, wmap, cnt = g.grid(_dev(np.array([10.0])), _dev(np.array([-5.0 + 1.0 / 60])),
                                 _dev(np.array([[2.5]], dtype=np.float32)))
        torch.cuda.synchronize()
        assert int(cnt[0]) == 1
        assert float(wmap[0]) == pytest.approx(np.exp(-0.5), rel=1e-6 if precision == "f32" else 1e-13)
        assert float(cube[0, 0]) == pytest.approx(2.5, rel=1e-6)
        g.close()


def test_nside_limits(oracle):
    """nside is a power of two up to 16384 (12 nside^2 <= 2^32: the pixel index fits the sort key); the largest one
    grids like any other (results do not depend on nside: reading c11)."""
    from paper_2012_13173_b200 import binding
    w, ref = mini(oracle, 1)
    a = run_gpu(w, "f32", nside=16384)
    compare(a[0], a[1], a[2], ref, w.sigma_deg, w.radius_deg, TOL_F32)
    assert a[3]["n_kept"] > 0
    d = run_gpu(w, "f64", nside=16384)
    compare(d[0], d[1], d[2], ref, w.sigma_deg, w.radius_deg, TOL_F64)
    for bad in (32768, 3000, 0):
        with pytest.raises(binding.HCGridError):
            binding.HCGrid(w.sigma_deg, w.radius_deg, bad)
    # device and host pixelisation agree at the largest nside (indices up to 3.2e9: beyond int32)
    rng = np.random.default_rng(16384)
    lon, lat = rng.uniform(0, 360, 4000), np.rad2deg(np.arcsin(rng.uniform(-1, 1, 4000)))
    dev = binding.ang2pix_ring(16384, _dev(lon), _dev(lat)).cpu().numpy()
    host = binding.host_ang2pix_ring(16384, lon, lat)
    assert np.array_equal(dev, host) and host.max() > 2 ** 31 and host.max() < 12 * 16384 ** 2


def test_error_statuses():
    from paper_2012_13173_b200 import binding
    with pytest.raises(binding.HCGridError):
        binding.HCGrid(-1.0, 0.1, 1024)
    with pytest.raises(binding.HCGridError):
        binding.HCGrid(0.1, 0.3, 1000)            # nside not a power of two
    g = binding.HCGrid(0.1, 0.3, 1024)
    x = torch.zeros(4, dtype=torch.float64, device="cuda")
    with pytest.raises(binding.HCGridError) as ei:
        g.grid(x, x, torch.zeros((4, 1), dtype=torch.float32, device="cuda"))
    assert ei.value.status == -2                   # HCGRID_ERR_NO_TARGET
    with pytest.raises(binding.HCGridError):
        g.set_target_car(10, 10, 0.0, 85.0, 0.1, 1.0)   # rows run past the pole
    with pytest.raises(binding.HCGridError):
        g.set_option(99, 1)
    g.close()


def test_host_buffer_entry_point(oracle):
    from paper_2012_13173_b200 import binding
    w, ref = mini(oracle, 5)
    g = binding.HCGrid(w.sigma_deg, w.radius_deg, w.nside)
    t = w.target
    g.set_target_car(t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat)
    cube, wmap, cnt = g.grid_host(w.lon, w.lat, w.values, w.weights)
    compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32, qmax(w))
    # context reuse: a second, different call on the same context
    cube2, wmap2, cnt2 = g.grid_host(w.lon[::2], w.lat[::2], w.values[::2], w.weights[::2])
    ref2 = oracle.grid(w.sigma_deg, w.radius_deg, *t.cell_centers(), w.lon[::2], w.lat[::2], w.values[::2],
                       w.weights[::2])
    compare(cube2, wmap2, cnt2, ref2, w.sigma_deg, w.radius_deg, TOL_F32, qmax(w))
    g.close()


# ------------------------------------------------------------ full size, bench launch configuration
def sampled_cells(ncell, nx, k, seed):
    """Stratified sample of the flat cell index: the four corners, a border band and seeded
    interior cells."""
    rng = np.random.default_rng([13173, 77, seed])
    ny = ncell // nx
    border = np.concatenate([np.arange(0, nx, max(1, nx // 16)), (ny - 1) * nx + np.arange(0, nx, max(1, nx // 16)),
                             np.arange(0, ny, max(1, ny // 16)) * nx, np.arange(0, ny, max(1, ny // 16)) * nx + nx - 1,
                             [0, nx - 1, (ny - 1) * nx, ncell - 1]])
    inner = rng.choice(ncell, size=k, replace=False)
    return np.unique(np.concatenate([border, inner])).astype(np.int64)


def golden_reference(w, cfg):
    """The oracle's results on the declared stratified subset (borders 8 cells deep + 64 seeded 32 x 32 interior
    blocks) of a full-size config, written once by tests/make_golden.py -- which calls only oracle/ --
    and keyed by a hash of the kernel, the target and the input arrays."""
    from golden_subset import golden_path, subset_cells, workload_key
    from oracle.oracle import OracleResult
    z = np.load(golden_path(cfg))
    assert str(z["key"]) == workload_key(w), "tests/golden is stale: rerun tests/make_golden.py"
    cells = subset_cells(w.target.nx, w.target.ny, cfg)
    assert np.array_equal(cells, z["cells"])
    ref = OracleResult(z["datacube"], z["weightmap"], z["counts"].astype(np.int64), z["absmap"],
                       z["near_boundary"].astype(np.int64), 0, None, float(z["vmax"]))
    return cells, ref


@pytest.mark.parametrize("cfg,k", [(2, 600), (3, 0), (4, 150), (5, 0)])
def test_full_size_sampled_cells(oracle, cfg, k):
    """Full-size configs in the launch configuration bench.py times.  Configs 3 and 5: ~1e5 and ~8e4 cells (the
    stratified subset, oracle results from tests/golden); configs 2 and 4: sampled cells computed live."""
    w = workloads.make(cfg, 1.0)
    if cfg in (3, 5):
        cells, ref = golden_reference(w, cfg)
        assert cells.size > 60000
    else:
        cells = sampled_cells(w.target.ncell, w.target.nx, k, cfg)
        ref = run_oracle(oracle, w, cells)
    cube, wmap, cnt, st = run_gpu(w, "f32")          # default options, with the count output
    r = compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32, qmax(w), cells=cells)
    assert r["n_hit"] > 0
    assert st["kernel"] == (8 if cfg == 4 else 6)     # config 4: the tensor-core cube kernel
    # exactly what bench.py times: default options, datacube + weight map only (no count output)
    cube_b, wmap_b, none, st_b = run_gpu(w, "f32", want_counts=False)
    assert none is None and st_b["kernel"] == st["kernel"]
    compare(cube_b, wmap_b, None, ref, w.sigma_deg, w.radius_deg, TOL_F32, qmax(w), cells=cells)
    # properties that hold at any size: W > 0 <=> count > 0 <=> finite V; count bounded by n
    assert np.array_equal(wmap > 0, cnt > 0)
    assert np.array_equal(np.isfinite(cube[:, 0]), cnt > 0)
    assert cnt.min() >= 0 and cnt.max() <= w.n
    if cfg in (3, 5):
        # fp64 mode at full size, same cells
        cube, wmap, cnt, _ = run_gpu(w, "f64")
        compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F64, qmax(w), cells=cells)


@pytest.mark.parametrize("precision,tol", [("f32", TOL_F32), ("f64", TOL_F64)])
def test_support_radius_of_five_sigma(oracle, precision, tol):
    """The upper end of the paper's sphere_radius range ("3 sigma_kernel - 5 sigma_kernel"): config 1
    with R = 5 sigma exactly (weights down to exp(-12.5) = 3.7e-6 at the edge), both precisions, with and
    without per-sample weights."""
    w = workloads.make(1, 1.0)
    w.radius_deg = 5.0 * w.sigma_deg
    for wts in (None, np.random.default_rng(55).uniform(0.5, 1.5, w.n).astype(np.float32)):
        w.weights = wts
        ref = run_oracle(oracle, w)
        cube, wmap, cnt, st = run_gpu(w, precision)
        r = compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, tol, qmax(w))
        assert r["n_hit"] > 2.5 * 1.27e6                  # (5 / 3)^2 times config 1's pairs


# ------------------------------------------------------------ randomised plate-carree targets
def _random_car_case(seed):
    """A seeded random problem: patch centre anywhere (including across lon = 0 and at high
    latitude), random cell size / kernel width / nside / channel count / step signs."""
    rng = np.random.default_rng([13173, 404, seed])
    lat_c = float(rng.uniform(-84.0, 84.0))
    lon_c = float(rng.choice([0.0, 359.7, 0.2, rng.uniform(0.0, 360.0)]))
    sigma = float(rng.uniform(0.6, 3.0)) / 60.0
    radius = sigma * float(rng.uniform(2.5, 5.0))               # the paper's range of sphere_radius: 3 - 5 sigma
    cell = sigma * float(rng.uniform(0.5, 1.2))
    nx, ny = int(rng.integers(5, 42)), int(rng.integers(5, 34))
    sx, sy = (1.0 if rng.random() < 0.5 else -1.0), (1.0 if rng.random() < 0.5 else -1.0)
    dlon = sx * cell / max(np.cos(np.deg2rad(lat_c)), 0.05)      # roughly square cells on the sky
    dlat = sy * cell
    tgt = workloads.CarTarget(nx, ny, lon_c - 0.5 * (nx - 1) * dlon, lat_c - 0.5 * (ny - 1) * dlat, dlon, dlat)
    half_lat = 0.5 * ny * cell + 1.5 * radius
    half_lon = (0.5 * nx * cell + 1.5 * radius) / max(np.cos(np.deg2rad(lat_c)), 0.05)
    n = int(rng.integers(2000, 9000))
    lon = np.mod(lon_c + rng.uniform(-half_lon, half_lon, n), 360.0)
    lat = np.clip(lat_c + rng.uniform(-half_lat, half_lat, n), -89.999, 89.999)
    nchan = int(rng.choice([1, 1, 1, 8, 20]))
    val = rng.standard_normal((n, nchan)).astype(np.float32)
    wts = rng.uniform(0.5, 1.5, n).astype(np.float32) if rng.random() < 0.5 else None
    nside = int(2 ** rng.integers(7, 14))
    return tgt, lon, lat, val, wts, sigma, radius, nside


@pytest.mark.parametrize("seed", range(48))
def test_random_car_targets(oracle, seed):
    """Default kernel choice (tile kernel for one channel, cube kernel for several) on random
    plate-carree problems, fp32 and fp64 modes, against the oracle."""
    from paper_2012_13173_b200 import binding
    tgt, lon, lat, val, wts, sigma, radius, nside = _random_car_case(seed)
    cl, cb = tgt.cell_centers()
    ref = oracle.grid(sigma, radius, cl, cb, lon, lat, val, wts)
    assert ref.counts.sum() > 0
    for precision, tol in (("f32", TOL_F32), ("f64", TOL_F64)):
        g = binding.HCGrid(sigma, radius, nside, precision=precision)
        g.set_target_car(tgt.nx, tgt.ny, tgt.lon0, tgt.lat0, tgt.dlon, tgt.dlat)
        cube, wmap, cnt = g.grid(_dev(lon), _dev(lat), _dev(val), None if wts is None else _dev(wts))
        torch.cuda.synchronize()
        st = g.stats()
        if precision == "f32":
            assert st["kernel"] in (6, 7, 3), st       # tile, cube, or the general kernel (nchan % 4 != 0)
        compare(cube.cpu().numpy(), wmap.cpu().numpy(), cnt.cpu().numpy(), ref, sigma, radius, tol,
                1.5 if wts is not None else 1.0)
        g.close()


@pytest.mark.parametrize("nx,ny", [(1, 1), (2, 1), (1, 3), (3, 2), (5, 7), (9, 4), (4, 9)])
def test_tiny_targets_every_tile_shape(oracle, nx, ny):
    """Targets of a handful of cells: the region is barely wider than one support disc, tiles are
    mostly ragged, and the farthest cell of a task is far from its cell 0 (the case that wrapped
    the fixed-point differences before the span fix)."""
    from paper_2012_13173_b200 import binding
    rng = np.random.default_rng([13173, 505, nx, ny])
    sigma, radius = 2.0 / 60.0, 6.5 / 60.0
    n = 3000
    lon = np.mod(359.9 + rng.uniform(-0.5, 0.5, n), 360.0)
    lat = -47.0 + rng.uniform(-0.4, 0.4, n)
    tgt = workloads.CarTarget(nx, ny, 359.9 + 0.03 * (nx - 1), -47.0 + 0.02 * (ny - 1), -0.06, -0.04)
    cl, cb = tgt.cell_centers()
    for nchan in (1, 4):
        val = rng.standard_normal((n, nchan)).astype(np.float32)
        ref = oracle.grid(sigma, radius, cl, cb, lon, lat, val, None)
        assert ref.counts.min() > 0
        shapes = TILE_SHAPES if nchan == 1 else [(0, 0)]
        for shape in shapes:
            g = binding.HCGrid(sigma, radius, 1024)
            g.set_option(binding.OPT_COARSEN, shape[0])
            g.set_option(binding.OPT_COARSEN_Y, shape[1])
            g.set_target_car(tgt.nx, tgt.ny, tgt.lon0, tgt.lat0, tgt.dlon, tgt.dlat)
            cube, wmap, cnt = g.grid(_dev(lon), _dev(lat), _dev(val))
            torch.cuda.synchronize()
            # a single-column target is a set of one-cell strips: it takes the staged / general kernels
            assert g.stats()["kernel"] == ((6 if nchan == 1 else 7) if nx > 1 else (2 if nchan == 1 else 3))
            compare(cube.cpu().numpy(), wmap.cpu().numpy(), cnt.cpu().numpy(), ref, sigma, radius, TOL_F32)
            g.close()


@pytest.mark.parametrize("seed", range(24))
def test_random_polar_and_wide_kernels(oracle, seed):
    """Random plate-carree targets near the poles (whole-ring windows, full-circle regions) and
    with wide kernels (series / full modes of the fp32 arithmetic, or the fp64 pair arithmetic when
    the small-angle series is not valid), default kernel choice, fp32 mode."""
    from paper_2012_13173_b200 import binding
    rng = np.random.default_rng([13173, 606, seed])
    polar = seed % 2 == 0
    sign = 1.0 if rng.random() < 0.5 else -1.0
    if polar:
        lat_c = sign * float(rng.uniform(86.0, 89.3))
        sigma = float(rng.uniform(2.0, 8.0)) / 60.0
    else:
        lat_c = float(rng.uniform(-70.0, 70.0))
        sigma = float(rng.uniform(5.0, 40.0)) / 60.0          # up to 0.67 deg
    radius = sigma * float(rng.uniform(2.5, 5.0))               # 3 - 5 sigma and a little below
    cell = sigma * float(rng.uniform(0.6, 1.2))
    nx, ny = int(rng.integers(4, 30)), int(rng.integers(3, 12))
    ny = max(1, min(ny, int((89.95 - abs(lat_c)) / (0.5 * cell)))) if polar else ny
    lon_c = float(rng.uniform(0.0, 360.0))
    dlon = cell * float(rng.uniform(1.0, 6.0)) * (1.0 if rng.random() < 0.5 else -1.0)
    dlat = cell * (1.0 if rng.random() < 0.5 else -1.0)
    tgt = workloads.CarTarget(nx, ny, lon_c - 0.5 * (nx - 1) * dlon, lat_c - 0.5 * (ny - 1) * dlat, dlon, dlat)
    cl, cb = tgt.cell_centers()
    assert np.abs(cb).max() <= 90.0
    n = 5000
    half = 0.5 * ny * cell + 1.3 * radius
    lat = np.clip(lat_c + rng.uniform(-half, half, n), -90.0, 90.0)
    if polar:
        lon = rng.uniform(0.0, 360.0, n)
    else:
        half_lon = 0.5 * nx * abs(dlon) + 1.3 * radius / np.cos(np.deg2rad(min(abs(lat_c) + half, 85.0)))
        lon = np.mod(lon_c + rng.uniform(-half_lon, half_lon, n), 360.0)
    nchan = int(rng.choice([1, 1, 4]))
    val = rng.standard_normal((n, nchan)).astype(np.float32)
    wts = rng.uniform(0.5, 1.5, n).astype(np.float32) if rng.random() < 0.5 else None
    nside = int(2 ** rng.integers(5, 11))
    ref = oracle.grid(sigma, radius, cl, cb, lon, lat, val, wts)
    assert ref.counts.sum() > 0
    g = binding.HCGrid(sigma, radius, nside)
    g.set_target_car(tgt.nx, tgt.ny, tgt.lon0, tgt.lat0, tgt.dlon, tgt.dlat)
    cube, wmap, cnt = g.grid(_dev(lon), _dev(lat), _dev(val), None if wts is None else _dev(wts))
    torch.cuda.synchronize()
    compare(cube.cpu().numpy(), wmap.cpu().numpy(), cnt.cpu().numpy(), ref, sigma, radius, TOL_F32,
            1.5 if wts is not None else 1.0)
    g.close()


@pytest.mark.parametrize("kernel,precision", [(1, "f32"), (3, "f32"), (0, "f64")])
def test_all_sky_target_starting_at_minus_180(oracle, kernel, precision):
    """A target that spans the whole circle and starts at lon = -180: the region is a full-circle region and every
    pixel window west of lon = 0 has negative pixel indices.  Windows are reduced modulo the ring length (two sample
    ranges where one crosses the ring's first pixel) instead of widening to the whole ring, so the number of pairs
    put to the distance test stays a small multiple of the hits on both halves of the sky."""
    from paper_2012_13173_b200 import binding
    rng = np.random.default_rng([13173, 808])
    n = 600000
    lon = rng.uniform(0.0, 360.0, n)
    lat = np.rad2deg(np.arcsin(rng.uniform(np.sin(np.deg2rad(-62.0)), np.sin(np.deg2rad(62.0)), n)))
    val = rng.standard_normal((n, 1)).astype(np.float32)
    sigma, radius = 0.075, 0.225                    # 3.9e-3 rad: the widest kernels the fp32 pair arithmetic takes
    tgt = workloads.CarTarget(360, 61, -180.0, -60.0, 1.0, 2.0)
    cl, cb = tgt.cell_centers()
    ref = oracle.grid(sigma, radius, cl, cb, lon, lat, val, None)
    pairs = {}
    for lon0 in (-180.0, 0.0, 97.0):                # the same 360 cells per row, listed from three starting points
        g = binding.HCGrid(sigma, radius, 1024, precision=precision)
        g.set_option(binding.OPT_PROFILE, 1)
        if kernel:
            g.set_option(binding.OPT_KERNEL, kernel)
        g.set_target_car(tgt.nx, tgt.ny, lon0, tgt.lat0, tgt.dlon, tgt.dlat)
        cube, wmap, cnt = g.grid(_dev(lon), _dev(lat), _dev(val))
        torch.cuda.synchronize()
        st = g.stats()
        g.close()
        assert st["kernel"] == (kernel if kernel else 5)
        assert st["n_hit"] == int(cnt.sum().item()) == int(ref.counts.sum())
        assert st["n_pairs_tested"] >= st["n_hit"]
        pairs[lon0] = st["n_pairs_tested"]
        assert pairs[lon0] < 8 * st["n_hit"], (lon0, st)     # a whole-ring scan would test ~100 x the hits
        if lon0 == -180.0:
            compare(cube.cpu().numpy(), wmap.cpu().numpy(), cnt.cpu().numpy(), ref, sigma, radius,
                    TOL_F32 if precision == "f32" else TOL_F64)
    assert max(pairs.values()) < 1.05 * min(pairs.values()), pairs


def test_large_sparse_target(oracle):
    """A 2048 x 2048 target (4.2 M cells) of which only a corner holds samples: every tile far from
    the data is empty (NaN / 0 / 0), the cells near the data match the oracle."""
    from paper_2012_13173_b200 import binding
    rng = np.random.default_rng([13173, 707])
    n = 40000
    tgt = workloads.CarTarget(2048, 2048, 100.0, -8.0, 0.5 / 60.0, 0.5 / 60.0)
    lon = 100.0 + rng.uniform(0.0, 0.4, n)
    lat = -8.0 + rng.uniform(0.0, 0.3, n)
    val = rng.standard_normal((n, 1)).astype(np.float32)
    sigma, radius = 0.5 / 60.0, 1.5 / 60.0
    g = binding.HCGrid(sigma, radius, 4096)
    g.set_target_car(tgt.nx, tgt.ny, tgt.lon0, tgt.lat0, tgt.dlon, tgt.dlat)
    cube, wmap, cnt = g.grid(_dev(lon), _dev(lat), _dev(val))
    torch.cuda.synchronize()
    assert g.stats()["kernel"] == 6
    cube, wmap, cnt = cube.cpu().numpy(), wmap.cpu().numpy(), cnt.cpu().numpy()
    g.close()
    iy, ix = np.divmod(np.arange(tgt.ncell), tgt.nx)
    far = (ix > 60) | (iy > 48)                      # beyond the data + support radius
    assert (cnt[far] == 0).all() and (wmap[far] == 0).all() and np.isnan(cube[far, 0]).all()
    assert int(cnt.sum()) > 0
    cells = np.flatnonzero(~far)[::7]
    cl, cb = tgt.cell_centers()
    ref = oracle.grid(sigma, radius, cl[cells], cb[cells], lon, lat, val, None)
    compare(cube, wmap, cnt, ref, sigma, radius, TOL_F32, cells=cells)


@pytest.mark.parametrize("split", [1, 2, 4])
@pytest.mark.parametrize("shape", [(1, 1), (4, 2), (8, 2)], ids=lambda s: f"{s[0]}x{s[1]}")
def test_split_tiles(oracle, shape, split):
    """Tile kernel with every tile's candidate stream shared by `split` warps of one CTA (few
    cells, many samples per cell: the paper's 90 x 90-cell experiments), forced and automatic."""
    from paper_2012_13173_b200 import binding
    rng = np.random.default_rng([13173, 808])
    n = 60000
    sigma, radius = 127.4 / 3600.0, 382.2 / 3600.0
    lon = 30.0 + rng.uniform(-0.6, 0.6, n)
    lat = 25.0 + rng.uniform(-0.6, 0.6, n)
    val = rng.standard_normal((n, 1)).astype(np.float32)
    wts = rng.uniform(0.5, 1.5, n).astype(np.float32)
    tgt = workloads.CarTarget(13, 11, 29.7, 24.75, 200.0 / 3600.0, 200.0 / 3600.0)
    cl, cb = tgt.cell_centers()
    ref = oracle.grid(sigma, radius, cl, cb, lon, lat, val, wts)
    opts = {binding.OPT_KERNEL: binding.KERNEL_TILE, binding.OPT_COARSEN: shape[0], binding.OPT_COARSEN_Y: shape[1],
            binding.OPT_SPLIT: split}
    for counts in (True, False):
        cube, wmap, cnt, st = run_gpu(wl_like(tgt, lon, lat, val, wts, sigma, radius), "f32", opts, want_counts=counts)
        assert st["split"] == split
        compare(cube, wmap, cnt, ref, sigma, radius, TOL_F32, 1.5)
    if shape == (4, 2) and split == 1:
        _, _, _, st = run_gpu(wl_like(tgt, lon, lat, val, wts, sigma, radius), "f32")
        assert st["split"] > 1          # 143 cells x ~5,000 contributors each: the automatic choice splits


def wl_like(tgt, lon, lat, val, wts, sigma, radius, nside=2048):
    w = workloads.make(1, 1.0)
    w.lon, w.lat, w.values, w.weights, w.target = lon, lat, val, wts, tgt
    w.sigma_deg, w.radius_deg, w.nside = sigma, radius, nside
    return w


# ------------------------------------------------------------ incremental gridding
@pytest.mark.parametrize("cfg,precision", [(1, "f32"), (3, "f32"), (5, "f32"), (4, "f32"), (2, "f64")])
def test_accumulate_batches_equal_the_union(oracle, cfg, precision):
    """hcgrid_accumulate over uneven batches (one of them empty) + hcgrid_finalize against the
    oracle on ALL samples; a second accumulation on the same context starts from zero."""
    from paper_2012_13173_b200 import binding
    w, ref = mini(oracle, cfg)
    t = w.target
    tol = TOL_F32 if precision == "f32" else TOL_F64
    g = binding.HCGrid(w.sigma_deg, w.radius_deg, w.nside, precision=precision)
    g.set_target_car(t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat)
    lon, lat, val = _dev(w.lon), _dev(w.lat), _dev(w.values)
    wts = None if w.weights is None else _dev(w.weights)
    cuts = [0, w.n // 5, w.n // 5, w.n // 2 + 7, w.n]
    for rep in range(2):
        for a, b in zip(cuts[:-1], cuts[1:]):
            g.accumulate(lon[a:b].contiguous(), lat[a:b].contiguous(), val[a:b].contiguous(),
                         None if wts is None else wts[a:b].contiguous())
        assert g.accumulated_batches == 4
        cube, wmap, cnt = g.finalize(reset=True)
        torch.cuda.synchronize()
        assert g.accumulated_batches == 0
        compare(cube.cpu().numpy(), wmap.cpu().numpy(), cnt.cpu().numpy(), ref, w.sigma_deg, w.radius_deg, tol, qmax(w))
    with pytest.raises(binding.HCGridError):
        g.finalize()
    # an EMPTY first batch (it becomes the accumulators), then everything
    g.accumulate(lon[:0].contiguous(), lat[:0].contiguous(), val[:0].contiguous(), None if wts is None else wts[:0].contiguous())
    g.accumulate(lon, lat, val, wts)
    cube, wmap, cnt = g.finalize()
    torch.cuda.synchronize()
    compare(cube.cpu().numpy(), wmap.cpu().numpy(), cnt.cpu().numpy(), ref, w.sigma_deg, w.radius_deg, tol, qmax(w))
    g.close()


def test_context_reuse_streams_and_retargeting(oracle):
    """One context through: a call on a non-default stream, a larger call (scratch grows), a new
    target, and a smaller call again -- each checked against the oracle."""
    from paper_2012_13173_b200 import binding
    w1, ref1 = mini(oracle, 1)
    w3, ref3 = mini(oracle, 3)
    g = binding.HCGrid(w1.sigma_deg, w1.radius_deg, w1.nside)
    t = w1.target
    g.set_target_car(t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat)
    side = torch.cuda.Stream()
    half = w1.n // 2
    lon, lat, val = _dev(w1.lon), _dev(w1.lat), _dev(w1.values)
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        cube_h, wmap_h, cnt_h = g.grid(lon[:half].contiguous(), lat[:half].contiguous(), val[:half].contiguous())
    side.synchronize()
    ref_h = oracle.grid(w1.sigma_deg, w1.radius_deg, *t.cell_centers(), w1.lon[:half], w1.lat[:half], w1.values[:half])
    compare(cube_h.cpu().numpy(), wmap_h.cpu().numpy(), cnt_h.cpu().numpy(), ref_h, w1.sigma_deg, w1.radius_deg, TOL_F32)
    cube, wmap, cnt = g.grid(lon, lat, val)                  # larger n: scratch grows
    torch.cuda.synchronize()
    compare(cube.cpu().numpy(), wmap.cpu().numpy(), cnt.cpu().numpy(), ref1, w1.sigma_deg, w1.radius_deg, TOL_F32)
    g.close()
    # same kernel parameters as config 3, two targets in turn on one context
    g = binding.HCGrid(w3.sigma_deg, w3.radius_deg, w3.nside)
    t3 = w3.target
    g.set_target_car(5, 4, t3.lon0, t3.lat0, t3.dlon, t3.dlat)
    small = g.grid(_dev(w3.lon), _dev(w3.lat), _dev(w3.values))
    g.set_target_car(t3.nx, t3.ny, t3.lon0, t3.lat0, t3.dlon, t3.dlat)
    cube, wmap, cnt = g.grid(_dev(w3.lon), _dev(w3.lat), _dev(w3.values))
    torch.cuda.synchronize()
    compare(cube.cpu().numpy(), wmap.cpu().numpy(), cnt.cpu().numpy(), ref3, w3.sigma_deg, w3.radius_deg, TOL_F32)
    # the 5 x 4 corner of the big target must agree with the small target's result bit for bit or to tolerance
    idx = (np.arange(4)[:, None] * t3.nx + np.arange(5)[None, :]).ravel()
    np.testing.assert_allclose(small[1].cpu().numpy(), wmap.cpu().numpy()[idx], rtol=2e-6)
    assert np.array_equal(small[2].cpu().numpy(), cnt.cpu().numpy()[idx])
    g.close()


def test_row_band_sharding_on_one_gpu(oracle):
    """The multi-GPU row-band sharding (dist.py), its ranks run one after the other on this GPU:
    the concatenated bands match the oracle on the whole target."""
    from paper_2012_13173_b200 import binding, dist as hdist
    w, ref = mini(oracle, 3)
    t = w.target
    world = 3
    cubes, wmaps, cnts = [], [], []
    for r in range(world):
        a, b = hdist.row_band(t.ny, world, r, align=4)
        bt = hdist.band_target(t, a, b)
        m = hdist.band_sample_mask(w.lat, t, a, b, w.radius_deg)
        g = binding.HCGrid(w.sigma_deg, w.radius_deg, w.nside)
        g.set_target_car(bt.nx, bt.ny, bt.lon0, bt.lat0, bt.dlon, bt.dlat)
        cube, wmap, cnt = g.grid(_dev(w.lon[m]), _dev(w.lat[m]), _dev(np.ascontiguousarray(w.values[m])))
        torch.cuda.synchronize()
        cubes.append(cube.cpu().numpy()); wmaps.append(wmap.cpu().numpy()); cnts.append(cnt.cpu().numpy())
        g.close()
    compare(np.concatenate(cubes), np.concatenate(wmaps), np.concatenate(cnts), ref, w.sigma_deg, w.radius_deg, TOL_F32)


@pytest.mark.parametrize("cfg,precision,chunks", [(1, "f32", 3), (3, "f32", 4), (4, "f32", 2), (5, "f32", 5), (2, "f64", 3)])
def test_host_entry_point_in_chunks(oracle, cfg, precision, chunks):
    """hcgrid_grid_host with the copy / compute pipeline forced on (HCGRID_OPT_HOST_CHUNKS): pieces gridded as
    they arrive, one normalisation at the end; pinned and pageable buffers; then the plain path again."""
    from paper_2012_13173_b200 import binding
    w, ref = mini(oracle, cfg)
    g = binding.HCGrid(w.sigma_deg, w.radius_deg, w.nside, precision=precision)
    t = w.target
    g.set_target_car(t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat)
    g.set_option(binding.OPT_HOST_CHUNKS, chunks)
    tol = TOL_F64 if precision == "f64" else TOL_F32
    pin = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
    for conv in (pin, lambda a: a):
        cube, wmap, cnt = g.grid_host(conv(w.lon), conv(w.lat), conv(w.values), conv(w.weights))
        compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, tol, qmax(w))
        assert g.accumulated_batches == 0
    again = g.grid_host(w.lon, w.lat, w.values, w.weights)
    assert np.array_equal(again[0], cube, equal_nan=True) and np.array_equal(again[1], wmap)   # deterministic
    g.set_option(binding.OPT_HOST_CHUNKS, 1)
    cube1, wmap1, cnt1 = g.grid_host(w.lon, w.lat, w.values, w.weights)
    compare(cube1, wmap1, cnt1, ref, w.sigma_deg, w.radius_deg, tol, qmax(w))
    assert np.array_equal(cnt1, cnt)
    with pytest.raises(binding.HCGridError):
        g.set_option(binding.OPT_HOST_CHUNKS, 17)
    g.close()
