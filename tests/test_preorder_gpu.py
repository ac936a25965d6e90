"""Device pre-ordering (a2..a4) inspected on its own: PAPER.md:120-124 (Sect. 3.3 I-III) and
the worked example of Fig. 3."""
import numpy as np
import pytest

from paper_2012_13173_b200 import workloads

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _dev(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


def test_device_pixelisation_equals_host_build():
    from paper_2012_13173_b200 import binding
    rng = np.random.default_rng(5)
    lon = rng.uniform(-10, 370, 200000)
    lat = np.degrees(np.arcsin(rng.uniform(-1, 1, 200000)))
    for nside in (1, 4, 2048, 8192):
        dev = binding.ang2pix_ring(nside, _dev(lon), _dev(lat)).cpu().numpy()
        host = binding.host_ang2pix_ring(nside, lon, lat)
        # same source compiled twice; device libm may differ by an ulp at pixel edges
        assert np.mean(dev != host) < 1e-5
        assert dev.min() >= 0 and dev.max() < 12 * nside * nside


def test_sorted_order_and_tables():
    from paper_2012_13173_b200 import binding
    w = workloads.make(3, 0.004)
    g = binding.HCGrid(w.sigma_deg, w.radius_deg, w.nside)
    t = w.target
    g.set_target_car(t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat)
    g.grid(_dev(w.lon), _dev(w.lat), _dev(w.values))
    pix, idx, ring_first, ring_start = g.debug_preorder()
    st = g.stats()
    nk = st["n_kept"]
    assert 0 < nk <= w.n and pix.size == nk
    # the "value" of the key-value sort is a permutation of distinct input indices
    assert np.unique(idx).size == nk and idx.min() >= 0 and idx.max() < w.n
    # S' carries the pixel of the sample it names
    assert np.array_equal(pix, binding.host_ang2pix_ring(w.nside, w.lon[idx], w.lat[idx])) or \
        np.mean(pix != binding.host_ang2pix_ring(w.nside, w.lon[idx], w.lat[idx])) < 1e-5
    # sorted by ring: ring index non-decreasing along S' ("contiguous"); within a ring the
    # order is by longitude measured from the region's western edge, i.e. pixel non-decreasing
    # except for at most one wrap per ring
    first = np.array([binding.host_ring_info(w.nside, r)[0] for r in range(ring_first, ring_first + st["n_rings"] + 1)])
    ring_of = np.searchsorted(first, pix, side="right") - 1
    assert np.all(np.diff(ring_of) >= 0)
    # R_start: CSR over rings
    assert ring_start[0] == 0 and ring_start[-1] == nk and np.all(np.diff(ring_start) >= 0)
    for r in range(st["n_rings"]):
        seg = ring_of[ring_start[r]:ring_start[r + 1]]
        assert seg.size == 0 or (seg.min() == r and seg.max() == r)
        p = pix[ring_start[r]:ring_start[r + 1]]
        assert np.sum(np.diff(p) < 0) <= 1
    # stable sort: equal pixels keep input order when they fall into the same lookup bin
    g.close()


def test_fig3_ring_table_semantics():
    """Fig. 3: 17 samples in 4 rings holding 6, 3, 7, 1 -> R_start = 1, 7, 10, 17 (1-based),
    ring i = [R_start[i], R_start[i+1] - 1]."""
    from paper_2012_13173_b200 import binding
    nside = 16
    r0 = 20
    hist = [6, 3, 7, 1]
    lon, lat = [], []
    for k, m in enumerate(hist):
        la = binding.host_ring_info(nside, r0 + k)[2]
        for j in range(m):
            lon.append(40.0 + 1.3 * j)
            lat.append(la)
    lon, lat = np.array(lon), np.array(lat)
    perm = np.random.default_rng(1).permutation(17)
    g = binding.HCGrid(1.0, 3.0, nside)
    g.set_target_car(12, 12, 38.0, lat.min() - 1.0, 1.0, (lat.max() - lat.min() + 2.0) / 11)
    g.grid(_dev(lon[perm]), _dev(lat[perm]), _dev(np.ones((17, 1), np.float32)))
    pix, idx, ring_first, ring_start = g.debug_preorder()
    assert pix.size == 17
    k0 = r0 - ring_first
    assert list(ring_start[k0:k0 + 5] - ring_start[k0] + 1) == [1, 7, 10, 17, 18]
    assert np.all(ring_start[:k0 + 1] == 0) and np.all(ring_start[k0 + 4:] == 17)
    g.close()


def test_measured_peaks_are_plausible():
    from paper_2012_13173_b200 import binding
    fp32, mufu = binding.measure_peaks(0)
    assert 5e12 < fp32 < 6e13 and 5e11 < mufu < 8e12


def _run_preorder_mode(w, mode, precision="f32", lon=None, lat=None, values=None, weights=None):
    from paper_2012_13173_b200 import binding
    g = binding.HCGrid(w.sigma_deg, w.radius_deg, w.nside, precision=precision)
    t = w.target
    g.set_target_car(t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat)
    g.set_option(binding.OPT_PREORDER, mode)
    lon = w.lon if lon is None else lon
    lat = w.lat if lat is None else lat
    values = w.values if values is None else values
    cube, wmap, cnt = g.grid(_dev(lon), _dev(lat), _dev(values), None if weights is None else _dev(weights))
    torch.cuda.synchronize()
    pre = g.debug_preorder()
    st = g.stats()
    g.close()
    return cube.cpu().numpy(), wmap.cpu().numpy(), cnt.cpu().numpy(), pre, st


@pytest.mark.parametrize("case", ["c1", "c3", "c4", "c3_f64", "pileup", "pileup_f64", "weights"])
def test_counting_preorder_gives_the_radix_sort_order(case):
    """The counting pre-order (atomics + scan + per-bin index sort) must reproduce the stable
    key-value sort of PAPER.md:120 exactly: same S' (sorted indices), same tables, and hence
    bit-identical maps."""
    from paper_2012_13173_b200 import binding
    precision = "f64" if case.endswith("f64") else "f32"
    kw = {}
    if case == "c1":
        w = workloads.make(1, 1.0)
    elif case == "c4":
        w = workloads.make(4, 0.01)
    else:
        w = workloads.make(3, 0.004)
    if case.startswith("pileup"):
        # a third of the samples stare at three points: bins of thousands of samples next to
        # sparse ones (the block-sorted path), plus exact duplicates
        rng = np.random.default_rng(77)
        lon, lat = w.lon.copy(), w.lat.copy()
        t = w.target
        n = lon.size
        for k, frac in enumerate((0.2, 0.1, 0.03)):
            sel = rng.choice(n, int(frac * n), replace=False)
            lon[sel] = t.lon0 + (0.3 + 0.2 * k) * t.nx * t.dlon + rng.normal(0, 1e-7, sel.size) * (k != 2)
            lat[sel] = t.lat0 + (0.4 + 0.1 * k) * t.ny * t.dlat + rng.normal(0, 1e-7, sel.size) * (k != 2)
        kw = {"lon": lon, "lat": lat}
    if case == "weights":
        kw = {"weights": np.random.default_rng(3).uniform(0.5, 2.0, w.n).astype(np.float32)}
    a = _run_preorder_mode(w, binding.PREORDER_RADIX, precision, **kw)
    b = _run_preorder_mode(w, binding.PREORDER_COUNTING, precision, **kw)
    assert a[4]["preorder"] == 1 and b[4]["preorder"] == 2
    assert a[4]["n_kept"] == b[4]["n_kept"] > 0
    assert np.array_equal(a[3][1], b[3][1])                   # sorted indices: the same S'
    assert np.array_equal(a[3][0], b[3][0]) and np.array_equal(a[3][3], b[3][3])
    assert np.array_equal(a[2], b[2])
    assert np.array_equal(a[1], b[1])
    assert np.array_equal(a[0], b[0], equal_nan=True)


def test_preorder_auto_choice():
    """Auto: counting unless samples outnumber bins many times over (or bins the samples)."""
    from paper_2012_13173_b200 import binding
    w = workloads.make(3, 0.004)
    st = _run_preorder_mode(w, binding.PREORDER_AUTO)[4]
    assert st["preorder"] == 2
    # the same field with 40 x the samples piled on: far more samples than bins
    rng = np.random.default_rng(1)
    lon = np.tile(w.lon, 40) + rng.normal(0, 1e-4, w.n * 40)
    lat = np.tile(w.lat, 40)
    val = np.tile(w.values, (40, 1))
    st2 = _run_preorder_mode(w, binding.PREORDER_AUTO, lon=lon, lat=lat, values=val)[4]
    assert st2["preorder"] == (2 if lon.size <= 10 * st2["n_bins"] else 1)


def test_dense_input_refines_the_lookup_bins(oracle):
    """More than 10 samples per lookup bin on a plate-carree target with automatic sub-pixel bits: the first call
    rebuilds the tables with finer bins, the counting pre-order applies, results match the oracle; a later sparse call
    keeps the finer tables; an explicit HCGRID_OPT_SUBPIX_BITS or a new target switches it off / starts over."""
    from paper_2012_13173_b200 import binding
    from parity import TOL_F32, compare
    rng = np.random.default_rng([13173, 4242])
    n = 1_500_000
    sigma, radius, nside = 127.4 / 3600.0, 382.2 / 3600.0, 2048
    tgt = workloads.CarTarget(90, 90, 27.5, 22.5, 200.0 / 3600.0, 200.0 / 3600.0)
    lon = 30.0 + rng.uniform(-2.5, 2.5, n)
    lat = 25.0 + rng.uniform(-2.5, 2.5, n)
    val = rng.standard_normal((n, 1)).astype(np.float32)
    cl, cb = tgt.cell_centers()
    cells = np.arange(0, tgt.ncell, 23)
    ref = oracle.grid(sigma, radius, cl[cells], cb[cells], lon, lat, val, None)
    d_lon, d_lat, d_val = _dev(lon), _dev(lat), _dev(val)
    g = binding.HCGrid(sigma, radius, nside)
    g.set_target_car(tgt.nx, tgt.ny, tgt.lon0, tgt.lat0, tgt.dlon, tgt.dlat)
    g.grid(d_lon[:1000], d_lat[:1000], d_val[:1000])
    s0 = g.stats()
    assert s0["subpix_bits"] == 2 and n > 10 * s0["n_bins"]
    for _ in range(2):                                   # the refining call and a plain one after it
        cube, wmap, cnt = g.grid(d_lon, d_lat, d_val)
        torch.cuda.synchronize()
        s1 = g.stats()
        assert s1["subpix_bits"] > 2 and s1["preorder"] == 2 and n <= 4 * s1["n_bins"] and s1["kernel"] == 6
        compare(cube.cpu().numpy(), wmap.cpu().numpy(), cnt.cpu().numpy(), ref, sigma, radius, TOL_F32, cells=cells)
    g.grid(d_lon[:1000], d_lat[:1000], d_val[:1000])     # sparse again: the tables stay
    assert g.stats()["subpix_bits"] == s1["subpix_bits"]
    g.set_target_car(tgt.nx, tgt.ny, tgt.lon0, tgt.lat0, tgt.dlon, tgt.dlat)
    g.grid(d_lon[:1000], d_lat[:1000], d_val[:1000])
    assert g.stats()["subpix_bits"] == 2                 # a new target starts over
    g.close()
    # two dense batches through hcgrid_accumulate on a fresh context: the first one refines, the sums do not care
    g = binding.HCGrid(sigma, radius, nside)
    g.set_target_car(tgt.nx, tgt.ny, tgt.lon0, tgt.lat0, tgt.dlon, tgt.dlat)
    h = n - n // 8                                        # 1.3 M samples: still more than 10 per quarter-pixel bin
    g.accumulate(d_lon[:h], d_lat[:h], d_val[:h])
    b1 = g.stats()["subpix_bits"]
    g.accumulate(d_lon[h:], d_lat[h:], d_val[h:])
    cube, wmap, cnt = g.finalize()
    torch.cuda.synchronize()
    assert b1 > 2 and g.stats()["subpix_bits"] == b1
    compare(cube.cpu().numpy(), wmap.cpu().numpy(), cnt.cpu().numpy(), ref, sigma, radius, TOL_F32, cells=cells)
    g.close()
    g = binding.HCGrid(sigma, radius, nside)
    g.set_option(binding.OPT_SUBPIX_BITS, 2)              # the caller's choice stands
    g.set_target_car(tgt.nx, tgt.ny, tgt.lon0, tgt.lat0, tgt.dlon, tgt.dlat)
    cube, wmap, cnt = g.grid(d_lon, d_lat, d_val)
    torch.cuda.synchronize()
    s2 = g.stats()
    assert s2["subpix_bits"] == 2 and s2["preorder"] == 1
    compare(cube.cpu().numpy(), wmap.cpu().numpy(), cnt.cpu().numpy(), ref, sigma, radius, TOL_F32, cells=cells)
    g.close()


def test_piled_up_input_switches_later_calls_to_the_radix_sort(oracle):
    """A tenth of 1.2 M samples within 1e-7 deg of one spot: the counting pre-order orders that bin one block at a
    time (slow but right); the call reports it to the host behind itself and the following calls on the target take the
    radix sort -- same S', same bits.  A few bins of a few thousand samples do not trigger it, a new target resets it."""
    from paper_2012_13173_b200 import binding
    from parity import TOL_F32, compare
    w = workloads.make(3, 0.12)
    t = w.target
    rng = np.random.default_rng(99)
    lon, lat = w.lon.copy(), w.lat.copy()
    sel = rng.choice(w.n, w.n // 10, replace=False)
    lon[sel] = t.lon0 + 0.37 * t.nx * t.dlon + rng.normal(0, 1e-7, sel.size)
    lat[sel] = t.lat0 + 0.61 * t.ny * t.dlat + rng.normal(0, 1e-7, sel.size)
    assert w.n >= 1 << 20
    d = (_dev(lon), _dev(lat), _dev(w.values))
    g = binding.HCGrid(w.sigma_deg, w.radius_deg, w.nside)
    g.set_target_car(t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat)
    res, pre = [], []
    for _ in range(3):
        r = g.grid(*d)
        torch.cuda.synchronize()
        res.append([x.clone() for x in r]); pre.append(g.stats()["preorder"])
    assert pre == [2, 1, 1]
    for a, b in zip(res[0], res[2]):
        assert torch.equal(a.nan_to_num(nan=-1.0), b.nan_to_num(nan=-1.0))
    cl, cb = t.cell_centers()
    cells = np.arange(0, t.ncell, 97)
    ref = oracle.grid(w.sigma_deg, w.radius_deg, cl[cells], cb[cells], lon, lat, w.values, None)
    compare(res[2][0].cpu().numpy(), res[2][1].cpu().numpy(), res[2][2].cpu().numpy(), ref, w.sigma_deg, w.radius_deg,
            TOL_F32, cells=cells)
    g.set_target_car(t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat)          # a new target: the counting sort again
    g.grid(*d)
    assert g.stats()["preorder"] == 2
    g.close()
    # three bins of ~3000 samples: left to the block-sort kernel, no switch
    lon2, lat2 = w.lon.copy(), w.lat.copy()
    for k in range(3):
        s2 = rng.choice(w.n, 3000, replace=False)
        lon2[s2] = t.lon0 + (0.2 + 0.2 * k) * t.nx * t.dlon + rng.normal(0, 1e-7, s2.size)
        lat2[s2] = t.lat0 + 0.5 * t.ny * t.dlat + rng.normal(0, 1e-7, s2.size)
    d2 = (_dev(lon2), _dev(lat2), _dev(w.values))
    g = binding.HCGrid(w.sigma_deg, w.radius_deg, w.nside)
    g.set_target_car(t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat)
    for _ in range(3):
        g.grid(*d2)
        torch.cuda.synchronize()
        assert g.stats()["preorder"] == 2
    g.close()
