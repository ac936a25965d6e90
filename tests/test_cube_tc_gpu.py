"""GPU parity of the tensor-core cube kernel conv_mc_tc_f32 (tcgen05 / TMEM, stats kernel 8;
SURVEY.md 8f NEXT-1) against the brute-force oracle, at the ordinary fp32 bar: counts exact up to
the pairs within 1e-9 rad of the support boundary, weight map and datacube within 1e-5."""
import numpy as np
import pytest

from paper_2012_13173_b200 import workloads

from parity import TOL_F32, compare
from test_parity_gpu import MINI, mini, qmax, run_gpu, run_oracle

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _cube_case(seed, nchan, n=5000, positive=False, target=(23, 19)):
    rng = np.random.default_rng([11, seed, nchan])
    w = workloads.make(1, 1.0)
    w.lon = 30.0 + rng.uniform(-0.3, 0.3, n)
    w.lat = 20.0 + rng.uniform(-0.3, 0.3, n)
    v = rng.normal(size=(n, nchan)).astype(np.float32)
    if positive:
        v = (5.0 + np.abs(v)).astype(np.float32)
    w.values = v
    w.weights = rng.uniform(0.5, 1.5, n).astype(np.float32)
    w.target = workloads.CarTarget(target[0], target[1], 29.8, 19.85, 1.0 / 60.0, 1.0 / 60.0)
    return w


@pytest.mark.parametrize("nchan", [32, 64, 96, 256, 288, 512])
def test_tc_kernel_channel_counts(oracle, nchan):
    """Partial and several 256-channel blocks, per-sample weights, ragged 16 x 8 tiles (23 x 19
    cells), with and without the count output; forced for the channel counts the auto choice
    leaves to the CUDA-core kernel."""
    from paper_2012_13173_b200 import binding
    w = _cube_case(0, nchan)
    ref = run_oracle(oracle, w)
    cube, wmap, cnt, st = run_gpu(w, "f32", {binding.OPT_KERNEL: 7})
    assert st["kernel"] == 8
    compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32, qmax(w))
    cube, wmap, cnt, st = run_gpu(w, "f32", {binding.OPT_KERNEL: 7}, want_counts=False)
    compare(cube, wmap, None, ref, w.sigma_deg, w.radius_deg, TOL_F32, qmax(w))


def test_tc_kernel_is_the_auto_choice_from_64_channels(oracle):
    w = _cube_case(1, 64)
    _, _, _, st = run_gpu(w, "f32")
    assert st["kernel"] == 8
    w = _cube_case(1, 32)
    _, _, _, st = run_gpu(w, "f32")
    assert st["kernel"] == 7


def test_tc_kernel_same_sign_values_deep_sums(oracle):
    """All-positive spectra and ~4000 candidates per tile: the case in which the tensor core's
    round-toward-zero accumulation would drift by ~1e-4 without the chunked fp32 hand-over."""
    from paper_2012_13173_b200 import binding
    w = _cube_case(2, 64, n=60000, positive=True, target=(37, 21))
    ref = run_oracle(oracle, w)
    cube, wmap, cnt, st = run_gpu(w, "f32", {binding.OPT_KERNEL: 7})
    assert st["kernel"] == 8
    r = compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32, qmax(w))
    assert r["max_rel_v_clear"] < 5e-6, r


def test_tc_kernel_config4_miniature_and_cuda_core_kernel_agree(oracle):
    from paper_2012_13173_b200 import binding
    w, ref = mini(oracle, 4)
    cube, wmap, cnt, st = run_gpu(w, "f32", {binding.OPT_KERNEL: 7})
    assert st["kernel"] == 8
    compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32)
    cube6, wmap6, cnt6, st6 = run_gpu(w, "f32", {binding.OPT_KERNEL: 6})
    assert st6["kernel"] == 7
    assert np.array_equal(cnt, cnt6)
    np.testing.assert_allclose(wmap, wmap6, rtol=2e-6)


def test_tc_kernel_deterministic_bitwise():
    from paper_2012_13173_b200 import binding
    w = _cube_case(3, 64, n=20000)
    a = run_gpu(w, "f32", {binding.OPT_KERNEL: 7})
    b = run_gpu(w, "f32", {binding.OPT_KERNEL: 7})
    assert np.array_equal(a[0], b[0], equal_nan=True) and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])


def test_tc_kernel_non_finite_values_poison_only_the_cells_they_reach(oracle):
    """Reading c8: a NaN value poisons the cells its sample reaches and no others.  Through the
    MMA 0 * NaN would poison the whole tile, so flagged tiles are recomputed cell by cell."""
    from paper_2012_13173_b200 import binding
    w = _cube_case(4, 64, n=3000)
    w.values[17, 5] = np.nan
    w.values[1234, 40] = np.nan
    ref = run_oracle(oracle, w)
    assert np.isnan(ref.datacube[:, 5]).sum() > 0
    cube, wmap, cnt, st = run_gpu(w, "f32", {binding.OPT_KERNEL: 7})
    assert st["kernel"] == 8
    compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32, qmax(w))


def test_tc_kernel_empty_input_and_empty_tiles(oracle):
    from paper_2012_13173_b200 import binding
    w = _cube_case(5, 64, n=40, target=(64, 40))            # most tiles see no sample at all
    ref = run_oracle(oracle, w)
    cube, wmap, cnt, st = run_gpu(w, "f32", {binding.OPT_KERNEL: 7})
    assert st["kernel"] == 8
    compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32, qmax(w))
    w.lon, w.lat, w.values, w.weights = w.lon[:0], w.lat[:0], w.values[:0], w.weights[:0]
    cube, wmap, cnt, st = run_gpu(w, "f32", {binding.OPT_KERNEL: 7})
    assert np.all(np.isnan(cube)) and np.all(wmap == 0) and np.all(cnt == 0)


@pytest.mark.parametrize("radius_deg,sigma_deg", [(0.1, 0.04), (0.2, 0.08), (0.225, 0.05)])
def test_tc_kernel_series_modes(oracle, radius_deg, sigma_deg):
    """Wider kernels switch the pair arithmetic to the series / full modes; several ring-table passes."""
    from paper_2012_13173_b200 import binding
    rng = np.random.default_rng(78)
    n = 6000
    w = workloads.make(1, 1.0)
    w.lon = 200.0 + rng.uniform(-2.0, 2.0, n)
    w.lat = 40.0 + rng.uniform(-2.0, 2.0, n)
    w.values = rng.normal(size=(n, 32)).astype(np.float32)
    w.sigma_deg, w.radius_deg, w.nside = sigma_deg, radius_deg, 256
    w.target = workloads.CarTarget(23, 19, 199.0, 39.1, 0.09, 0.1)
    ref = run_oracle(oracle, w)
    cube, wmap, cnt, st = run_gpu(w, "f32", {binding.OPT_KERNEL: 7})
    assert st["kernel"] == 8
    compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32)


def test_tc_kernel_many_rings_per_tile(oracle):
    """nside 16384 (the largest) under a 4.5' kernel: a tile's ring range (~200) exceeds one 128-entry table pass."""
    from paper_2012_13173_b200 import binding
    rng = np.random.default_rng(79)
    n = 30000
    w = workloads.make(1, 1.0)
    w.lon = 100.0 + rng.uniform(-0.5, 0.5, n)
    w.lat = -10.0 + rng.uniform(-0.5, 0.5, n)
    w.values = rng.normal(size=(n, 32)).astype(np.float32)
    w.sigma_deg, w.radius_deg, w.nside = 4.5 / 60, 13.5 / 60, 16384
    w.target = workloads.CarTarget(20, 12, 99.8, -10.15, 2.0 / 60, -(-2.0) / 60)
    ref = run_oracle(oracle, w)
    cube, wmap, cnt, st = run_gpu(w, "f32", {binding.OPT_KERNEL: 7})
    assert st["kernel"] == 8
    compare(cube, wmap, cnt, ref, w.sigma_deg, w.radius_deg, TOL_F32)


def test_tc_kernel_accumulate_batches(oracle):
    from paper_2012_13173_b200 import binding
    w = _cube_case(6, 64, n=9000)
    ref = run_oracle(oracle, w)
    g = binding.HCGrid(w.sigma_deg, w.radius_deg, w.nside, precision="f32")
    g.set_option(binding.OPT_KERNEL, 7)
    t = w.target
    g.set_target_car(t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat)
    dev = lambda a: torch.as_tensor(np.ascontiguousarray(a)).cuda()
    for lo, hi in ((0, 4000), (4000, 4000), (4000, 9000)):
        g.accumulate(dev(w.lon[lo:hi]), dev(w.lat[lo:hi]), dev(w.values[lo:hi]), dev(w.weights[lo:hi]))
    cube, wmap, cnt = g.finalize()
    torch.cuda.synchronize()
    g.close()
    compare(cube.cpu().numpy(), wmap.cpu().numpy(), cnt.cpu().numpy(), ref, w.sigma_deg, w.radius_deg, TOL_F32, qmax(w))
