"""Replay of repeated hcgrid_grid calls as a CUDA graph (HCGRID_OPT_GRAPH; small problems are bound by launch gaps):
the replayed call must read the arrays' current contents and give what an eager call gives, and anything that changes
what a launch depends on must fall back to an eager call."""
import numpy as np
import pytest

from paper_2012_13173_b200 import workloads

from parity import TOL_F32, TOL_F64, compare

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _dev(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


def _oracle(oracle, w, values=None):
    cl, cb = w.target.cell_centers()
    return oracle.grid(w.sigma_deg, w.radius_deg, cl, cb, w.lon, w.lat, w.values if values is None else values, w.weights)


@pytest.mark.parametrize("cfg,scale,precision", [(1, 1.0, "f32"), (1, 1.0, "f64"), (4, 0.012, "f32"), (2, 0.03, "f32")])
def test_repeated_calls_replay_and_read_current_contents(oracle, cfg, scale, precision):
    from paper_2012_13173_b200 import binding
    w = workloads.make(cfg, scale)
    t = w.target
    tol = TOL_F32 if precision == "f32" else TOL_F64
    g = binding.HCGrid(w.sigma_deg, w.radius_deg, w.nside, precision=precision)
    g.set_target_car(t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat)
    lon, lat, val = _dev(w.lon), _dev(w.lat), _dev(w.values)
    wts = None if w.weights is None else _dev(w.weights)
    dt = torch.float32 if precision == "f32" else torch.float64
    out = (torch.empty((t.ncell, w.nchan), dtype=dt, device="cuda"), torch.empty(t.ncell, dtype=dt, device="cuda"),
           torch.empty(t.ncell, dtype=torch.int32, device="cuda"))
    ref = _oracle(oracle, w)
    seen = []
    for _ in range(4):
        out[0].fill_(7.0); out[1].fill_(7.0); out[2].fill_(7)
        g.grid(lon, lat, val, wts, out=out)
        torch.cuda.synchronize()
        seen.append(g.stats()["graph"])
        compare(out[0].cpu().numpy(), out[1].cpu().numpy(), out[2].cpu().numpy(), ref, w.sigma_deg, w.radius_deg, tol,
                1.0 if w.weights is None else float(w.weights.max()))
    assert seen == [0, 1, 1, 1]                       # eager, captured, replayed, replayed
    eager = [x.clone() for x in out]
    # new contents in the same arrays: other values, and the samples mirrored about the field centre
    rng = np.random.default_rng(9)
    v2 = rng.standard_normal(w.values.shape).astype(np.float32)
    lon2 = (2 * (t.lon0 + 0.5 * (t.nx - 1) * t.dlon) - w.lon) % 360.0
    val.copy_(_dev(v2)); lon.copy_(_dev(lon2))
    g.grid(lon, lat, val, wts, out=out)
    torch.cuda.synchronize()
    assert g.stats()["graph"] == 1 and g.stats()["n_kept"] > 0
    cl, cb = t.cell_centers()
    ref2 = oracle.grid(w.sigma_deg, w.radius_deg, cl, cb, lon2, w.lat, v2, w.weights)
    compare(out[0].cpu().numpy(), out[1].cpu().numpy(), out[2].cpu().numpy(), ref2, w.sigma_deg, w.radius_deg, tol,
            1.0 if w.weights is None else float(w.weights.max()))
    assert not torch.equal(out[1], eager[1])
    # the replay is bit-identical to an eager call on the same contents
    g.set_option(binding.OPT_GRAPH, 0)
    out2 = tuple(torch.empty_like(x) for x in out)
    g.grid(lon, lat, val, wts, out=out2)
    torch.cuda.synchronize()
    assert g.stats()["graph"] == 0
    for a, b in zip(out, out2):
        assert torch.equal(a.nan_to_num(nan=-1.0), b.nan_to_num(nan=-1.0))
    g.close()


def test_anything_a_launch_depends_on_ends_the_replay(oracle):
    from paper_2012_13173_b200 import binding
    w = workloads.make(1, 1.0)
    t = w.target
    g = binding.HCGrid(w.sigma_deg, w.radius_deg, w.nside)
    g.set_target_car(t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat)
    lon, lat, val = _dev(w.lon), _dev(w.lat), _dev(w.values)
    ref = _oracle(oracle, w)

    def call(**kw):
        r = g.grid(kw.get("lon", lon), lat, val, **{k: v for k, v in kw.items() if k != "lon"})
        torch.cuda.synchronize()
        return r, g.stats()["graph"]

    def check(r):
        compare(r[0].cpu().numpy(), r[1].cpu().numpy(), None if r[2] is None else r[2].cpu().numpy(), ref, w.sigma_deg,
                w.radius_deg, TOL_F32)

    out = (torch.empty((t.ncell, 1), device="cuda"), torch.empty(t.ncell, device="cuda"),
           torch.empty(t.ncell, dtype=torch.int32, device="cuda"))
    assert [call(out=out)[1] for _ in range(3)] == [0, 1, 1]
    g.set_option(binding.OPT_KERNEL, binding.KERNEL_GENERAL)          # an option
    r, gr = call(out=out); assert gr == 0 and g.stats()["kernel"] == 3; check(r)
    r, gr = call(out=out); assert gr == 1 and g.stats()["kernel"] == 3; check(r)
    g.set_option(binding.OPT_KERNEL, binding.KERNEL_AUTO)
    lon_b = lon.clone()                                                 # another input array
    r, gr = call(out=out, lon=lon_b); assert gr == 0; check(r)
    r, gr = call(out=out); assert gr == 0; check(r)                     # back to the first: the key changed again
    r, gr = call(out=out); assert gr == 1; check(r)
    out_nc = (out[0], out[1], None)                                     # without the count output
    r, gr = call(out=out_nc, want_counts=False); assert gr == 0; check(r)
    r, gr = call(out=out_nc, want_counts=False); assert gr == 1; check(r)
    g.set_kernel(binding.KERNEL_ELLIPTICAL_GAUSS, 0.5, 30.0)            # another kernel function
    r, gr = call(out=out_nc, want_counts=False); assert gr == 0
    cl, cb = t.cell_centers()
    ref_e = oracle.grid(w.sigma_deg, w.radius_deg, cl, cb, w.lon, w.lat, w.values, None,
                        kernel=(oracle.ELLIPTICAL_GAUSS, 0.5, 30.0))
    compare(r[0].cpu().numpy(), r[1].cpu().numpy(), None, ref_e, w.sigma_deg, w.radius_deg, TOL_F32)
    r, gr = call(out=out_nc, want_counts=False); assert gr == 1
    compare(r[0].cpu().numpy(), r[1].cpu().numpy(), None, ref_e, w.sigma_deg, w.radius_deg, TOL_F32)
    g.set_kernel(binding.KERNEL_GAUSS)
    r, gr = call(out=out_nc, want_counts=False); assert gr == 0; check(r)
    g.set_target_car(t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat)       # a new target, even if equal
    r, gr = call(out=out_nc, want_counts=False); assert gr == 0; check(r)
    g.set_option(binding.OPT_PROFILE, 1)                               # per-stage events need an eager call
    for _ in range(3):
        r, gr = call(out=out); assert gr == 0; check(r)
    assert g.stats()["us_total"] > 0
    g.set_option(binding.OPT_PROFILE, 0)
    s = torch.cuda.Stream()                                             # a side stream
    with torch.cuda.stream(s):
        for want in (0, 1, 1):
            r = g.grid(lon, lat, val, out=out)
            s.synchronize()
            assert g.stats()["graph"] == want
            check(r)
    g.close()


def test_large_inputs_are_not_captured_unless_asked():
    from paper_2012_13173_b200 import binding
    w = workloads.make(3, 0.25)                                          # 2.5e6 samples > 2^21
    t = w.target
    g = binding.HCGrid(w.sigma_deg, w.radius_deg, w.nside)
    g.set_target_car(t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat)
    lon, lat, val = _dev(w.lon), _dev(w.lat), _dev(w.values)
    out = (torch.empty((t.ncell, 1), device="cuda"), torch.empty(t.ncell, device="cuda"), None)
    for _ in range(3):
        g.grid(lon, lat, val, want_counts=False, out=out)
        assert g.stats()["graph"] == 0
    eager = out[1].clone()
    g.set_option(binding.OPT_GRAPH, 1)
    seen = []
    for _ in range(3):
        g.grid(lon, lat, val, want_counts=False, out=out)
        torch.cuda.synchronize()
        seen.append(g.stats()["graph"])
    assert seen == [0, 1, 1]
    assert torch.equal(eager, out[1])
    g.close()
