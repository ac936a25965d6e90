"""hcgrid_count_hits_static, the entry point that allocates nothing (its scratch is a fixed __device__ array inside
the library): its output against the existing path's -- hcgrid_stats.n_hit, which sum_counts_kernel forms in a
cudaMalloc'ed buffer under HCGRID_OPT_PROFILE -- on calls in a row that share the scratch array.  Integer sums: exact.

Collected last on purpose (pytest -x: a failure here must not hide other tests).
"""
import numpy as np
import pytest

from paper_2012_13173_b200 import workloads

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _dev(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


def _grid_with_profile(cfg, scale):
    """(count output, n_hit of the existing path) of one hcgrid_grid call."""
    from paper_2012_13173_b200 import binding
    w = workloads.make(cfg, scale)
    t = w.target
    g = binding.HCGrid(w.sigma_deg, w.radius_deg, w.nside)
    g.set_option(binding.OPT_PROFILE, 1)
    g.set_target_car(t.nx, t.ny, t.lon0, t.lat0, t.dlon, t.dlat)
    cube, wmap, cnt = g.grid(_dev(w.lon), _dev(w.lat), _dev(w.values), None if w.weights is None else _dev(w.weights))
    torch.cuda.synchronize()
    n_hit = g.stats()["n_hit"]
    g.close()
    assert n_hit > 0
    return cnt, wmap, n_hit


def test_two_calls_in_a_row_match_the_existing_path():
    from paper_2012_13173_b200 import binding
    out = torch.full((2,), -1, dtype=torch.int64, device="cuda")
    # first call, second call with another problem (other size, other grid shape), then the first again: the shared
    # scratch keeps the previous call's partial sums and must not leak them
    cases = [_grid_with_profile(1, 1.0), _grid_with_profile(3, 0.05), _grid_with_profile(1, 1.0)]
    for cnt, wmap, n_hit in cases:
        r = binding.count_hits_static(cnt, out)
        assert r is out
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        assert int(got[0]) == n_hit == int(cnt.sum(dtype=torch.int64).item())
        assert int(got[1]) == int((cnt > 0).sum().item()) == int((wmap > 0).sum().item())
    # back to back on the stream without a host synchronisation in between, each into its own output
    outs = [torch.empty(2, dtype=torch.int64, device="cuda") for _ in cases]
    for (cnt, _, _), o in zip(cases, outs):
        binding.count_hits_static(cnt, o)
    torch.cuda.synchronize()
    for (cnt, _, n_hit), o in zip(cases, outs):
        assert int(o[0].item()) == n_hit


@pytest.mark.parametrize("ncell", [0, 1, 255, 2049, 300_001, 5_000_000])
def test_sizes_from_empty_to_every_block(ncell):
    """One block, a ragged tail, and more cells than 1024 blocks x 256 threads take in one sweep (grid-stride)."""
    from paper_2012_13173_b200 import binding
    gen = torch.Generator(device="cuda")
    gen.manual_seed(13173 + ncell)
    cnt = torch.randint(0, 2000, (ncell,), dtype=torch.int32, device="cuda", generator=gen)
    cnt[cnt < 600] = 0                                              # ~30 % empty cells
    for _ in range(2):
        out = binding.count_hits_static(cnt)
        torch.cuda.synchronize()
        assert int(out[0].item()) == int(cnt.sum(dtype=torch.int64).item())
        assert int(out[1].item()) == int((cnt > 0).sum().item())
    if ncell > 10:                                                   # a prefix of a larger array
        out = binding.count_hits_static(cnt, ncell=ncell // 3)
        torch.cuda.synchronize()
        assert int(out[0].item()) == int(cnt[:ncell // 3].sum(dtype=torch.int64).item())


def test_sizes_beyond_the_maximum_are_refused():
    from paper_2012_13173_b200 import binding
    assert binding.static_max_cells() == 1 << 30
    cnt = torch.ones(16, dtype=torch.int32, device="cuda")
    out = torch.full((2,), -7, dtype=torch.int64, device="cuda")
    with pytest.raises(binding.HCGridError) as e:
        binding.count_hits_static(cnt, out, ncell=(1 << 30) + 1)     # refused before anything is launched
    assert "at most" in str(e.value)
    with pytest.raises(binding.HCGridError):
        binding.count_hits_static(cnt, out, ncell=-1)
    torch.cuda.synchronize()
    assert out.tolist() == [-7, -7]
    binding.count_hits_static(cnt, out)                              # and the entry point still works afterwards
    torch.cuda.synchronize()
    assert out.tolist() == [16, 16]
