"""The N > 1 plumbing of bench.py on CPU: world_size 2, gloo backend (no GPU needed)."""
import os
import socket

import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    from paper_2012_13173_b200 import dist as hdist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE=str(world), RANK=str(rank),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    assert hdist.env_world() == (world, rank, rank)
    hdist.barrier(world)
    # rank r "measured" (10 + r, 3 - r) ms: the job is as slow as the slowest rank, per quantity
    mx = hdist.max_over_ranks([10.0 + rank, 3.0 - rank], world)
    rate = hdist.whole_job_rate(units_per_rank=1000, world=world, steps=4, ms_total_max=mx[0])
    out.put((rank, mx, rate))
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_rate_world2():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, mx, rate in got:
        assert mx == [11.0, 3.0]                       # max over ranks of each timing
        assert rate == pytest.approx(1000 * 2 * 4 / 11.0e-3)   # units of ALL ranks / slowest time


def test_single_rank_needs_no_process_group():
    from paper_2012_13173_b200 import dist as hdist
    assert hdist.max_over_ranks([1.5, 2.5], 1) == [1.5, 2.5]
    hdist.barrier(1)
    assert hdist.whole_job_rate(10, 1, 2, 4.0) == pytest.approx(10 * 2 / 4e-3)


def test_row_bands_partition_the_target():
    from paper_2012_13173_b200 import dist as hdist
    for ny in (1, 7, 300, 1201):
        for world in (1, 2, 3, 8):
            for align in (1, 2, 4):
                rows = []
                for r in range(world):
                    a, b = hdist.row_band(ny, world, r, align)
                    assert 0 <= a <= b <= ny and (a % align == 0 or a == ny)
                    rows += list(range(a, b))
                assert rows == list(range(ny))           # every row exactly once, in order


def test_band_sharding_equals_the_whole_problem(oracle):
    """Gridding each band with only its latitude-selected samples and concatenating the bands
    gives exactly the oracle's result on the whole target (the halo selection is a superset)."""
    import numpy as np
    from paper_2012_13173_b200 import dist as hdist, workloads
    w = workloads.make(1, 1.0)
    t = w.target
    cl, cb = t.cell_centers()
    full = oracle.grid(w.sigma_deg, w.radius_deg, cl, cb, w.lon, w.lat, w.values, None)
    world = 3
    cubes, wmaps, counts, kept = [], [], [], 0
    for r in range(world):
        a, b = hdist.row_band(t.ny, world, r, align=2)
        bt = hdist.band_target(t, a, b)
        m = hdist.band_sample_mask(w.lat, t, a, b, w.radius_deg)
        kept += int(m.sum())
        bl, bb = bt.cell_centers()
        assert np.array_equal(bl, cl[a * t.nx:b * t.nx])
        np.testing.assert_allclose(bb, cb[a * t.nx:b * t.nx], rtol=0, atol=1e-12)
        res = oracle.grid(w.sigma_deg, w.radius_deg, cl[a * t.nx:b * t.nx], cb[a * t.nx:b * t.nx], w.lon[m], w.lat[m],
                          w.values[m], None)
        cubes.append(res.datacube); wmaps.append(res.weightmap); counts.append(res.counts)
    assert np.array_equal(np.concatenate(counts), full.counts)
    np.testing.assert_allclose(np.concatenate(wmaps), full.weightmap, rtol=1e-13)
    np.testing.assert_allclose(np.concatenate(cubes), full.datacube, rtol=1e-11, equal_nan=True)
    assert kept < world * w.n                              # the bands do not all need every sample
