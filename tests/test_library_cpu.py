"""CPU-only checks of the CUDA library: it builds, loads, exports every symbol include/hcgrid.h
declares, and its HEALPix RING code (step a2, compiled for the host) is self-consistent with
the published definition of the pixelisation.
No compute call needs a GPU here."""
import os
import re

import numpy as np
import pytest

from paper_2012_13173_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol(hcgrid_lib):
    hdr = open(os.path.join(ROOT, "include", "hcgrid.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(hcgrid_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert hasattr(hcgrid_lib, name), name


def test_create_fails_loudly_without_gpu_or_with_bad_args(hcgrid_lib):
    # invalid arguments are rejected before any CUDA call
    with pytest.raises(binding.HCGridError) as ei:
        binding.HCGrid(0.0, 1.0, 1024)
    assert ei.value.status == -1
    with pytest.raises(binding.HCGridError):
        binding.HCGrid(0.1, 0.3, 3)
    import torch
    if not torch.cuda.is_available():
        # no device: the product path refuses (no CPU fallback)
        with pytest.raises(binding.HCGridError) as ei:
            binding.HCGrid(0.1, 0.3, 1024)
        assert ei.value.status in (-4, -1)


def test_product_path_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2012_13173_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert "oracle" not in open(os.path.join(dirpath, f)).read().lower() or f == "workloads.py", f
    ora = os.path.join(ROOT, "oracle")
    for f in os.listdir(ora):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ora, f)).read()
            assert "import paper_2012_13173_b200" not in src and "from paper_2012_13173_b200" not in src
            assert "hcgrid.h" not in src


# ------------------------------------------------------------------ HEALPix RING self-consistency
def ring_table(nside):
    info = [binding.host_ring_info(nside, r) for r in range(1, 4 * nside)]
    return (np.array([i[0] for i in info]), np.array([i[1] for i in info]),
            np.array([i[2] for i in info]), np.array([i[3] for i in info]))


@pytest.mark.parametrize("nside", [1, 2, 4, 16, 64])
def test_ring_geometry_counts(nside):
    first, npix, lat, lon0 = ring_table(nside)
    assert npix.sum() == 12 * nside * nside
    assert first[0] == 0 and np.array_equal(first[1:], np.cumsum(npix)[:-1])
    assert np.all(np.diff(lat) < 0)                          # ring 1 is the northernmost
    assert np.allclose(lat, -lat[::-1], atol=1e-12)          # mirror symmetry
    z = np.sin(np.deg2rad(lat))
    i = np.arange(1, 4 * nside)
    zz = np.where(i < nside, 1 - i ** 2 / (3.0 * nside ** 2),
                  np.where(i <= 3 * nside, (2 * nside - i) * 2.0 / (3 * nside), -(1 - (4 * nside - i) ** 2 / (3.0 * nside ** 2))))
    assert np.allclose(z, zz, atol=1e-14)


def test_nside1_textbook():
    first, npix, lat, lon0 = ring_table(1)
    assert list(npix) == [4, 4, 4]
    assert np.allclose(np.sin(np.deg2rad(lat)), [2 / 3, 0.0, -2 / 3], atol=1e-15)
    assert np.allclose(lon0, [45.0, 0.0, 45.0])
    # the 12 base pixels: centres map to themselves
    lon = np.concatenate([lon0[k] + 90.0 * np.arange(4) for k in range(3)])
    la = np.repeat(lat, 4)
    assert list(binding.host_ang2pix_ring(1, lon, la)) == list(range(12))


@pytest.mark.parametrize("nside", [2, 4, 16, 64])
def test_pixel_centres_round_trip(nside):
    first, npix, lat, lon0 = ring_table(nside)
    lon = np.concatenate([lon0[r] + 360.0 / npix[r] * np.arange(npix[r]) for r in range(npix.size)])
    la = np.concatenate([np.full(npix[r], lat[r]) for r in range(npix.size)])
    assert np.array_equal(binding.host_ang2pix_ring(nside, lon, la), np.arange(12 * nside * nside))
    # longitude is periodic
    assert np.array_equal(binding.host_ang2pix_ring(nside, lon + 360.0, la), np.arange(12 * nside * nside))
    assert np.array_equal(binding.host_ang2pix_ring(nside, lon - 360.0, la), np.arange(12 * nside * nside))


@pytest.mark.parametrize("nside", [4, 16, 2048, 8192])
def test_containment_bounds_and_sorted_by_ring(nside):
    """The two facts the gather relies on: a point of pixel j in ring r lies within half the
    in-ring spacing of the pixel centre in longitude, and between the centre latitudes of
    rings r-1 and r+1.  And: sorted by pixel => sorted by ring."""
    rng = np.random.default_rng(nside)
    n = 200000
    lon = rng.uniform(0, 360, n)
    lat = np.degrees(np.arcsin(rng.uniform(-1, 1, n)))
    lat[:2000] = rng.uniform(89.0, 90.0, 2000)               # polar caps, densely
    lat[2000:4000] = rng.uniform(-90.0, -89.0, 2000)
    lat[4000:6000] = np.degrees(np.arcsin(2 / 3)) + rng.uniform(-0.01, 0.01, 2000)   # cap/belt transition
    pix = binding.host_ang2pix_ring(nside, lon, lat)
    assert pix.min() >= 0 and pix.max() < 12 * nside * nside
    i = np.arange(1, 4 * nside)
    ic = np.minimum(i, 4 * nside - i)
    npr = 4 * np.minimum(ic, nside)
    first = np.concatenate([[0], np.cumsum(npr)[:-1]])
    r = np.searchsorted(first, pix, side="right") - 1        # 0-based ring
    ring = r + 1
    j = pix - first[r]
    info_lat = np.empty(4 * nside + 1)
    info_lat[0], info_lat[-1] = 90.0, -90.0
    zc = np.where(i < nside, 1 - i.astype(float) ** 2 / (3.0 * nside ** 2),
                  np.where(i <= 3 * nside, (2 * nside - i) * 2.0 / (3 * nside),
                           -(1 - (4 * nside - i).astype(float) ** 2 / (3.0 * nside ** 2))))
    info_lat[1:-1] = np.degrees(np.arcsin(zc))
    assert np.all(lat <= info_lat[ring - 1] + 1e-9) and np.all(lat >= info_lat[ring + 1] - 1e-9)
    belt = (ring >= nside) & (ring <= 3 * nside)
    off = np.where(belt & (((ring - nside + 1) & 1) == 0), 0.0, 0.5)   # centre of pixel 0 in pixel units
    centre = (j + off) * 360.0 / npr[r]
    d = np.abs((lon - centre + 180.0) % 360.0 - 180.0)
    assert np.all(d <= 180.0 / npr[r] * (1 + 1e-9))
    order = np.argsort(pix, kind="stable")
    assert np.all(np.diff(ring[order]) >= 0)
