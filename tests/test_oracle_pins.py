"""Pins for the brute-force oracle (oracle/): it is checked against what the paper and the
mathematics fix, not against itself.

Eq. 1 + Gaussian kernel truncated at sphere_radius.
Each test names the mistake it is meant to catch.
"""
import math
import os

import numpy as np
import pytest
from hypothesis import given, settings, strategies as st

from paper_2012_13173_b200 import workloads

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
AM = 1.0 / 60.0


def vec_dist(lon1, lat1, lon2, lat2):
    """Independent great-circle formula: atan2(|a x b|, a . b) on fp64 unit vectors
    (textbook; shares nothing with the oracle's haversine)."""
    l1, b1, l2, b2 = map(np.deg2rad, (lon1, lat1, lon2, lat2))
    a = np.stack([np.cos(b1) * np.cos(l1), np.cos(b1) * np.sin(l1), np.sin(b1)], -1)
    b = np.stack([np.cos(b2) * np.cos(l2), np.cos(b2) * np.sin(l2), np.sin(b2)], -1)
    a, b = np.broadcast_arrays(a, b)
    return np.arctan2(np.linalg.norm(np.cross(a, b), axis=-1), (a * b).sum(-1))


# ---------------------------------------------------------------- distance (reading c3)
def test_distance_closed_forms(oracle):
    # same meridian: d = |dlat|   (catches a missing 1/2 in the haversine, deg/rad slips)
    assert oracle.distance(10.0, -20.0, 10.0, 35.0) == pytest.approx(math.radians(55.0), abs=1e-15)
    # both on the equator: d = |dlon|, including across the 0/360 seam
    assert oracle.distance(3.0, 0.0, 47.0, 0.0) == pytest.approx(math.radians(44.0), abs=1e-15)
    assert oracle.distance(359.5, 0.0, 0.25, 0.0) == pytest.approx(math.radians(0.75), abs=1e-15)
    # across the pole: (l, 89.9) to (l+180, 89.9) is 0.2 deg  (catches a dropped cos factor)
    assert oracle.distance(12.0, 89.9, 192.0, 89.9) == pytest.approx(math.radians(0.2), abs=1e-13)
    # 1 deg of longitude at lat 60 is NOT 0.5 deg exactly: spherical law of cosines value
    d = math.acos(math.sin(math.radians(60)) ** 2 + math.cos(math.radians(60)) ** 2 * math.cos(math.radians(1)))
    assert oracle.distance(0.0, 60.0, 1.0, 60.0) == pytest.approx(d, rel=1e-9)
    # symmetric, zero on the diagonal, antipode = pi
    assert oracle.distance(5, 6, 7, 8) == oracle.distance(7, 8, 5, 6)
    assert oracle.distance(123.4, -56.7, 123.4, -56.7) == 0.0
    assert oracle.distance(0.0, 0.0, 180.0, 0.0) == pytest.approx(math.pi, abs=1e-12)


def test_distance_vs_vector_formula_near_pairs(oracle):
    rng = np.random.default_rng(7)
    lon1 = rng.uniform(0, 360, 20000)
    lat1 = np.degrees(np.arcsin(rng.uniform(-1, 1, 20000)))
    lon2 = lon1 + rng.uniform(-0.2, 0.2, 20000) / np.maximum(np.cos(np.deg2rad(lat1)), 0.05)
    lat2 = np.clip(lat1 + rng.uniform(-0.2, 0.2, 20000), -90, 90)
    ref = vec_dist(lon1, lat1, lon2, lat2)
    got = np.array([oracle.distance(a, b, c, d) for a, b, c, d in zip(lon1, lat1, lon2, lat2)])
    # both formulas are conditioned to ~1e-16 absolute on unit vectors at these separations
    assert np.max(np.abs(got - ref)) < 2e-15 + 1e-12 * np.max(ref)


# ---------------------------------------------------------------- hand case (golden)
def test_hand_3x3_golden(oracle):
    rows = np.loadtxt(os.path.join(GOLDEN, "hand_3x3.txt"))
    clon, clat = rows[:, 0] * AM, rows[:, 1] * AM
    slon = np.array([0, 1, 0, -1, 10]) * AM
    slat = np.array([0, 0, -1, 1, 10]) * AM
    val = np.array([1, 2, 4, 8, 100], dtype=np.float32)
    r = oracle.grid(1.0 * AM, 1.2 * AM, clon, clat, slon, slat, val)
    assert np.array_equal(r.counts, rows[:, 2].astype(np.int64))
    np.testing.assert_allclose(r.weightmap, rows[:, 3], rtol=1e-6)
    np.testing.assert_allclose(r.datacube[:, 0], rows[:, 4], rtol=1e-6)
    assert np.all(r.near_boundary == 0)


# ---------------------------------------------------------------- kernel + normalisation (c1, c5)
def test_single_sample_reproduces_gaussian_weight_map(oracle):
    sig, R = 2.0 * AM, 7.2 * AM   # no cell sits exactly on the boundary
    # cells on the sample's meridian: d = |dlat| in closed form (no distance code involved)
    off = np.linspace(-9, 9, 37) * AM
    clat = 40.0 + off
    clon = np.full_like(clat, 77.0)
    r = oracle.grid(sig, R, clon, clat, [77.0], [40.0], np.array([3.25], np.float32))
    d = np.abs(off)
    inside = d <= R
    expect = np.where(inside, np.exp(-np.deg2rad(d) ** 2 / (2 * np.deg2rad(sig) ** 2)), 0.0)
    np.testing.assert_allclose(r.weightmap, expect, rtol=1e-12, atol=0)
    assert np.array_equal(r.counts, inside.astype(np.int64))
    np.testing.assert_allclose(r.datacube[inside, 0], 3.25, rtol=4e-16)   # V = v wherever W > 0
    assert np.all(np.isnan(r.datacube[~inside, 0]))       # c5: empty cell -> NaN
    assert np.all(r.weightmap[~inside] == 0.0)
    # peak is 1 (no 1/(2 pi sigma^2) factor, reading c1)
    assert r.weightmap[off == 0][0] == 1.0
    # cells on the equator: d = |dlon| in closed form
    clon2 = 200.0 + off
    r2 = oracle.grid(sig, R, clon2, np.zeros_like(clon2), [200.0], [0.0], np.array([1.0], np.float32))
    d2 = np.abs(clon2 - 200.0)          # the representable offsets (200 + off rounds at 3e-14 deg)
    expect2 = np.where(d2 <= R, np.exp(-np.deg2rad(d2) ** 2 / (2 * np.deg2rad(sig) ** 2)), 0.0)
    np.testing.assert_allclose(r2.weightmap, expect2, rtol=1e-12)


def test_constant_field_grids_to_constant(oracle):
    w = workloads.make(1, scale=0.05)
    clon, clat = w.target.cell_centers()
    const = np.full((w.n, 1), 2.718281828, dtype=np.float32)
    r = oracle.grid(w.sigma_deg, w.radius_deg, clon, clat, w.lon, w.lat, const)
    ok = r.weightmap > 0
    assert ok.sum() > 0.9 * ok.size
    np.testing.assert_allclose(r.datacube[ok, 0], float(const[0, 0]), rtol=1e-15)
    np.testing.assert_allclose(r.absmap[ok, 0], float(const[0, 0]), rtol=1e-15)


def test_permutation_invariance(oracle):
    w = workloads.make(1, scale=0.05)
    clon, clat = w.target.cell_centers()
    r0 = oracle.grid(w.sigma_deg, w.radius_deg, clon, clat, w.lon, w.lat, w.values)
    p = np.random.default_rng(3).permutation(w.n)
    r1 = oracle.grid(w.sigma_deg, w.radius_deg, clon, clat, w.lon[p], w.lat[p], w.values[p])
    assert np.array_equal(r0.counts, r1.counts)
    np.testing.assert_allclose(r1.weightmap, r0.weightmap, rtol=1e-15)
    np.testing.assert_allclose(r1.datacube, r0.datacube, rtol=0, atol=1e-14 * np.nanmax(r0.absmap))


def test_rotation_about_pole_axis_and_seam(oracle):
    """Adding a constant to every longitude leaves the result unchanged; moving the patch
    onto the 0/360 seam exercises the wrap (catches a missing remainder / wrong sign)."""
    lon, lat, val, wts, clon, clat = workloads.random_case(1, 400, 60, 100.0, 55.0, 0.3)
    sig, R = 3 * AM, 9 * AM
    r0 = oracle.grid(sig, R, clon, clat, lon, lat, val)
    shift = 260.0 - 0.1     # patch now straddles lon = 0
    r1 = oracle.grid(sig, R, np.mod(clon + shift, 360), clat, np.mod(lon + shift, 360), lat, val)
    assert r0.counts.sum() > 0
    # the shift is not exact in fp64 (1 ulp of 360 = 6e-14 deg ~ 1e-15 rad): tolerance 1e-9 rel
    ok = r0.near_boundary == 0
    assert np.array_equal(r0.counts[ok], r1.counts[ok])
    np.testing.assert_allclose(r1.weightmap[ok], r0.weightmap[ok], rtol=1e-9)


# ---------------------------------------------------------------- brute force by another route
@settings(max_examples=25, deadline=None)
@given(seed=st.integers(0, 10_000), lat_c=st.sampled_from([0.0, 33.0, -61.0, 84.0, 89.7, -89.9]),
       lon_c=st.sampled_from([0.05, 180.0, 359.97]), nchan=st.sampled_from([1, 3]),
       use_w=st.booleans())
def test_brute_force_numpy_vector_formula(oracle, seed, lat_c, lon_c, nchan, use_w):
    """Eq. 1 re-evaluated with numpy broadcasting and the VECTOR distance formula
    (a different route to d), math.fsum-free plain float64 sums: counts equal away from
    the boundary, W and V to 1e-11."""
    lon, lat, val, wts, clon, clat = workloads.random_case(seed, 300, 25, lon_c, lat_c, 0.25,
                                                           nchan=nchan, with_weights=use_w)
    sig, R = 4 * AM, 10 * AM
    r = oracle.grid(sig, R, clon, clat, lon, lat, val, wts)
    d = vec_dist(clon[:, None], clat[:, None], lon[None, :], lat[None, :])
    Rr, sr = np.deg2rad(R), np.deg2rad(sig)
    inside = d <= Rr
    q = np.ones(lon.size) if wts is None else wts.astype(np.float64)
    w = np.where(inside, np.exp(-d * d / (2 * sr * sr)), 0.0) * q[None, :]
    W = w.sum(1)
    S = w @ val.astype(np.float64)
    band = (np.abs(d - Rr) < 1e-9).sum(1)
    assert np.all(np.abs(inside.sum(1) - r.counts) <= band)
    np.testing.assert_allclose(r.weightmap, W, rtol=1e-11, atol=1e-300)
    ok = W > 0
    np.testing.assert_allclose(r.datacube[ok], S[ok] / W[ok, None], rtol=0,
                               atol=1e-11 * max(1.0, float(np.nanmax(r.absmap[ok]))))
    assert np.all(np.isnan(r.datacube[~ok]))


# ---------------------------------------------------------------- weights (c6) and channels (c7)
def test_weight_semantics(oracle):
    lon, lat, val, wts, clon, clat = workloads.random_case(5, 500, 40, 10.0, -30.0, 0.3,
                                                           with_weights=True)
    sig, R = 3 * AM, 9 * AM
    base = oracle.grid(sig, R, clon, clat, lon, lat, val)
    k = oracle.grid(sig, R, clon, clat, lon, lat, val, np.full(lon.size, 2.5, np.float32))
    np.testing.assert_allclose(k.weightmap, 2.5 * base.weightmap, rtol=1e-14)
    ok = base.weightmap > 0
    np.testing.assert_allclose(k.datacube[ok], base.datacube[ok], rtol=0, atol=1e-13)
    assert np.array_equal(k.counts, base.counts)
    # q in {0,1}: same W, V as dropping the zero-weight samples; count stays geometric
    m = np.random.default_rng(1).random(lon.size) < 0.6
    z = oracle.grid(sig, R, clon, clat, lon, lat, val, m.astype(np.float32))
    dpd = oracle.grid(sig, R, clon, clat, lon[m], lat[m], val[m])
    np.testing.assert_allclose(z.weightmap, dpd.weightmap, rtol=1e-14)
    ok2 = dpd.weightmap > 0
    np.testing.assert_allclose(z.datacube[ok2], dpd.datacube[ok2], rtol=0, atol=1e-13)
    assert np.array_equal(z.counts, base.counts)
    # general weights: W is linear in q
    a = oracle.grid(sig, R, clon, clat, lon, lat, val, wts)
    b = oracle.grid(sig, R, clon, clat, lon, lat, val, (2 * wts).astype(np.float32))
    np.testing.assert_allclose(b.weightmap, 2 * a.weightmap, rtol=1e-14)


def test_multichannel_is_per_channel(oracle):
    lon, lat, val, wts, clon, clat = workloads.random_case(9, 300, 30, 250.0, 12.0, 0.2, nchan=5)
    sig, R = 3 * AM, 9 * AM
    full = oracle.grid(sig, R, clon, clat, lon, lat, val)
    for k in range(5):
        one = oracle.grid(sig, R, clon, clat, lon, lat, val[:, k].copy())
        assert np.array_equal(np.isnan(one.datacube[:, 0]), np.isnan(full.datacube[:, k]))
        ok = one.weightmap > 0
        assert np.array_equal(one.datacube[ok, 0], full.datacube[ok, k])
        assert np.array_equal(one.weightmap, full.weightmap)


# ---------------------------------------------------------------- boundary, empties, errors (c4)
def test_support_boundary_and_band(oracle):
    sig, R = 1.0, 3.0      # degrees; meridian pairs so d = |dlat| in closed form
    eps_deg = math.degrees(5e-10)
    clat = np.array([0.0, 0.0, 0.0, 0.0])
    slat = np.array([R - 10 * eps_deg, R - eps_deg, R + eps_deg, R + 10 * eps_deg])
    for i, (inside, band) in enumerate([(1, 0), (1, 1), (0, 1), (0, 0)]):
        r = oracle.grid(sig, R, [5.0], [0.0], [5.0], [slat[i]], np.array([1.0], np.float32))
        assert r.counts[0] == inside and r.near_boundary[0] == band


def test_empty_inputs_and_errors(oracle):
    r = oracle.grid(1 * AM, 3 * AM, [1.0, 2.0], [3.0, 4.0], [], [], np.zeros((0, 1), np.float32))
    assert np.all(r.weightmap == 0) and np.all(r.counts == 0) and np.all(np.isnan(r.datacube))
    r = oracle.grid(1 * AM, 3 * AM, [], [], [1.0], [1.0], np.ones((1, 1), np.float32))
    assert r.weightmap.size == 0
    with pytest.raises(ValueError):
        oracle.grid(0.0, 1.0, [0.0], [0.0], [0.0], [0.0], np.ones(1, np.float32))
    with pytest.raises(ValueError):
        oracle.grid(1.0, -1.0, [0.0], [0.0], [0.0], [0.0], np.ones(1, np.float32))


def test_duplicates_all_count(oracle):
    r = oracle.grid(1.0, 3.0, [0.0], [0.0], [0.5] * 4, [0.0] * 4, np.array([1, 2, 3, 6], np.float32))
    assert r.counts[0] == 4
    assert r.datacube[0, 0] == pytest.approx(3.0, rel=1e-15)
    assert r.weightmap[0] == pytest.approx(4 * math.exp(-0.5 * 0.25), rel=1e-14)


def test_batches_are_additive_in_the_unnormalised_sums(oracle):
    """Eq. 1 is a ratio of two sums over the samples, so gridding two batches and
    combining  V = (V_a W_a + V_b W_b) / (W_a + W_b),  W = W_a + W_b,  counts added,  must equal
    gridding their union (the semantics of incremental gridding, hcgrid_accumulate)."""
    rng = np.random.default_rng(31)
    n = 900
    lon = 10.0 + rng.uniform(-0.2, 0.2, n)
    lat = -30.0 + rng.uniform(-0.2, 0.2, n)
    val = rng.normal(size=(n, 3)).astype(np.float32)
    wts = rng.uniform(0.5, 1.5, n).astype(np.float32)
    gx, gy = np.meshgrid(10.0 + np.linspace(-0.45, 0.45, 9), -30.0 + np.linspace(-0.45, 0.45, 8))
    cl, cb = gx.ravel(), gy.ravel()
    sigma, radius = 2.0 / 60.0, 6.0 / 60.0
    cut = 350
    full = oracle.grid(sigma, radius, cl, cb, lon, lat, val, wts)
    a = oracle.grid(sigma, radius, cl, cb, lon[:cut], lat[:cut], val[:cut], wts[:cut])
    b = oracle.grid(sigma, radius, cl, cb, lon[cut:], lat[cut:], val[cut:], wts[cut:])
    w = a.weightmap + b.weightmap
    s = np.nan_to_num(a.datacube) * a.weightmap[:, None] + np.nan_to_num(b.datacube) * b.weightmap[:, None]
    with np.errstate(invalid="ignore", divide="ignore"):
        v = np.where(w[:, None] > 0, s / w[:, None], np.nan)
    assert np.array_equal(a.counts + b.counts, full.counts)
    np.testing.assert_allclose(w, full.weightmap, rtol=1e-13)
    np.testing.assert_allclose(v, full.datacube, rtol=1e-11, atol=1e-13, equal_nan=True)
    assert (full.weightmap == 0).any() and (full.weightmap > 0).any()      # the case has empty cells too


# ---------------------------------------------------------------- tapered-sinc kernel (S:8f NEXT-3)
def test_tapered_sinc_zeros_sign_and_special_points(oracle):
    """One sample on the cells' meridian, so d is a latitude difference exactly.  sinc(d/(b sigma)) has
    its zeros at d = k b sigma, is 1 at d = 0 and -2/(3 pi) at d = 1.5 b sigma (sin(3 pi/2) = -1);
    catches: a missing pi, a and b swapped, sigma^2 against sigma, a Gaussian taper with the
    factor 1/2 left in."""
    sigma, a, b = 0.1, 2.52, 1.55
    d_deg = np.array([0.0, b * sigma, 2 * b * sigma, 1.5 * b * sigma, 0.5 * b * sigma])
    res = oracle.grid(sigma, 5 * sigma, np.full(5, 40.0), 10.0 + d_deg, [40.0], [10.0], [2.0],
                      kernel=(oracle.TAPERED_SINC, a, b))
    w = res.weightmap
    assert w[0] == 1.0
    assert abs(w[1]) < 1e-12 and abs(w[2]) < 1e-12                      # zeros of the sinc
    assert w[3] == pytest.approx(-2.0 / (3.0 * math.pi) * math.exp(-(1.5 * b / a) ** 2), rel=1e-12)
    assert w[4] == pytest.approx(2.0 / math.pi * math.exp(-(0.5 * b / a) ** 2), rel=1e-12)   # sin(pi/2) = 1
    assert np.all(res.counts == 1)
    assert np.allclose(res.datacube[[0, 3, 4], 0], 2.0, rtol=1e-12)     # one sample: V = v whatever the sign of w
    assert np.allclose(res.abswmap, np.abs(w), rtol=0, atol=1e-18)


def test_tapered_sinc_reduces_to_the_gaussian(oracle):
    """b -> infinity switches the sinc off; what is left, exp(-(d/(a sigma))^2), is the Gaussian of
    width a sigma / sqrt 2 -- the routine pinned above.  Catches: taper exponent, any change to the
    distance or the accumulation on the kernel path."""
    rng = np.random.default_rng(5)
    n = 400
    lon = 100.0 + rng.uniform(-0.5, 0.5, n)
    lat = -30.0 + rng.uniform(-0.5, 0.5, n)
    val = rng.normal(size=(n, 3)).astype(np.float32)
    wts = rng.uniform(0.5, 2.0, n).astype(np.float32)
    clon, clat = np.meshgrid(100.0 + np.linspace(-0.4, 0.4, 7), -30.0 + np.linspace(-0.4, 0.4, 7))
    sigma, a = 0.05, 2.52
    k = oracle.grid(sigma, 0.2, clon, clat, lon, lat, val, wts, kernel=(oracle.TAPERED_SINC, a, 1e12))
    g = oracle.grid(a * sigma / math.sqrt(2.0), 0.2, clon, clat, lon, lat, val, wts)
    assert np.array_equal(k.counts, g.counts)
    assert np.allclose(k.weightmap, g.weightmap, rtol=1e-12)
    assert np.allclose(k.datacube, g.datacube, rtol=1e-11, atol=1e-13, equal_nan=True)
    # and ktype 0 through the kernel entry IS the Gaussian entry
    k0 = oracle.grid(sigma, 0.2, clon, clat, lon, lat, val, wts, kernel=(oracle.GAUSS, 0.0, 0.0))
    g0 = oracle.grid(sigma, 0.2, clon, clat, lon, lat, val, wts)
    assert np.array_equal(k0.weightmap, g0.weightmap) and np.array_equal(k0.datacube, g0.datacube, equal_nan=True)


def test_tapered_sinc_constant_field_and_negative_lobes(oracle):
    """Eq. 1 normalises by W, so a constant field grids to the constant wherever W != 0 even
    with negative weights; with R = 3 sigma (> b sigma) some pairs do sit in the negative lobe."""
    rng = np.random.default_rng(6)
    n = 3000
    lon = 10.0 + rng.uniform(-1, 1, n)
    lat = 50.0 + rng.uniform(-1, 1, n)
    clon, clat = np.meshgrid(10.0 + np.linspace(-0.8, 0.8, 9), 50.0 + np.linspace(-0.8, 0.8, 9))
    res = oracle.grid(0.1, 0.3, clon, clat, lon, lat, np.full(n, 3.25, np.float32),
                      kernel=(oracle.TAPERED_SINC, 2.52, 1.55))
    assert np.all(res.counts > 0)
    assert np.all(res.abswmap > np.abs(res.weightmap) * (1 + 1e-9))     # negative contributions exist
    assert np.allclose(res.datacube[:, 0], 3.25, rtol=1e-10)
    with pytest.raises(ValueError):
        oracle.grid(0.1, 0.3, [0.0], [0.0], [0.0], [0.0], [1.0], kernel=(1, 2.52, 0.0))
    with pytest.raises(ValueError):
        oracle.grid(0.1, 0.3, [0.0], [0.0], [0.0], [0.0], [1.0], kernel=(7, 1.0, 1.0))


# ---------------------------------------------------------------- elliptical Gaussian kernel (S:8f NEXT-3, reading c17)
def _ell(oracle, s1, ratio, pa, clon, clat, lon, lat, val=None, wts=None, radius=None):
    val = np.ones(np.size(lon), np.float32) if val is None else val
    return oracle.grid(s1, radius or 5 * s1 * max(1.0, ratio), clon, clat, lon, lat, val, wts,
                       kernel=(oracle.ELLIPTICAL_GAUSS, ratio, pa))


def test_elliptical_equals_the_circular_gaussian_at_ratio_one(oracle):
    """s2 = s1: the exponent's second term is exactly zero, whatever the position angle -- bit for bit the routine
    pinned above.  Catches: any change to the distance, the support test or the accumulation on the ktype-2 path."""
    rng = np.random.default_rng(21)
    n = 500
    lon = 359.8 + rng.uniform(-0.5, 0.5, n)
    lat = 70.0 + rng.uniform(-0.5, 0.5, n)
    val = rng.normal(size=(n, 2)).astype(np.float32)
    wts = rng.uniform(0.5, 2.0, n).astype(np.float32)
    clon, clat = np.meshgrid(359.8 + np.linspace(-0.4, 0.4, 6), 70.0 + np.linspace(-0.4, 0.4, 5))
    g = oracle.grid(0.06, 0.21, clon, clat, lon, lat, val, wts)
    for pa in (0.0, 33.0, -120.0):
        e = oracle.grid(0.06, 0.21, clon, clat, lon, lat, val, wts, kernel=(oracle.ELLIPTICAL_GAUSS, 1.0, pa))
        assert np.array_equal(e.weightmap, g.weightmap) and np.array_equal(e.counts, g.counts)
        assert np.array_equal(e.datacube, g.datacube, equal_nan=True)


def test_elliptical_closed_forms_along_the_axes(oracle):
    """One sample due north / south of the cell (same meridian: d = |dlat|, bearing 0 / 180 deg) and one due east on
    the equator (d = dlon, bearing 90 deg).  PA = 0 puts axis 1 on the meridian, PA = 90 on the east-west line, PA = 45
    halves sin^2.  Catches: s1 and s2 swapped, PA measured from east, degrees taken as radians, a dropped 1/2."""
    s1, ratio = 0.1, 0.4
    s2 = s1 * ratio
    d = 0.07
    g1, g2 = math.exp(-d * d / (2 * s1 * s1)), math.exp(-d * d / (2 * s2 * s2))
    g45 = math.exp(-d * d / 4 * (1 / s1 ** 2 + 1 / s2 ** 2))
    for (clon, clat, slon, slat) in [(40.0, 10.0, 40.0, 10.0 + d), (40.0, 10.0, 40.0, 10.0 - d),
                                     (200.0, -35.0, 200.0, -35.0 + d), (12.0, 0.0, 12.0 + d, 0.0),
                                     (359.99, 0.0, 359.99 + d - 360.0, 0.0), (12.0, 0.0, 12.0 - d, 0.0)]:
        on_meridian = clon == slon
        for pa, want in [(0.0, g1 if on_meridian else g2), (90.0, g2 if on_meridian else g1), (180.0, g1 if on_meridian else g2),
                         (-90.0, g2 if on_meridian else g1), (45.0, g45), (135.0, g45)]:
            w = _ell(oracle, s1, ratio, pa, [clon], [clat], [slon], [slat], radius=0.2).weightmap[0]
            assert w == pytest.approx(want, rel=2e-12), (clon, clat, slon, slat, pa)
    # coincident pair: weight 1 whatever the angle (the bearing of a zero offset is irrelevant)
    assert _ell(oracle, s1, ratio, 77.0, [5.0], [5.0], [5.0], [5.0], radius=0.2).weightmap[0] == 1.0


def test_elliptical_position_angle_runs_from_north_through_east(oracle):
    """A sample to the north-east of a cell on the equator, placed so that its bearing is exactly 45 deg
    (tan lat_s = sin dlon): PA = +45 puts it on axis 1, PA = -45 on axis 2.  Catches a mirrored position angle
    (north through west) and a bearing built with the arguments of atan2 exchanged."""
    s1, ratio = 0.1, 0.5
    dlon = 0.05
    slat = math.degrees(math.atan(math.sin(math.radians(dlon))))
    d = oracle.distance(30.0, 0.0, 30.0 + dlon, slat)
    on1 = math.exp(-d * d / (2 * math.radians(s1) ** 2))
    on2 = math.exp(-d * d / (2 * math.radians(s1 * ratio) ** 2))
    assert _ell(oracle, s1, ratio, 45.0, [30.0], [0.0], [30.0 + dlon], [slat]).weightmap[0] == pytest.approx(on1, rel=1e-11)
    assert _ell(oracle, s1, ratio, -45.0, [30.0], [0.0], [30.0 + dlon], [slat]).weightmap[0] == pytest.approx(on2, rel=1e-11)
    # the mirror image (north-west) swaps the two
    assert _ell(oracle, s1, ratio, 45.0, [30.0], [0.0], [30.0 - dlon], [slat]).weightmap[0] == pytest.approx(on2, rel=1e-11)


def test_elliptical_quarter_turn_swaps_the_axes_and_half_turn_changes_nothing(oracle):
    """(s1, s2, PA) and (s2, s1, PA + 90) describe the same ellipse; PA + 180 is the same axis."""
    rng = np.random.default_rng(22)
    n = 600
    lon = 120.0 + rng.uniform(-0.6, 0.6, n)
    lat = -48.0 + rng.uniform(-0.4, 0.4, n)
    val = rng.normal(size=(n, 2)).astype(np.float32)
    clon, clat = np.meshgrid(120.0 + np.linspace(-0.4, 0.4, 6), -48.0 + np.linspace(-0.3, 0.3, 5))
    s1, ratio, pa, radius = 0.09, 0.45, 27.0, 0.3
    a = oracle.grid(s1, radius, clon, clat, lon, lat, val, kernel=(oracle.ELLIPTICAL_GAUSS, ratio, pa))
    b = oracle.grid(s1 * ratio, radius, clon, clat, lon, lat, val, kernel=(oracle.ELLIPTICAL_GAUSS, 1.0 / ratio, pa + 90.0))
    c = oracle.grid(s1, radius, clon, clat, lon, lat, val, kernel=(oracle.ELLIPTICAL_GAUSS, ratio, pa + 180.0))
    assert a.counts.sum() > 0 and np.array_equal(a.counts, b.counts)
    assert np.allclose(a.weightmap, b.weightmap, rtol=1e-11) and np.allclose(a.weightmap, c.weightmap, rtol=1e-11)
    assert np.allclose(a.datacube, b.datacube, rtol=1e-10, atol=1e-12, equal_nan=True)
    assert np.allclose(a.datacube, c.datacube, rtol=1e-10, atol=1e-12, equal_nan=True)
    # and it is not the circular kernel
    g = oracle.grid(s1, radius, clon, clat, lon, lat, val)
    assert np.abs(a.weightmap - g.weightmap).max() > 1e-3 * g.weightmap.max()


@pytest.mark.parametrize("lon_c,lat_c,pa", [(0.0, 0.0, 30.0), (359.9, 62.0, -71.0), (181.0, -88.9, 100.0), (45.0, 89.5, 10.0)])
def test_elliptical_brute_force_with_tangent_vectors(oracle, lon_c, lat_c, pa):
    """Independent brute force in numpy: unit vectors, the cell's east / north tangent vectors, d from
    atan2(|c x s|, c . s), offsets along and across the axis by rotating (east, north) components -- the first form of
    the exponent, none of the oracle's haversine / bearing identities.  Includes polar caps and the lon = 0 seam."""
    rng = np.random.default_rng(23)
    n = 300
    s1, ratio, radius = 0.2, 0.35, 0.7
    lat = np.clip(lat_c + rng.uniform(-0.8, 0.8, n), -90.0, 90.0)
    lon = np.mod(lon_c + rng.uniform(-0.8, 0.8, n) / max(math.cos(math.radians(lat_c)), 0.02), 360.0)
    val = rng.normal(size=(n, 1)).astype(np.float32)
    wts = rng.uniform(0.5, 1.5, n).astype(np.float32)
    clat = np.clip(lat_c + np.array([-0.3, 0.0, 0.25, 0.4]), -89.99, 89.99)
    clon = np.mod(lon_c + np.array([0.2, 0.0, -0.3, 0.1]), 360.0)
    res = oracle.grid(s1, radius, clon, clat, lon, lat, val, wts, kernel=(oracle.ELLIPTICAL_GAUSS, ratio, pa))

    def unit(lo, la):
        lo, la = np.radians(lo), np.radians(la)
        return np.stack([np.cos(la) * np.cos(lo), np.cos(la) * np.sin(lo), np.sin(la)], -1)
    s = unit(lon, lat)
    S1, S2, R, PA = math.radians(s1), math.radians(s1 * ratio), math.radians(radius), math.radians(pa)
    for i in range(clon.size):
        c = unit(clon[i], clat[i])
        lo, la = math.radians(clon[i]), math.radians(clat[i])
        east = np.array([-math.sin(lo), math.cos(lo), 0.0])
        north = np.array([-math.sin(la) * math.cos(lo), -math.sin(la) * math.sin(lo), math.cos(la)])
        d = np.arctan2(np.linalg.norm(np.cross(c, s), axis=1), s @ c)
        x, y = s @ east, s @ north
        r = np.hypot(x, y)
        xi, eta = d * x / r, d * y / r                       # azimuthal equidistant offsets (east, north)
        u = eta * math.cos(PA) + xi * math.sin(PA)            # along the axis at PA (from north through east)
        v = xi * math.cos(PA) - eta * math.sin(PA)            # across it
        hit = d <= R
        assert np.abs(d - R).min() > 1e-7                     # no pair near the boundary in this draw
        w = np.exp(-u * u / (2 * S1 * S1) - v * v / (2 * S2 * S2)) * wts * hit
        assert res.counts[i] == hit.sum() and hit.sum() > 0
        assert res.weightmap[i] == pytest.approx(w.sum(), rel=1e-9)
        assert res.datacube[i, 0] == pytest.approx((w * val[:, 0]).sum() / w.sum(), rel=1e-8, abs=1e-11)


def test_elliptical_constant_field_and_errors(oracle):
    rng = np.random.default_rng(24)
    n = 2000
    lon = 10.0 + rng.uniform(-1, 1, n)
    lat = 50.0 + rng.uniform(-1, 1, n)
    clon, clat = np.meshgrid(10.0 + np.linspace(-0.8, 0.8, 9), 50.0 + np.linspace(-0.8, 0.8, 9))
    res = oracle.grid(0.1, 0.3, clon, clat, lon, lat, np.full(n, -1.75, np.float32),
                      kernel=(oracle.ELLIPTICAL_GAUSS, 0.5, 60.0))
    assert np.all(res.counts > 0) and np.all(res.weightmap > 0)
    assert np.allclose(res.datacube[:, 0], -1.75, rtol=1e-12)
    with pytest.raises(ValueError):
        oracle.grid(0.1, 0.3, [0.0], [0.0], [0.0], [0.0], [1.0], kernel=(2, 0.0, 10.0))
    with pytest.raises(ValueError):
        oracle.grid(0.1, 0.3, [0.0], [0.0], [0.0], [0.0], [1.0], kernel=(2, 0.5, float("nan")))
