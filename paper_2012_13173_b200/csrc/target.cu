// target.cu -- step a1: target set-up.
//
// From the target cells and the kernel support radius R this derives (i) the REGION of
// the sphere the target can reach -- the ring range [ring_first, ring_first + nring) and
// the longitude window [lon_lo, lon_lo + wx) -- which fixes the layout of the ring table
// and the per-pixel table, and (ii) per (strip, ring) the lookup-bin window of the
// support disc, PAPER.md:136 step (i) "minimum and maximum ring indices within the range
// of influence" and step (ii) "starting contributing pixel" of each ring.
//
// Disc geometry: a disc of radius R centred at latitude phi_c has, at latitude phi, the
// longitude half-width dl with
//     sin^2(dl/2) = [sin^2(R/2) - sin^2((phi - phi_c)/2)] / (cos(phi) cos(phi_c)),
// maximal at sin(phi*) = sin(phi_c) / cos(R).  A point in HEALPix ring r has a latitude
// between the centres of rings r+1 and r-1 (hcg_healpix.cuh fact 2), so the window of ring
// r is the half-width at phi* clamped into that band (clipped to phi_c +- R).
#include <algorithm>
#include <cmath>
#include <vector>

#include "hcg_common.cuh"

namespace hcg {

__global__ void ring_window_kernel(const Strip* __restrict__ strips, RingWin* __restrict__ wins,
                                   RingWinF* __restrict__ winsf, int nstrip, int kmax, Region rg,
                                   double radius) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)nstrip * kmax) return;
    const int s = (int)(t / kmax), k = (int)(t % kmax);
    const Strip st = strips[s];
    RingWin w;
    w.a_lo = w.a_hi = w.step = 0.0;
    w.ring_rel = st.ring_lo + k;
    w.flags = 0;
    w.nb = 0;
    w.pad_ = 0;
    if (k < st.nring) {
        const int r = rg.ring_first + w.ring_rel;                  // HEALPix ring number
        const double eps = 1e-10;
        double band_hi = kHalfPi - ring_colat(r - 1, rg.nside) + eps;   // latitude band of ring r
        double band_lo = kHalfPi - ring_colat(r + 1, rg.nside) - eps;
        const double lo = fmax(band_lo, st.lat - radius);
        const double hi = fmin(band_hi, st.lat + radius);
        w.nb = (int)ring_nbins(r, rg.nside, rg.subpix);
        if (lo <= hi) {
            bool whole = fabs(st.lat) + radius >= kHalfPi - 1e-9;    // disc holds a pole
            double dl = 0.0;
            if (!whole) {
                const double sstar = sin(st.lat) / cos(radius);
                const double pstar = asin(fmin(1.0, fmax(-1.0, sstar)));
                const double pe = fmin(hi, fmax(lo, pstar));
                const double sr = sin(0.5 * radius), sd = sin(0.5 * (pe - st.lat));
                const double f = (sr * sr - sd * sd) / (cos(pe) * cos(st.lat));
                if (f >= 1.0) whole = true;
                else dl = 2.0 * asin(sqrt(fmax(f, 0.0))) + 1e-9;
            }
            if (whole) {
                w.flags = 2;
            } else {
                const double c = ldexp((double)ring_npix(r, rg.nside) / kTwoPi, rg.subpix);
                const double g0 = ring_bin_coord(r, rg.nside, rg.lon_lo, rg.subpix);
                const double frac0 = g0 - (floor(g0) - 2.0);       // in [2, 3)
                w.a_lo = frac0 + (st.u0 - dl) * c;
                w.a_hi = frac0 + (st.u0 + dl) * c;
                w.step = st.du * c;
                w.flags = 1;
            }
        }
    }
    wins[t] = w;
    // fp32 copy, bounds moved outwards by the fp32 evaluation error of a + ix * step
    // (|a + ix step| < m + 4, two roundings of 2^-24 relative each, plus step's own)
    const double slack = 2.5e-7 * ((double)rg.m + 8.0) + 1e-4;
    RingWinF f;
    f.a_lo = __double2float_rd(w.a_lo - slack);
    f.a_hi = __double2float_ru(w.a_hi + slack);
    f.step = (float)w.step;
    f.flags = w.flags;
    winsf[t] = f;
}

static double wrap_pm_pi(double x) {
    x = fmod(x + kPi, kTwoPi);
    if (x < 0) x += kTwoPi;
    return x - kPi;
}

struct HostStrip { double lon0_deg, dlon_deg, lat_deg; };

// Common tail of both set_target flavours: region, strips, ring windows.
static int finish_target(hcgrid_ctx* c, const std::vector<HostStrip>& hs, int strip_cells,
                         double west, double east /* unwrapped rad, of all cell centres */) {
    const double R = c->kp.radius;
    const int nside = c->nside;
    double latmin = 1e9, latmax = -1e9, maxabs = 0;
    for (const auto& h : hs) {
        const double la = h.lat_deg * kDeg2Rad;
        latmin = std::min(latmin, la); latmax = std::max(latmax, la);
        maxabs = std::max(maxabs, std::fabs(la));
    }
    Region rg{};
    rg.nside = nside;
    // rings the target can reach (PAPER.md:136 step i over the whole target)
    const double th_a = std::max(0.0, kHalfPi - (latmax + R));
    const double th_b = std::min(kPi, kHalfPi - (latmin - R));
    int rf = (int)std::floor(ring_coord(th_a, nside)) - 1;
    int rl = (int)std::ceil(ring_coord(th_b, nside)) + 1;
    rf = std::max(rf, 1); rl = std::min(rl, 4 * nside - 1);
    rg.ring_first = rf;
    rg.nring = rl - rf + 1;
    const bool pole = maxabs + R >= kHalfPi - 1e-6;
    const double dlmax = pole ? kPi : std::asin(std::min(1.0, std::sin(R) / std::cos(maxabs))) + 1e-9;
    int npr_max = 0, npr_min = 1 << 30;
    for (int r = rf; r <= rl; ++r) {
        npr_max = std::max(npr_max, ring_npix(r, nside));
        npr_min = std::min(npr_min, ring_npix(r, nside));
    }
    // sub-pixel bits: auto = 2 (quarter-pixel bins), reduced until the table fits
    int b = c->opt_subpix > -100 ? c->opt_subpix : (c->subpix_refined > -100 ? c->subpix_refined : 2);
    b = std::min(b, 6);
    const int64_t cap = (int64_t)1 << 28;
    for (;; --b) {
        const double binw = kTwoPi / std::ldexp((double)npr_min, b);   // widest bin, rad
        const double width = (east - west) + 2.0 * dlmax + 4.0 * binw + 1e-6;
        const bool full = pole || width >= 0.98 * kTwoPi;
        int64_t m;
        if (full) {
            m = 0;
            for (int r = rf; r <= rl; ++r) m = std::max<int64_t>(m, ring_nbins(r, nside, b));
        } else {
            m = (int64_t)std::ceil(width * std::ldexp((double)npr_max / kTwoPi, b)) + 6;
        }
        if (m * rg.nring <= cap || b < -20) {
            rg.subpix = b;
            rg.m = (int32_t)m;
            rg.full_circle = full ? 1 : 0;
            if (full) { rg.lon_lo = 0.0; rg.wx = kTwoPi; }
            else {
                double lo = std::fmod(west - dlmax - 2.0 * binw - 5e-7, kTwoPi);
                if (lo < 0) lo += kTwoPi;
                rg.lon_lo = lo; rg.wx = width;
            }
            break;
        }
    }
    if ((int64_t)rg.m * rg.nring > cap)
        return fail(c, HCGRID_ERR_UNSUPPORTED, "lookup table too large (%lld bins)",
                    (long long)rg.m * rg.nring);
    rg.nbins = (int64_t)rg.m * rg.nring;
    rg.lat_lo = kHalfPi - ring_colat(rl + 1, nside) - 1e-7;
    const double lat_hi = kHalfPi - ring_colat(rf - 1, nside) + 1e-7;
    rg.wy = lat_hi - rg.lat_lo;
    // Fixed-point scales of the packed records.  A kernel forms (int)(x_sample - x_cell0) for
    // every candidate of a task, and a task's cell 0 can be up to 8 columns / rows away from the
    // cell whose window brought the candidate in, so 2^32 must span at least twice that reach --
    // otherwise the difference wraps (a target of a handful of cells is narrower than that).
    {
        const double du_abs = strip_cells > 1 ? std::fabs(hs[0].dlon_deg) * kDeg2Rad : 0.0;
        const double dv_abs = strip_cells > 1 ? std::fabs(c->car_dlat) : 0.0;
        const double ring_sp = (lat_hi - rg.lat_lo) / std::max(1, rg.nring);
        const double span_x = rg.full_circle ? kTwoPi : std::max(rg.wx, 2.2 * (dlmax + 8.0 * du_abs));
        const double span_y = std::max(rg.wy, 2.2 * (R + 8.0 * dv_abs + 3.0 * ring_sp));
        rg.sx32 = 4294967296.0 / span_x;
        rg.sy32 = 4294967296.0 / span_y;
    }
    c->region = rg;

    // strips
    std::vector<Strip> st(hs.size());
    int kmax = 1;
    double cw = 1e9;
    const double sy = rg.sy32;
    for (size_t i = 0; i < hs.size(); ++i) {
        Strip& s = st[i];
        const HostStrip& h = hs[i];
        s.lon0_deg = h.lon0_deg; s.dlon_deg = h.dlon_deg; s.lat_deg = h.lat_deg;
        s.lat = h.lat_deg * kDeg2Rad;
        double u = std::fmod(h.lon0_deg * kDeg2Rad - rg.lon_lo, kTwoPi);
        if (u < 0) u += kTwoPi;
        s.u0 = u;
        s.du = h.dlon_deg * kDeg2Rad;
        const double ta = std::max(0.0, kHalfPi - (s.lat + R));
        const double tb = std::min(kPi, kHalfPi - (s.lat - R));
        int a = std::max(rf, (int)std::floor(ring_coord(ta, nside)) - 1);
        int bb = std::min(rl, (int)std::ceil(ring_coord(tb, nside)) + 1);
        s.ring_lo = a - rf;
        s.nring = bb - a + 1;
        kmax = std::max(kmax, s.nring);
        s.yi = (uint32_t)(long long)std::llrint((s.lat - rg.lat_lo) * sy);
        const double cc = std::cos(s.lat), sc = std::sin(s.lat);
        s.c0 = (float)(cc * cc); s.c1 = (float)(-cc * sc);
        s.c2 = (float)(-0.5 * cc * cc); s.c3 = (float)(cc * sc / 6.0);
        s.du_f = (float)s.du;
        s.pad_ = 0;
        if (strip_cells > 1) cw = std::min(cw, std::fabs(s.du) * cc);
    }
    c->kmax = kmax;
    c->nstrip = (int32_t)hs.size();
    c->strip_cells = strip_cells;
    c->cell_width_sky = strip_cells > 1 ? cw : 0.0;
    // small-angle series of the fp32 pair arithmetic: valid while R and the widest
    // longitude half-window stay below 0.05 rad (dropped x^6/360 term < 2e-8 relative)
    c->small_series_ok = !pole && R <= 0.05 && dlmax <= 0.05;
    // The fp32 pair arithmetic itself delivers 4 sin^2(d/2) to ~4 ulp (2.4e-7 relative), i.e. d to 1.2e-7 relative:
    // it settles "d <= R" to better than the 1e-9 rad the count parity allows (reading c4) only while
    // R <= 0.004 rad (0.23 deg; the paper's five workloads have R <= 0.0013 rad).  Wider kernels take the fp64
    // pair arithmetic (series form where valid) with the accumulation of the chosen mode.
    c->f32_series_ok = c->small_series_ok && R <= kF32RadiusMax;

    HCG_CUDA(c, c->d_strips.ensure(st.size() * sizeof(Strip)));
    HCG_CUDA(c, cudaMemcpy(c->d_strips.p, st.data(), st.size() * sizeof(Strip), cudaMemcpyHostToDevice));
    const size_t nw = st.size() * (size_t)kmax;
    HCG_CUDA(c, c->d_wins.ensure(nw * sizeof(RingWin)));
    HCG_CUDA(c, c->d_winsf.ensure(nw * sizeof(RingWinF)));
    std::vector<RowF> rows(st.size());
    for (size_t i = 0; i < st.size(); ++i) {
        RowF& r = rows[i];
        r.yi = st[i].yi; r.ring_lo = st[i].ring_lo; r.nring = st[i].nring;
        r.cc = (float)std::cos(st[i].lat); r.sc = (float)std::sin(st[i].lat);
        r.pad_[0] = r.pad_[1] = r.pad_[2] = 0;
    }
    HCG_CUDA(c, c->d_rowsf.ensure(rows.size() * sizeof(RowF)));
    HCG_CUDA(c, cudaMemcpy(c->d_rowsf.p, rows.data(), rows.size() * sizeof(RowF), cudaMemcpyHostToDevice));
    c->dlmax = dlmax;
    c->car_u0 = st[0].u0; c->car_du = st[0].du;
    // the tile kernel walks a plate-carree target whose region is a plain longitude window
    // (no wrap) with a per-ring table narrow enough for fp32 bin arithmetic
    c->tile_ok = strip_cells > 1 && !rg.full_circle && c->f32_series_ok && rg.m < (1 << 22);
    const int threads = 128;
    const unsigned blocks = (unsigned)((nw + threads - 1) / threads);
    ring_window_kernel<<<blocks, threads>>>(c->d_strips.as<Strip>(), c->d_wins.as<RingWin>(),
                                            c->d_winsf.as<RingWinF>(), (int)st.size(), kmax, rg, R);
    HCG_CUDA(c, cudaGetLastError());
    HCG_CUDA(c, cudaDeviceSynchronize());
    c->has_target = true;
    return HCGRID_OK;
}

int build_target_car(hcgrid_ctx* c, int nx, int ny, double lon0, double lat0, double dlon, double dlat) {
    std::vector<HostStrip> hs((size_t)ny);
    for (int iy = 0; iy < ny; ++iy) {
        volatile double prod = (double)iy * dlat;     // one rounding per operation, no FMA
        volatile double la = lat0 + prod;
        if (la > 90.0 || la < -90.0)
            return fail(c, HCGRID_ERR_INVALID_ARG, "target row %d has latitude %.17g outside [-90, 90]", iy, (double)la);
        hs[(size_t)iy] = HostStrip{lon0, dlon, la};
    }
    volatile double span = (double)(nx - 1) * dlon;
    const double a = lon0 * kDeg2Rad, b = (lon0 + span) * kDeg2Rad;
    c->is_car = true;
    c->ncell = (int64_t)nx * ny;
    c->car_dlat = dlat * kDeg2Rad;
    c->car_nx = nx; c->car_ny = ny;
    c->car_lon0_deg = lon0; c->car_lat0_deg = lat0; c->car_dlon_deg = dlon; c->car_dlat_deg = dlat;
    return finish_target(c, hs, nx, std::min(a, b), std::max(a, b));
}

// Step of an arithmetic progression v[0], v[stride], ..., v[(n - 1) stride] in the plate-carree convention
// v0 + k * d (one rounding per operation): tried are the first difference, the mean difference and their
// neighbours within two units in the last place.  tol = 0: every term must match bit for bit.
static bool find_step(const double* v, int64_t n, int64_t stride, double tol, double& d_out) {
    if (n < 2) return false;
    const double v0 = v[0];
    const double base[2] = {v[stride] - v0, (v[(n - 1) * stride] - v0) / (double)(n - 1)};
    for (int b = 0; b < 2; ++b)
        for (int k = -2; k <= 2; ++k) {
            double d = base[b];
            for (int s = 0; s < std::abs(k); ++s) d = std::nextafter(d, k > 0 ? HUGE_VAL : -HUGE_VAL);
            if (d == 0.0 || !std::isfinite(d)) continue;
            bool ok = true;
            for (int64_t i = 0; i < n && ok; ++i) {
                volatile double prod = (double)i * d;
                volatile double x = v0 + prod;
                ok = tol == 0.0 ? x == v[i * stride] : std::fabs(x - v[i * stride]) <= tol;
            }
            if (ok) { d_out = d; return true; }
        }
    return false;
}

// Per-cell targets that are a plate-carree grid listed row by row (what a WCS CAR header expands to) are recognised
// and take the plate-carree path with its tile kernels.  fp64 mode: only if lon0 + ix * dlon, lat0 + iy * dlat
// reproduce every given centre bit for bit (the results are then those of the general path on the same centres);
// fp32 mode: to 1e-10 deg (1.7e-12 rad: far inside the 1e-9 rad of the count bar and 1e-7 of the fp32 tolerance).
static bool detect_car(const std::vector<double>& hl, const std::vector<double>& hb, bool exact, int& nx, int& ny,
                       double& dlon, double& dlat) {
    const int64_t ncell = (int64_t)hl.size();
    const double tol = exact ? 0.0 : 1e-10;
    int64_t w = 1;
    while (w < ncell && (exact ? hb[(size_t)w] == hb[0] : std::fabs(hb[(size_t)w] - hb[0]) <= tol)) ++w;
    if (w < 2 || ncell % w != 0 || w > (1 << 30) || ncell / w > (1 << 30)) return false;
    const int64_t h = ncell / w;
    if (!find_step(hl.data(), w, 1, tol, dlon)) return false;
    dlat = 1.0;                                               // a single row: any non-zero step
    if (h > 1 && !find_step(hb.data(), h, w, tol, dlat)) return false;
    if (std::fabs(dlon) * (double)(w - 1) >= 360.0) return false;
    for (int64_t iy = 0; iy < h; ++iy) {
        const double lat_row = hb[(size_t)(iy * w)];
        for (int64_t ix = 0; ix < w; ++ix) {
            const double l = hl[(size_t)(iy * w + ix)], b = hb[(size_t)(iy * w + ix)];
            if (exact ? (l != hl[(size_t)ix] || b != lat_row)
                      : (std::fabs(l - hl[(size_t)ix]) > tol || std::fabs(b - lat_row) > tol))
                return false;
        }
    }
    nx = (int)w; ny = (int)h;
    return true;
}

int refine_target_for_density(hcgrid_ctx* c, int64_t n, cudaStream_t st, bool* rebuilt) {
    *rebuilt = false;
    const Region& rg = c->region;
    if (!c->is_car || c->opt_subpix > -100 || rg.subpix >= 6 || n <= 10 * rg.nbins) return HCGRID_OK;
    // finer bins double the table per bit: as many bits as bring the density down to 4 samples per bin -- or as many
    // as there are -- while the per-ring table stays narrow enough for the tile kernels' fp32 bin arithmetic and the
    // whole table modest; pointless if even that leaves more than 10 per bin (the radix path does not care about bins)
    int b = rg.subpix;
    int64_t nbins = rg.nbins, m = rg.m;
    while (b < 6 && n > 4 * nbins && 2 * m < ((int64_t)1 << 22) && 2 * nbins <= ((int64_t)1 << 25)) { ++b; nbins *= 2; m *= 2; }
    if (b == rg.subpix || n > 10 * nbins) return HCGRID_OK;
    HCG_CUDA(c, cudaStreamSynchronize(st));                            // earlier calls may still read the tables
    const int keep = c->subpix_refined;
    c->subpix_refined = b;
    const int rc = build_target_car(c, c->car_nx, c->car_ny, c->car_lon0_deg, c->car_lat0_deg, c->car_dlon_deg,
                                    c->car_dlat_deg);
    if (rc != HCGRID_OK) { c->subpix_refined = keep; return rc; }
    *rebuilt = true;
    return HCGRID_OK;
}

int build_target_cells(hcgrid_ctx* c, int64_t ncell, const double* lon, const double* lat, cudaStream_t st) {
    std::vector<double> hl((size_t)ncell), hb((size_t)ncell);
    HCG_CUDA(c, cudaMemcpyAsync(hl.data(), lon, sizeof(double) * (size_t)ncell, cudaMemcpyDeviceToHost, st));
    HCG_CUDA(c, cudaMemcpyAsync(hb.data(), lat, sizeof(double) * (size_t)ncell, cudaMemcpyDeviceToHost, st));
    HCG_CUDA(c, cudaStreamSynchronize(st));
    {
        int nx = 0, ny = 0;
        double dlon = 0.0, dlat = 0.0;
        bool valid = true;
        for (int64_t i = 0; i < ncell && valid; ++i)
            valid = hb[(size_t)i] >= -90.0 && hb[(size_t)i] <= 90.0 && std::isfinite(hl[(size_t)i]);
        if (valid && c->opt_cells_as_grid && detect_car(hl, hb, c->precision == HCGRID_F64, nx, ny, dlon, dlat))
            return build_target_car(c, nx, ny, hl[0], hb[0], dlon, dlat);
    }
    std::vector<HostStrip> hs((size_t)ncell);
    double sx = 0, sy = 0;
    for (int64_t i = 0; i < ncell; ++i) {
        if (!(hb[(size_t)i] >= -90.0 && hb[(size_t)i] <= 90.0) || !std::isfinite(hl[(size_t)i]))
            return fail(c, HCGRID_ERR_INVALID_ARG, "target cell %lld has invalid coordinates", (long long)i);
        hs[(size_t)i] = HostStrip{hl[(size_t)i], 0.0, hb[(size_t)i]};
        sx += std::cos(hl[(size_t)i] * kDeg2Rad); sy += std::sin(hl[(size_t)i] * kDeg2Rad);
    }
    // longitude extent about the circular mean of the cells
    const double lm = std::atan2(sy, sx);
    double dmin = 0, dmax = 0;
    for (int64_t i = 0; i < ncell; ++i) {
        const double d = wrap_pm_pi(hl[(size_t)i] * kDeg2Rad - lm);
        dmin = std::min(dmin, d); dmax = std::max(dmax, d);
    }
    c->is_car = false;
    c->ncell = ncell;
    c->car_dlat = 0.0;
    return finish_target(c, hs, 1, lm + dmin, lm + dmax);
}

}  // namespace hcg
