/* hcgrid_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.  See hcgrid_oracle.h.
 *
 * The definition written out (Eq. 1; PAPER.md:186 kernel):
 * for every cell c and every sample s, in input order,
 *     d   = great-circle angle between cell centre and sample
 *     if d <= R:  w = exp(-d^2 / (2 sigma^2));  W_c += q_s w;  S_ck += q_s w v_sk
 * and V_ck = S_ck / W_c.  fp64 arithmetic per pair, long double (x87 80-bit)
 * accumulators so the oracle's own summation error (~1e-19 n) is irrelevant at
 * the 1e-12 tier.  No blocking, no spatial index, no reordering.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC (no -ffast-math).
 */
#include "hcgrid_oracle.h"

#include <math.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define DEG2RAD (3.14159265358979323846 / 180.0)

static int g_last_threads = 1;

double hcgrid_oracle_distance(double lon1_deg, double lat1_deg,
                              double lon2_deg, double lat2_deg)
{
    /* differences in degrees first (SURVEY 8c "fp64 pin"), then radians */
    double dlat = (lat2_deg - lat1_deg) * DEG2RAD;
    double dlon = remainder(lon2_deg - lon1_deg, 360.0) * DEG2RAD; /* [-pi, pi] */
    double c1 = cos(lat1_deg * DEG2RAD);
    double c2 = cos(lat2_deg * DEG2RAD);
    double sa = sin(0.5 * dlat);
    double sb = sin(0.5 * dlon);
    double hav = sa * sa + c1 * c2 * sb * sb;          /* haversine of d */
    if (hav > 1.0) hav = 1.0;
    return 2.0 * asin(sqrt(hav));
}

int hcgrid_oracle_last_threads(void) { return g_last_threads; }

/* Kernel weight as a function of the great-circle angle d (rad).
 *   ktype 0: Gaussian exp(-d^2 / (2 sigma^2))                       (the default)
 *   ktype 1: tapered sinc  sinc(d / (b sigma)) exp(-(d / (a sigma))^2),  sinc(x) = sin(pi x)/(pi x)
 *            -- the finite-length stand-in for the "sinc function with infinite length" of
 *            PAPER.md:186, in the form of the work the paper follows for its kernel set-up
 *            (Winkel et al. 2016b); may be negative. */
static double kernel_weight(int ktype, double d, double sigma, double ka, double kb)
{
    if (ktype == 0) return exp(-d * d / (2.0 * sigma * sigma));
    const double x = d / sigma;
    const double y = 3.14159265358979323846 * x / kb;
    const double sinc = y == 0.0 ? 1.0 : sin(y) / y;
    return sinc * exp(-(x / ka) * (x / ka));
}

/* ktype 2: elliptical Gaussian (reading c17; PAPER.md:186 only names the radially symmetric Gaussian
 * as the default and follows Winkel et al. 2016b, whose kernel set has a two-dimensional Gaussian).
 * Polar coordinates of the sample about the cell centre: the great-circle angle d and the bearing beta of the
 * sample as seen from the cell, measured from north through east (the azimuthal equidistant offsets are
 * xi = d sin beta towards east, eta = d cos beta towards north).  With phi = beta - PA the angle from the major
 * axis, u = d cos phi along it and v = d sin phi across it,
 *     w = exp(-u^2 / (2 smaj^2) - v^2 / (2 smin^2))
 *       = exp(-( d^2 / (2 smaj^2) + d^2 sin^2(phi) (1 / (2 smin^2) - 1 / (2 smaj^2)) )),
 * written in the second form so that smin == smaj gives the circular kernel's expression exactly.
 * The bearing comes from the components of the sample's direction along the cell's east and north unit
 * vectors, x = cos(lat_s) sin(dlon) and y = cos(lat_c) sin(lat_s) - sin(lat_c) cos(lat_s) cos(dlon), the latter
 * rewritten as sin(dlat) + 2 sin(lat_c) cos(lat_s) sin^2(dlon / 2) (the same identity that turns the cosine rule
 * into the haversine form) so that it keeps its accuracy for near pairs; differences are formed in degrees first,
 * like hcgrid_oracle_distance. */
static double bearing(double lon_c_deg, double lat_c_deg, double lon_s_deg, double lat_s_deg)
{
    const double dlat = (lat_s_deg - lat_c_deg) * DEG2RAD;
    const double dlon = remainder(lon_s_deg - lon_c_deg, 360.0) * DEG2RAD;
    const double sb = sin(0.5 * dlon);
    const double x = cos(lat_s_deg * DEG2RAD) * sin(dlon);
    const double y = sin(dlat) + 2.0 * sin(lat_c_deg * DEG2RAD) * cos(lat_s_deg * DEG2RAD) * sb * sb;
    return atan2(x, y);      /* from north (y) through east (x); 0 for a coincident pair */
}

static double elliptical_weight(double d, double beta, double inv2s2_maj, double inv2s2_min, double pa)
{
    const double sphi = sin(beta - pa);
    return exp(-(d * d * inv2s2_maj + d * d * sphi * sphi * (inv2s2_min - inv2s2_maj)));
}

static int grid_core(int ktype, double ka, double kb, double sigma_deg, double radius_deg,
                     int64_t ncell, const double* cell_lon, const double* cell_lat,
                     int64_t n, const double* lon, const double* lat,
                     const float* values, int32_t nchan, const float* weights,
                     double* datacube, double* weightmap, int64_t* counts,
                     double* absmap, double* abswmap, int64_t* near_boundary, int nthreads)
{
    if (!(sigma_deg > 0.0) || !(radius_deg > 0.0) || ncell < 0 || n < 0 || nchan < 1)
        return -1;
    if (!datacube || !weightmap) return -1;
    if (ncell > 0 && (!cell_lon || !cell_lat)) return -1;
    if (n > 0 && (!lon || !lat || !values)) return -1;

    const double sigma = sigma_deg * DEG2RAD;
    const double R = radius_deg * DEG2RAD;
    const double inv2s2 = 1.0 / (2.0 * sigma * sigma);
    /* ktype 2: sigma is the standard deviation along the axis at position angle kb (degrees), ka * sigma the one
     * across it (ka < 1: the axis at the position angle is the major one) */
    const double sigma_min = sigma * ka;
    const double inv2s2_min = ktype == 2 ? 1.0 / (2.0 * sigma_min * sigma_min) : inv2s2;
    const double pa = kb * DEG2RAD;
    /* exact early-out: d >= |dlat| always, so |dlat| > R(1+1e-12) cannot
     * contribute (and cannot be within 1e-9 of R unless R itself is ~1e3) */
    const double dlat_cut_deg = (R * (1.0 + 1e-12) + 1e-9) / DEG2RAD;

#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#else
    nthreads = 1;
#endif
    g_last_threads = nthreads;

    int failed = 0;
#pragma omp parallel num_threads(nthreads)
    {
        long double* S = (long double*)malloc(sizeof(long double) * (size_t)nchan);
        long double* A = (long double*)malloc(sizeof(long double) * (size_t)nchan);
        if (!S || !A) {
#pragma omp atomic write
            failed = 1;
        }
#pragma omp for schedule(dynamic, 16)
        for (int64_t c = 0; c < ncell; ++c) {
            if (!S || !A) continue;
            long double W = 0.0L, Wabs = 0.0L;
            int64_t cnt = 0, nb = 0;
            for (int k = 0; k < nchan; ++k) { S[k] = 0.0L; A[k] = 0.0L; }
            const double clon = cell_lon[c], clat = cell_lat[c];
            for (int64_t s = 0; s < n; ++s) {
                if (fabs(lat[s] - clat) > dlat_cut_deg) continue;
                const double d = hcgrid_oracle_distance(clon, clat, lon[s], lat[s]);
                if (fabs(d - R) < 1e-9) nb++;
                if (d <= R) {
                    const double w = ktype == 0 ? exp(-d * d * inv2s2)
                                   : ktype == 2 ? elliptical_weight(d, bearing(clon, clat, lon[s], lat[s]), inv2s2,
                                                                    inv2s2_min, pa)
                                                : kernel_weight(ktype, d, sigma, ka, kb);
                    const double q = weights ? (double)weights[s] : 1.0;
                    const double qw = q * w;
                    W += (long double)qw;
                    Wabs += (long double)fabs(qw);
                    cnt++;
                    const float* v = values + (size_t)s * (size_t)nchan;
                    for (int k = 0; k < nchan; ++k) {
                        const double vk = (double)v[k];
                        S[k] += (long double)(qw * vk);
                        A[k] += (long double)(fabs(qw) * fabs(vk));
                    }
                }
            }
            weightmap[c] = (double)W;
            if (abswmap) abswmap[c] = (double)Wabs;
            if (counts) counts[c] = cnt;
            if (near_boundary) near_boundary[c] = nb;
            /* Gaussians: W > 0 as soon as one sample contributes.  Signed kernels: W != 0. */
            const int defined = ktype != 1 ? (W > 0.0L) : (W != 0.0L);
            for (int k = 0; k < nchan; ++k) {
                size_t o = (size_t)c * (size_t)nchan + (size_t)k;
                if (defined) {
                    datacube[o] = (double)(S[k] / W);
                    /* tolerance scale: sum |q w| |v| over |W| (equals sum q w |v| / W for w >= 0) */
                    if (absmap) absmap[o] = (double)(A[k] / fabsl(W));
                } else {
                    datacube[o] = NAN;
                    if (absmap) absmap[o] = NAN;
                }
            }
        }
        free(S);
        free(A);
    }
    return failed ? -1 : 0;
}

int hcgrid_oracle_grid(double sigma_deg, double radius_deg,
                       int64_t ncell, const double* cell_lon, const double* cell_lat,
                       int64_t n, const double* lon, const double* lat,
                       const float* values, int32_t nchan, const float* weights,
                       double* datacube, double* weightmap, int64_t* counts,
                       double* absmap, int64_t* near_boundary, int nthreads)
{
    return grid_core(0, 0.0, 0.0, sigma_deg, radius_deg, ncell, cell_lon, cell_lat, n, lon, lat, values, nchan,
                     weights, datacube, weightmap, counts, absmap, NULL, near_boundary, nthreads);
}

int hcgrid_oracle_grid_kernel(int ktype, double ka, double kb, double sigma_deg, double radius_deg,
                              int64_t ncell, const double* cell_lon, const double* cell_lat,
                              int64_t n, const double* lon, const double* lat,
                              const float* values, int32_t nchan, const float* weights,
                              double* datacube, double* weightmap, int64_t* counts,
                              double* absmap, double* abswmap, int64_t* near_boundary, int nthreads)
{
    if (ktype != 0 && ktype != 1 && ktype != 2) return -1;
    if (ktype == 1 && (!(ka > 0.0) || !(kb > 0.0))) return -1;
    if (ktype == 2 && (!(ka > 0.0) || !(kb == kb))) return -1;
    return grid_core(ktype, ka, kb, sigma_deg, radius_deg, ncell, cell_lon, cell_lat, n, lon, lat, values, nchan,
                     weights, datacube, weightmap, counts, absmap, abswmap, near_boundary, nthreads);
}
