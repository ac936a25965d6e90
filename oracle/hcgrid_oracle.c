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

int hcgrid_oracle_grid(double sigma_deg, double radius_deg,
                       int64_t ncell, const double* cell_lon, const double* cell_lat,
                       int64_t n, const double* lon, const double* lat,
                       const float* values, int32_t nchan, const float* weights,
                       double* datacube, double* weightmap, int64_t* counts,
                       double* absmap, int64_t* near_boundary, int nthreads)
{
    if (!(sigma_deg > 0.0) || !(radius_deg > 0.0) || ncell < 0 || n < 0 || nchan < 1)
        return -1;
    if (!datacube || !weightmap) return -1;
    if (ncell > 0 && (!cell_lon || !cell_lat)) return -1;
    if (n > 0 && (!lon || !lat || !values)) return -1;

    const double sigma = sigma_deg * DEG2RAD;
    const double R = radius_deg * DEG2RAD;
    const double inv2s2 = 1.0 / (2.0 * sigma * sigma);
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
            long double W = 0.0L;
            int64_t cnt = 0, nb = 0;
            for (int k = 0; k < nchan; ++k) { S[k] = 0.0L; A[k] = 0.0L; }
            const double clon = cell_lon[c], clat = cell_lat[c];
            for (int64_t s = 0; s < n; ++s) {
                if (fabs(lat[s] - clat) > dlat_cut_deg) continue;
                const double d = hcgrid_oracle_distance(clon, clat, lon[s], lat[s]);
                if (fabs(d - R) < 1e-9) nb++;
                if (d <= R) {
                    const double w = exp(-d * d * inv2s2);
                    const double q = weights ? (double)weights[s] : 1.0;
                    const double qw = q * w;
                    W += (long double)qw;
                    cnt++;
                    const float* v = values + (size_t)s * (size_t)nchan;
                    for (int k = 0; k < nchan; ++k) {
                        const double vk = (double)v[k];
                        S[k] += (long double)(qw * vk);
                        A[k] += (long double)(qw * fabs(vk));
                    }
                }
            }
            weightmap[c] = (double)W;
            if (counts) counts[c] = cnt;
            if (near_boundary) near_boundary[c] = nb;
            for (int k = 0; k < nchan; ++k) {
                size_t o = (size_t)c * (size_t)nchan + (size_t)k;
                if (W > 0.0L) {
                    datacube[o] = (double)(S[k] / W);
                    if (absmap) absmap[o] = (double)(A[k] / W);
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
