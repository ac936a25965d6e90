/* hcgrid_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, brute-force fp64 CPU gridder written from the paper's definition
 * (arXiv 2012.13173, Sect. 2.1, Eq. 1):
 *
 *     V[g_ij] = (1 / W_ij) * sum_n V[s_n] * w(alpha_ij, delta_ij; alpha_n, delta_n)
 *     W_ij    = sum_n w(alpha_ij, delta_ij; alpha_n, delta_n)
 *
 * with the kernel of PAPER.md:186 (Sect. 3.6 iii): a radially symmetric Gaussian
 * of standard deviation sigma_kernel, truncated at "sphere_radius".
 *
 * Every (cell, sample) pair is tested.  There is no HEALPix, no sort, no lookup
 * table here, and this directory shares no code with paper_2012_13173_b200/.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may call it.
 *
 * Readings of the paper taken here:
 *   c1  w(d) = exp(-d^2 / (2 sigma^2)), peak 1, no 1/(2 pi sigma^2) factor.
 *   c3  d is the true great-circle angle (haversine form).
 *   c4  a pair contributes iff d <= R.
 *   c5  W == 0  ->  V = NaN, W = 0, count = 0.
 *   c6  optional per-sample weight q_s multiplies the kernel; count ignores q.
 *   c7  multi-channel: Eq. 1 per channel with the same w and the same W.
 *
 * Pins: tests/test_oracle_pins.py (hand case tests/golden/hand_3x3.txt, single
 * sample closed form, constant field, permutation, rotation about the pole
 * axis, closed-form distances, independent vector-formula brute force; for the
 * elliptical Gaussian: equality with the circular one at ka = 1, closed forms
 * along the meridian and the equator, PA + 90 deg swapping the axes, an
 * independent tangent-vector brute force, constant field).
 */
#ifndef HCGRID_ORACLE_H
#define HCGRID_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Great-circle angle in radians between (lon1,lat1) and (lon2,lat2), all in
 * degrees.  Differences are formed in degrees first (exact for nearby
 * doubles), then converted; d = 2 asin(sqrt(hav)).  The gridder below calls
 * exactly this function for every pair it does not early-out. */
double hcgrid_oracle_distance(double lon1_deg, double lat1_deg,
                              double lon2_deg, double lat2_deg);

/* Brute-force gridding.  All pointers are HOST pointers owned by the caller.
 *   cell_lon/lat [ncell]   target cell centres, degrees
 *   lon/lat      [n]       sample positions, degrees
 *   values       [n][nchan] float32, channel fastest
 *   weights      [n] float32 or NULL (q_s = 1)
 * Outputs (any may be NULL except datacube and weightmap):
 *   datacube     [ncell][nchan]  sum_s q w v / W     (NaN where W == 0)
 *   weightmap    [ncell]         W = sum_s q w
 *   counts       [ncell]         number of samples with d <= R (geometric)
 *   absmap       [ncell][nchan]  sum_s q w |v| / W   (tolerance scale, c16)
 *   near_boundary[ncell]         number of samples with |d - R| < 1e-9 rad
 * nthreads <= 0 means "all cores".  Returns 0, or -1 on invalid arguments. */
int hcgrid_oracle_grid(double sigma_deg, double radius_deg,
                       int64_t ncell, const double* cell_lon, const double* cell_lat,
                       int64_t n, const double* lon, const double* lat,
                       const float* values, int32_t nchan, const float* weights,
                       double* datacube, double* weightmap, int64_t* counts,
                       double* absmap, int64_t* near_boundary, int nthreads);

/* The same loop with the kernel function chosen by ktype:
 *   0  Gaussian exp(-d^2 / (2 sigma^2)) (ka, kb ignored) -- identical to hcgrid_oracle_grid;
 *   1  tapered sinc: sinc(d / (kb sigma)) * exp(-(d / (ka sigma))^2), sinc(x) = sin(pi x) / (pi x)
 *      (PAPER.md:186 names the sinc as the optimal kernel and finite-length functions as what
 *      is used in practice; the tapered form is that of the work it follows, Winkel et al. 2016b).
 *   2  elliptical Gaussian exp(-u^2 / (2 s1^2) - v^2 / (2 s2^2)) (reading c17): s1 = sigma_deg is the
 *      standard deviation along the axis at position angle kb (degrees, from north through east), s2 = ka * s1
 *      (ka > 0; ka < 1 makes the axis at the position angle the major one) the one across it;
 *      (u, v) = d (cos(beta - PA), sin(beta - PA)) with d the great-circle angle and beta the bearing of the
 *      sample from the cell centre; the support stays the circle d <= R (reading c4).  ka = 1 gives ktype 0 bit
 *      for bit.
 * Signed weights change two outputs: datacube = S / W wherever W != 0 (NaN otherwise), and
 * absmap = sum |q w| |v| / |W|.  abswmap[ncell] (may be NULL) = sum |q w|, the scale against
 * which W itself is to be compared (W can cancel to ~0).  Returns 0, or -1 on invalid arguments. */
int hcgrid_oracle_grid_kernel(int ktype, double ka, double kb, double sigma_deg, double radius_deg,
                              int64_t ncell, const double* cell_lon, const double* cell_lat,
                              int64_t n, const double* lon, const double* lat,
                              const float* values, int32_t nchan, const float* weights,
                              double* datacube, double* weightmap, int64_t* counts,
                              double* absmap, double* abswmap, int64_t* near_boundary, int nthreads);

/* Number of OpenMP threads the last hcgrid_oracle_grid call used. */
int hcgrid_oracle_last_threads(void);

#ifdef __cplusplus
}
#endif
#endif
