/* oracle_sanitize_driver.c -- TEST INFRASTRUCTURE.
 *
 * Exercises oracle/hcgrid_oracle.c under AddressSanitizer + UndefinedBehaviorSanitizer
 * (tests/test_oracle_sanitizers.py builds this file together with the oracle source with
 * -fsanitize=address,undefined -fno-sanitize-recover=all and runs it).  Outputs are allocated
 * with exactly the sizes hcgrid_oracle.h states, so a write one element past any of them, a read
 * past an input, a signed overflow in an index or a misaligned access ends the program non-zero.
 *
 * Cases: a ragged problem (7 x 5 cells, 211 samples, 3 channels, per-sample weights), every
 * optional output NULL, one sample / one cell, no samples, no cells, samples at the poles and
 * on the +-180 seam, non-finite values, both kernel types of hcgrid_oracle_grid_kernel.
 */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

#include "hcgrid_oracle.h"

static uint64_t lcg_state = 0x9e3779b97f4a7c15ull;
static double lcg(void) {
    lcg_state = lcg_state * 6364136223846793005ull + 1442695040888963407ull;
    return (double)(lcg_state >> 11) / 9007199254740992.0;
}

#define CHECK(c) do { if (!(c)) { fprintf(stderr, "driver check failed: %s (line %d)\n", #c, __LINE__); exit(3); } } while (0)

static void run(int ktype, int64_t nx, int64_t ny, int64_t n, int32_t nchan, int with_weights, int with_optional,
                double lon0, double lat0, double step, int nonfinite) {
    int64_t ncell = nx * ny;
    /* exact-size allocations (malloc(0) is avoided: one byte, never touched) */
    double* cl = malloc(ncell ? (size_t)ncell * sizeof(double) : 1);
    double* cb = malloc(ncell ? (size_t)ncell * sizeof(double) : 1);
    double* lon = malloc(n ? (size_t)n * sizeof(double) : 1);
    double* lat = malloc(n ? (size_t)n * sizeof(double) : 1);
    float* val = malloc(n ? (size_t)n * nchan * sizeof(float) : 1);
    float* q = with_weights ? malloc(n ? (size_t)n * sizeof(float) : 1) : NULL;
    double* cube = malloc(ncell ? (size_t)ncell * nchan * sizeof(double) : 1);
    double* wmap = malloc(ncell ? (size_t)ncell * sizeof(double) : 1);
    int64_t* cnt = with_optional ? malloc(ncell ? (size_t)ncell * sizeof(int64_t) : 1) : NULL;
    double* absm = with_optional ? malloc(ncell ? (size_t)ncell * nchan * sizeof(double) : 1) : NULL;
    double* absw = with_optional ? malloc(ncell ? (size_t)ncell * sizeof(double) : 1) : NULL;
    int64_t* nearb = with_optional ? malloc(ncell ? (size_t)ncell * sizeof(int64_t) : 1) : NULL;
    for (int64_t j = 0; j < ny; j++)
        for (int64_t i = 0; i < nx; i++) {
            cl[j * nx + i] = lon0 + step * (double)i;
            cb[j * nx + i] = lat0 + step * (double)j;
        }
    for (int64_t s = 0; s < n; s++) {
        lon[s] = lon0 - step + lcg() * step * (double)(nx + 1);
        lat[s] = lat0 - step + lcg() * step * (double)(ny + 1);
        if (lat[s] > 90.0) lat[s] = 90.0;
        if (lat[s] < -90.0) lat[s] = -90.0;
        if (lon[s] > 180.0) lon[s] -= 360.0;
        for (int32_t c = 0; c < nchan; c++) val[s * nchan + c] = (float)(lcg() - 0.5);
        if (q) q[s] = (float)(0.25 + lcg());
    }
    if (nonfinite && n > 2) {
        val[0] = NAN;
        val[(size_t)nchan] = INFINITY;
    }
    double sigma = step * 0.8, radius = 3.0 * sigma;
    int rc;
    if (ktype < 0)
        rc = hcgrid_oracle_grid(sigma, radius, ncell, cl, cb, n, lon, lat, val, nchan, q, cube, wmap, cnt, absm, nearb,
                                (n & 1) ? 1 : 3);
    else
        rc = hcgrid_oracle_grid_kernel(ktype, 2.52, 1.55, sigma, radius, ncell, cl, cb, n, lon, lat, val, nchan, q, cube,
                                       wmap, cnt, absm, absw, nearb, 2);
    CHECK(rc == 0);
    CHECK(hcgrid_oracle_last_threads() >= 1);
    for (int64_t c = 0; c < ncell; c++) {
        if (cnt) CHECK(cnt[c] >= 0 && cnt[c] <= n);
        if (ktype <= 0 && !nonfinite) CHECK(wmap[c] >= 0.0);
        if (cnt && cnt[c] == 0) CHECK(wmap[c] == 0.0 && isnan(cube[c * nchan]));
    }
    free(cl); free(cb); free(lon); free(lat); free(val); free(q);
    free(cube); free(wmap); free(cnt); free(absm); free(absw); free(nearb);
}

int main(void) {
    for (int ktype = -1; ktype <= 1; ktype++) {
        run(ktype, 7, 5, 211, 3, 1, 1, 30.0, 41.0, 0.05, 0);     /* ragged, weights, all outputs */
        run(ktype, 7, 5, 211, 3, 0, 0, 30.0, 41.0, 0.05, 0);     /* optional outputs NULL */
        run(ktype, 1, 1, 1, 1, 0, 1, 0.0, 0.0, 0.01, 0);         /* one cell, one sample */
        run(ktype, 4, 3, 0, 2, 1, 1, 10.0, -5.0, 0.1, 0);        /* no samples */
        run(ktype, 0, 0, 17, 2, 0, 1, 10.0, -5.0, 0.1, 0);       /* no cells */
        run(ktype, 6, 6, 300, 2, 1, 1, 179.8, 89.75, 0.05, 0);   /* pole and +-180 seam */
        run(ktype, 6, 6, 300, 2, 0, 1, -180.0, -90.0, 0.05, 0);  /* south pole, west seam */
        run(ktype, 5, 4, 97, 4, 1, 1, 30.0, 41.0, 0.05, 1);      /* NaN and Inf values */
    }
    /* invalid arguments are refused, not dereferenced */
    double d = 0.0;
    CHECK(hcgrid_oracle_grid(-1.0, 1.0, 1, &d, &d, 0, NULL, NULL, NULL, 1, NULL, &d, &d, NULL, NULL, NULL, 1) == -1);
    CHECK(hcgrid_oracle_grid(1.0, 1.0, 1, &d, &d, 0, NULL, NULL, NULL, 0, NULL, &d, &d, NULL, NULL, NULL, 1) == -1);
    CHECK(fabs(hcgrid_oracle_distance(0.0, 0.0, 90.0, 0.0) - 1.5707963267948966) < 1e-15);
    puts("oracle sanitizer driver: ok");
    return 0;
}
