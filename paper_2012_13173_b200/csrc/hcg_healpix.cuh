// hcg_healpix.cuh -- HEALPix RING-scheme geometry used by the pre-ordering (a2) and the
// target set-up (a1).  Written from the published definition of the pixelisation
// (Gorski et al. 2005, the reference of PAPER.md:96-98); the paper calls the HEALPix C++
// library for this on the CPU, here it is device code.
//
// Rings are numbered 1 .. 4*nside-1 from the north pole.  Ring i has
//   north cap  (i <  nside):        4 i pixels, centre z = 1 - i^2 / (3 nside^2)
//   belt       (nside <= i <= 3n):  4 nside pixels, centre z = (2 nside - i) * 2 / (3 nside)
//   south cap  by mirror symmetry (i' = 4 nside - i).
// Two containment facts the gather relies on (tests/test_library_cpu.py checks both):
//   (1) a point assigned to pixel j of ring r satisfies j <= g_r(lon) <= j+1 with
//       g_r(lon) = lon * npix_ring(r) / (2 pi) + off_r   (off_r = 1/2 on belt rings whose
//       pixel centres sit at multiples of the pixel width, else 0);
//   (2) its z lies between the centre z of ring r+1 and of ring r-1.
#pragma once
#include <cstdint>
#include <cmath>

#ifdef __CUDACC__
#define HCG_HD __host__ __device__ __forceinline__
#else
#define HCG_HD inline
#endif

namespace hcg {

constexpr double kPi = 3.14159265358979323846;
constexpr double kTwoPi = 6.28318530717958647692;
constexpr double kHalfPi = 1.57079632679489661923;
constexpr double kDeg2Rad = kPi / 180.0;
constexpr double kSqrt6 = 2.44948974278317809820;
constexpr double kInvTwoPi = 0.15915494309189533577;
constexpr double kInvHalfPi = 0.63661977236758134308;

// pixels in ring `iring` (1 .. 4 nside - 1)
HCG_HD int ring_npix(int iring, int nside) {
    int i = iring < 4 * nside - iring ? iring : 4 * nside - iring;
    return 4 * (i < nside ? i : nside);
}

// offset of the in-ring coordinate g_r(lon) = lon * npix / 2pi + off
HCG_HD double ring_off(int iring, int nside) {
    if (iring < nside || iring > 3 * nside) return 0.0;
    return ((iring - nside + 1) & 1) ? 0.0 : 0.5;
}

// index of the first pixel of ring `iring`
HCG_HD int64_t ring_first_pixel(int iring, int64_t nside) {
    const int64_t ncap = 2 * nside * (nside - 1);
    if (iring < nside) return 2 * (int64_t)iring * (iring - 1);
    if (iring <= 3 * nside) return ncap + (int64_t)(iring - nside) * 4 * nside;
    const int64_t ip = 4 * nside - iring;
    return 12 * nside * nside - 2 * ip * (ip + 1);
}

// colatitude (rad) of the centre of ring `iring`; iring = 0 -> 0 (north pole),
// iring = 4 nside -> pi (south pole).  Caps use 1 - z = 2 sin^2(theta/2) (no cancellation).
HCG_HD double ring_colat(int iring, int nside) {
    const double n = (double)nside;
    if (iring <= 0) return 0.0;
    if (iring >= 4 * nside) return kPi;
    if (iring < nside) return 2.0 * asin((double)iring / (n * kSqrt6));
    if (iring <= 3 * nside) return acos((2.0 * n - (double)iring) * 2.0 / (3.0 * n));
    return kPi - 2.0 * asin((double)(4 * nside - iring) / (n * kSqrt6));
}

// continuous ring coordinate rho(theta): the real-valued inverse of ring_colat
// (rho(ring_colat(i)) = i).  Monotone increasing in theta.
HCG_HD double ring_coord(double colat, int nside) {
    const double n = (double)nside;
    if (colat <= 0.0) return 0.0;
    if (colat >= kPi) return 4.0 * n;
    const double z = cos(colat);
    if (z > 2.0 / 3.0) return n * kSqrt6 * sin(0.5 * colat);
    if (z >= -2.0 / 3.0) return 2.0 * n - 1.5 * n * z;
    return 4.0 * n - n * kSqrt6 * sin(0.5 * (kPi - colat));
}

// Point -> (ring number, pixel-in-ring).  lon in [0, 2pi), lat in [-pi/2, pi/2].
HCG_HD void ang2ring(int nside, double lon, double lat, int& iring, int& ip) {
    const double n = (double)nside;
    const double z = sin(lat);
    const double za = fabs(z);
    double tt = lon * kInvHalfPi;                  // [0, 4)
    if (tt >= 4.0) tt -= 4.0;
    if (tt < 0.0) tt = 0.0;
    if (za <= 2.0 / 3.0) {                         // equatorial belt
        const double t1 = n * (0.5 + tt);
        const double t2 = n * z * 0.75;
        // all of these are below 6 nside <= 49152 in magnitude: 32-bit integers throughout
        const int jp = (int)floor(t1 - t2);               // ascending edge line index
        const int jm = (int)floor(t1 + t2);               // descending edge line index
        const int ir = nside + 1 + jp - jm;               // in {1, 2n+1}
        const int kshift = 1 - (ir & 1);
        int p = (jp + jm - nside + kshift + 1) >> 1;      // in (-nside, 5 nside]
        if (p >= 4 * nside) p -= 4 * nside;
        if (p < 0) p += 4 * nside;
        iring = ir + nside - 1;
        ip = p;
    } else {                                       // polar caps
        const double tp = tt - floor(tt);
        const double sh = sin(0.5 * (kHalfPi - fabs(lat)));
        const double tmp = n * kSqrt6 * sh;     // n sqrt(3 (1 - |z|)), 1-|z| = 2 sin^2(colat/2)
        const int jp = (int)(tp * tmp);
        const int jm = (int)((1.0 - tp) * tmp);
        int ir = jp + jm + 1;                      // ring counted from the closest pole
        if (ir > nside) ir = nside;
        int p = (int)(tt * (double)ir);            // tt in [0, 4): p in [0, 4 ir]
        if (p >= 4 * ir) p -= 4 * ir;
        iring = z > 0 ? ir : 4 * nside - ir;
        ip = p;
    }
}

// Lookup-bin index along ring `iring` of a point with pixel-in-ring `ip` and longitude
// lon: 2^b bins per pixel for b >= 0 (sub-pixel refinement of the per-pixel table),
// 2^-b pixels per bin for b < 0.  Monotone in lon within the ring and consistent with ip.
HCG_HD long long ring_bin(int iring, int nside, int ip, double lon, int b) {
    if (b <= 0) return (long long)(ip >> (-b));
    const int npr = ring_npix(iring, nside);
    const double g = lon * ((double)npr * kInvTwoPi) + ring_off(iring, nside);
    double d = g - (double)ip;
    if (d > 0.5 * npr) d -= npr;
    if (d < -0.5 * npr) d += npr;
    int sub = (int)floor(d * (double)(1 << b));
    if (sub < 0) sub = 0;
    if (sub > (1 << b) - 1) sub = (1 << b) - 1;
    return (long long)((ip << b) + sub);           // < 4 nside 2^b <= 2^21
}

// number of lookup bins along ring `iring`
HCG_HD long long ring_nbins(int iring, int nside, int b) {
    const int npr = ring_npix(iring, nside);
    return (long long)(b >= 0 ? (npr << b) : (((npr - 1) >> (-b)) + 1));
}

// bin coordinate (real) of longitude lon on ring iring: floor() of it is the bin of a
// point sitting at the ring's centre latitude
HCG_HD double ring_bin_coord(int iring, int nside, double lon, int b) {
    const int npr = ring_npix(iring, nside);
    const double g = lon * ((double)npr * kInvTwoPi) + ring_off(iring, nside);
    // g * 2^b, exact (the value ldexp(g, b) returns); |b| < 16
    return b >= 0 ? g * (double)(1 << b) : g * (1.0 / (double)(1 << (-b)));
}

}  // namespace hcg
