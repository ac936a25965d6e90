// convolve_gen.cu -- step a6, the general kernel: any channel count, fp32 or fp64 pair
// arithmetic, fp32 or fp64 accumulation (Sect. 3.4 i-v; Eq. 1).
//
// One warp owns one cell.  Phase 1: the 32 lanes evaluate 32 consecutive candidates of the
// cell's ring windows (distance test + kernel weight).  Phase 2 (nchan > 1): the accepted
// candidates of the batch are visited one by one and the whole warp reads that sample's
// spectrum row in place (values[idx][*], contiguous, coalesced) -- lane l owns channels
// 4l..4l+3 and 128+4l..128+4l+3 of a 256-channel tile -- so every channel has one register
// accumulator and Eq. 1's "same weight for all channels" costs one FMA per
// channel per accepted pair.  The spectra are never moved (a5: values stay in input order).
//
// fp64 pair arithmetic follows the definition with no shortcut: differences formed in
// degrees first, haversine, d = 2 asin(sqrt(hav)), w = exp(-d^2/(2 sigma^2)).
#include <algorithm>

#include "hcg_conv.cuh"

namespace hcg {

template <typename T> struct NanOf;
template <> struct NanOf<float> { static __device__ float v() { return __int_as_float(0x7fc00000); } };
template <> struct NanOf<double> { static __device__ double v() { return __longlong_as_double(0x7ff8000000000000LL); } };

template <typename T>
__device__ __forceinline__ T warp_sum(T x) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

// Tapered sinc (PAPER.md:186 names the sinc; form of Winkel et al. 2016b, the work the paper
// follows for its kernel set-up): sinc(d / (b sigma)) exp(-(d / (a sigma))^2), sinc(x) = sin(pi x)/(pi x).
__device__ __forceinline__ double tapered_sinc64(double d2, const KernelParams& kp) {
    const double y = sqrt(d2) * kp.pi_bs;
    const double sinc = y == 0.0 ? 1.0 : sin(y) / y;
    return sinc * exp(-d2 * kp.inv_a2s2);
}

// The same from the fp32 path's exponent: e2 = -t, t = d^2 log2e / (2 sigma^2) (what pair32
// hands to ex2 for the Gaussian).  sinf, not the approximate intrinsic: the argument reaches
// pi R / (b sigma) ~ 10 and the weight changes sign there.
__device__ __forceinline__ float tapered_sinc32(float e2, const KernelParams& kp) {
    const float t = fmaxf(-e2, 0.0f);
    const float y = kp.ts1 * sqrtf(t);
    const float sinc = y < 1e-4f ? 1.0f : sinf(y) / y;
    return sinc * ex2_approx(-t * kp.tg2);
}

// Elliptical Gaussian (reading c21).  x, y: components of the sample's direction along the cell's east
// and north unit vectors (x = cos(lat_s) sin(dlon), y = sin(dlat) + 2 sin(lat_c) cos(lat_s) sin^2(dlon / 2));
// sin(beta - PA) = (x cos PA - y sin PA) / hypot(x, y), beta the bearing from north through east.
__device__ __forceinline__ double elliptical64(double d2, double x, double y, const KernelParams& kp) {
    const double r2 = x * x + y * y;
    const double t = x * kp.ell_cp - y * kp.ell_sp;
    const double s2phi = r2 > 0.0 ? t * t / r2 : 0.0;
    return exp(-(d2 * kp.inv2s2 + d2 * s2phi * kp.ell_k));
}

// fp64 pair: returns hit; w = q-less kernel weight.  The definition with no shortcut:
// differences formed in degrees first, haversine, d = 2 asin(sqrt(hav)), w = exp(-d^2/(2 sigma^2)).
template <int KFN>
__device__ __forceinline__ bool pair64(const Rec64& r, double clon_deg, double clat_deg, double ccos, double csin,
                                       const KernelParams& kp, double& w) {
    const double dlat = (r.lat_deg - clat_deg) * kDeg2Rad;
    const double dlon = remainder(r.lon_deg - clon_deg, 360.0) * kDeg2Rad;
    const double sa = sin(0.5 * dlat), sb = sin(0.5 * dlon);
    double hav = sa * sa + ccos * r.coslat * sb * sb;
    if (hav > 1.0) hav = 1.0;
    const double d = 2.0 * asin(sqrt(hav));
    if (KFN == 2)
        w = elliptical64(d * d, r.coslat * sin(dlon), sin(dlat) + 2.0 * csin * r.coslat * sb * sb, kp);
    else
        w = KFN == 0 ? exp(-d * d * kp.inv2s2) : tapered_sinc64(d * d, kp);
    return d <= kp.radius;
}

// sin^2(y) = y^2 (1 - y^2/3 + 2 y^4/45 - y^6/315 + 2 y^8/14175 - ...): for |y| <= 0.025 the first
// omitted term is below 1e-21 relative.
__device__ __forceinline__ double sin2_small(double y) {
    const double t = y * y;
    return t * fma(t, fma(t, fma(t, fma(t, 2.0 / 14175.0, -1.0 / 315.0), 2.0 / 45.0), -1.0 / 3.0), 1.0);
}

// The same pair for small angles (support radius and longitude half-window <= 0.05 rad, the
// condition of the fp32 series path): sin^2 by its series and d^2 = 4 asin^2(sqrt(h)) =
// 4 h (1 + h/3 + 8 h^2/45 + 4 h^3/35 + ...), both exact to < 1e-16 relative there (h <= 6.3e-4), so the
// result agrees with pair64 far inside the 1e-12 tier while costing a third of its fp64 instructions.
// d <= R is tested as hav <= sin^2(R/2) (the same statement, asin and sqrt being monotone).
template <int KFN>
__device__ __forceinline__ bool pair64_small(const Rec64& r, double clon_deg, double clat_deg, double ccos, double csin,
                                             const KernelParams& kp, double& w) {
    const double dlat = (r.lat_deg - clat_deg) * kDeg2Rad;
    const double dlon = remainder(r.lon_deg - clon_deg, 360.0) * kDeg2Rad;
    const double sb2 = sin2_small(0.5 * dlon);
    const double h = sin2_small(0.5 * dlat) + ccos * r.coslat * sb2;
    const double d2 = 4.0 * h * fma(h, fma(h, fma(h, fma(h, 128.0 / 1575.0, 4.0 / 35.0), 8.0 / 45.0), 1.0 / 3.0), 1.0);
    if (KFN == 2)
        w = elliptical64(d2, r.coslat * sin(dlon), sin(dlat) + 2.0 * csin * r.coslat * sb2, kp);
    else
        w = KFN == 0 ? exp(-d2 * kp.inv2s2) : tapered_sinc64(d2, kp);
    return h <= kp.hav_max;
}

// Elliptical Gaussian from the fp32 pair arithmetic (series path: support radius and longitude half-window
// <= 0.05 rad).  With dx, dy the exact coordinate differences (rad), C = cos(lat_c) cos(lat_s) (the strip's
// polynomial in dy) and B = 4 sin^2(dx / 2) (series):
//     x = cos(lat_s) sin dx          = C sin(dx) / cos(lat_c)
//     y = sin dy + 2 sin(lat_c) cos(lat_s) sin^2(dx / 2) = sin(dy) + (tan(lat_c) / 2) C B
//     (d sin(beta - PA))^2 = (x cos PA - y sin PA)^2 (d / sin d)^2,  (d / sin d)^2 = 1 + d^2/3 + ... = 1 + h4/3 + O(d^4)
// sin z = z (1 - z^2/6 + z^4/120): next term 1.6e-12 relative at 0.05 rad.  icc = 1 / cos(lat_c), th = tan(lat_c) / 2.
__device__ __forceinline__ bool pair32_elliptical(const Rec32& r, const TaskConst& tc, float icc, float th,
                                                  const KernelParams& kp, float& w) {
    const float dx = (float)(int)(r.xi - tc.xc0) * tc.qx;
    const float dy = (float)(int)(r.yi - tc.yc) * tc.qy;
    const float u = dy * dy;
    const float u2 = u * fmaf(u, -1.0f / 12.0f, 1.0f);
    const float C = fmaf(dy, fmaf(dy, fmaf(dy, tc.c3, tc.c2), tc.c1), tc.c0);
    const float v = dx * dx;
    const float B = v * fmaf(v, -1.0f / 12.0f, 1.0f);
    const float CB = C * B;
    const float h4 = CB + u2;
    const float sdx = dx * fmaf(v, fmaf(v, 1.0f / 120.0f, -1.0f / 6.0f), 1.0f);
    const float sdy = dy * fmaf(u, fmaf(u, 1.0f / 120.0f, -1.0f / 6.0f), 1.0f);
    const float x = C * sdx * icc;
    const float y = fmaf(th, CB, sdy);
    const float t = x * kp.ecp - y * kp.esp;
    const float e2 = fmaf(h4, fmaf(h4, tc.k2, tc.k1), t * t * fmaf(h4, 1.0f / 3.0f, 1.0f) * kp.ek2);
    w = ex2_approx(e2);
    return h4 <= tc.h4max;
}

// KFN: kernel function (hcgrid_set_kernel), 0 Gaussian, 1 tapered sinc, 2 elliptical Gaussian -- a template parameter so
// that the Gaussian instantiations carry none of the other's code.
// one cell (strip s, column ix) by one warp
template <bool PAIR64, typename AccT, bool VEC4, int KFN>
__device__ __forceinline__ void conv_general_cell(const ConvArgs& a, const int s, const int ix, const int lane) {
    const int64_t task = (int64_t)s * a.strip_cells + ix;
    const Strip st = a.strips[s];
    const int nchan = a.nchan;
    const float* __restrict__ values = a.values;
    AccT* __restrict__ cube = (AccT*)a.cube;
    AccT* __restrict__ wmap = (AccT*)a.wmap;

    // cell constants
    TaskConst tc;
    double clon_deg = 0.0, clat_deg = 0.0, ccos = 0.0, csin = 0.0;
    float icc = 0.0f, th = 0.0f;                    // elliptical Gaussian, fp32 pairs: 1 / cos(lat_c), tan(lat_c) / 2
    if (PAIR64) {
        clon_deg = __dadd_rn(st.lon0_deg, __dmul_rn((double)ix, st.dlon_deg));   // no FMA (SURVEY 8c fp64 pin)
        clat_deg = st.lat_deg;
        ccos = cos(clat_deg * kDeg2Rad);
        if (KFN == 2) csin = sin(clat_deg * kDeg2Rad);
    } else {
        tc = make_task_const(a, st, ix);
        if (KFN == 2) {
            const double cl = cos(st.lat);
            icc = (float)(1.0 / cl);
            th = (float)(0.5 * sin(st.lat) / cl);
        }
    }

    for (int ch0 = 0; ch0 < nchan; ch0 += 256) {
        AccT acc[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[j] = (AccT)0;
        AccT W = (AccT)0;
        int cnt = 0;
        for (int k = 0; k < st.nring; ++k) {
            const RingWin w = a.wins[(size_t)s * a.kmax + k];
            int sa, sn, sa2, sn2;
            ring_segment(w, ix, 1, a.rg, a.bin_start, sa, sn, sa2, sn2);
            // second range: only where the window crosses the seam of a full-circle region (warp-uniform)
            for (int seg = 0; seg < 2; ++seg, sa = sa2, sn = sn2)
            for (int base = 0; base < sn; base += 32) {
                const int i = base + lane;
                bool hit = false;
                AccT wq = (AccT)0;
                uint32_t idx = 0;
                if (i < sn) {
                    if (PAIR64) {
                        const Rec64 r = ((const Rec64*)a.rec)[sa + i];
                        double wd;
                        hit = a.small64 ? pair64_small<KFN>(r, clon_deg, clat_deg, ccos, csin, a.kp, wd)
                                        : pair64<KFN>(r, clon_deg, clat_deg, ccos, csin, a.kp, wd);
                        wq = (AccT)(wd * (double)r.q);
                        idx = r.idx;
                    } else {
                        const uint4 raw = __ldg((const uint4*)a.rec + sa + i);
                        Rec32 r;
                        r.xi = raw.x; r.yi = raw.y; r.idx = raw.z; r.q = __uint_as_float(raw.w);
                        float wf, e2;
                        if (KFN == 2) {
                            hit = pair32_elliptical(r, tc, icc, th, a.kp, wf);
                        } else {
                            hit = pair32(r, tc, wf, &e2);
                            if (KFN == 1) wf = tapered_sinc32(e2, a.kp);
                        }
                        wq = (AccT)(wf * r.q);
                        idx = r.idx;
                    }
                }
                if (hit) { W += wq; cnt += 1; }
                if (nchan == 1) {
                    if (hit) acc[0] += wq * (AccT)(PAIR64 ? __ldg(values + idx) : __uint_as_float(idx));
                } else {
                    unsigned m = __ballot_sync(0xffffffffu, hit);
                    while (m) {
                        const int b = __ffs(m) - 1;
                        m &= m - 1;
                        const AccT wb = __shfl_sync(0xffffffffu, wq, b);
                        const uint32_t ib = __shfl_sync(0xffffffffu, idx, b);
                        const float* __restrict__ row = values + (size_t)ib * nchan + ch0;
                        if (VEC4) {
#pragma unroll
                            for (int j = 0; j < 2; ++j) {
                                const int c = 4 * lane + 128 * j;
                                if (ch0 + c < nchan) {
                                    const float4 v = __ldg((const float4*)(row + c));
                                    acc[4 * j + 0] += wb * (AccT)v.x;
                                    acc[4 * j + 1] += wb * (AccT)v.y;
                                    acc[4 * j + 2] += wb * (AccT)v.z;
                                    acc[4 * j + 3] += wb * (AccT)v.w;
                                }
                            }
                        } else {
#pragma unroll
                            for (int j = 0; j < 8; ++j) {
                                const int c = lane + 32 * j;
                                if (ch0 + c < nchan) acc[j] += wb * (AccT)__ldg(row + c);
                            }
                        }
                    }
                }
            }
        }
        W = warp_sum(W);
        cnt = warp_sum(cnt);
        const AccT nan = NanOf<AccT>::v();
        if (nchan == 1) {
            const AccT S = warp_sum(acc[0]);
            if (lane == 0) cube[task] = a.raw ? S : (W != (AccT)0 ? S / W : nan);
        } else if (VEC4) {
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const int c = ch0 + 4 * lane + 128 * j;
                if (c < nchan) {
                    AccT* o = cube + (size_t)task * nchan + c;
#pragma unroll
                    for (int t = 0; t < 4; ++t) o[t] = a.raw ? acc[4 * j + t] : (W != (AccT)0 ? acc[4 * j + t] / W : nan);
                }
            }
        } else {
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int c = ch0 + lane + 32 * j;
                if (c < nchan) cube[(size_t)task * nchan + c] = a.raw ? acc[j] : (W != (AccT)0 ? acc[j] / W : nan);
            }
        }
        if (ch0 == 0 && lane == 0) {
            wmap[task] = W;
            if (a.counts) a.counts[task] = cnt;
        }
    }
}

template <bool PAIR64, typename AccT, bool VEC4, int KFN>
__global__ void __launch_bounds__(256)
conv_general(const ConvArgs a) {
    const int64_t task = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (task >= a.ntasks) return;
    conv_general_cell<PAIR64, AccT, VEC4, KFN>(a, (int)(task / a.strip_cells), (int)(task % a.strip_cells), threadIdx.x & 31);
}

// The fix-up pass after the tensor-core cube kernel: only the cells of the 16 x 8-cell tiles on the list (tiles that met a
// non-finite value; usually none, and then every warp leaves at once), a warp at a time.
template <bool PAIR64, typename AccT, bool VEC4, int KFN>
__global__ void __launch_bounds__(256)
conv_general_listed(const ConvArgs a) {
    const int64_t ncells = (int64_t)__ldg(a.dirty_count) * 128;
    const int64_t nw = (int64_t)gridDim.x * (blockDim.x >> 5);
    for (int64_t wt = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); wt < ncells; wt += nw) {
        const int t16 = __ldg(a.dirty_list + (wt >> 7)), cl = (int)(wt & 127);
        const int s = (t16 / a.dirty_tiles_x) * 8 + (cl >> 4), ix = (t16 % a.dirty_tiles_x) * 16 + (cl & 15);
        if (s < a.nstrip && ix < a.strip_cells) conv_general_cell<PAIR64, AccT, VEC4, KFN>(a, s, ix, threadIdx.x & 31);
    }
}

// list of the tiles flagged in any channel block of dirty[nblk][ntiles]; *count must be zero on entry
__global__ void __launch_bounds__(256)
dirty_list_kernel(const int32_t* __restrict__ dirty, int nblk, int ntiles, int32_t* __restrict__ list, int32_t* __restrict__ count) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ntiles) return;
    int any = 0;
    for (int b = 0; b < nblk; ++b) any |= __ldg(dirty + (size_t)b * ntiles + t);
    if (any) list[atomicAdd(count, 1)] = t;             // order irrelevant: every cell is computed on its own
}

int launch_conv_general(hcgrid_ctx* c, const ConvArgs& a0, bool pair_f64, bool out_double, cudaStream_t st,
                        const int32_t* dirty) {
    ConvArgs a = a0;
    a.ntasks = c->ncell;
    a.tasks_per_strip = a.strip_cells;
    a.nstrip = c->nstrip;
    const bool vec4 = (a.nchan % 4 == 0) && ((uintptr_t)a.values % 16 == 0);
    const int threads = 256;
    unsigned blocks = (unsigned)((a.ntasks + 7) / 8);
    if (blocks == 0) return HCGRID_OK;
    if (dirty) {
        // dirty [nblk][ntiles] is followed by the list of flagged tiles [ntiles] and their count (convolve.cu sizes it)
        const int ntiles = mc_tc_tiles(c), nblk = (a.nchan + 255) / 256;
        a.dirty_tiles_x = (c->strip_cells + 15) / 16;
        int32_t* list = const_cast<int32_t*>(dirty) + (size_t)nblk * ntiles;
        int32_t* count = list + ntiles;
        a.dirty_list = list;
        a.dirty_count = count;
        HCG_CUDA(c, cudaMemsetAsync(count, 0, 4, st));
        dirty_list_kernel<<<(unsigned)((ntiles + 255) / 256), 256, 0, st>>>(dirty, nblk, ntiles, list, count);
        HCG_CUDA(c, cudaGetLastError());
        blocks = std::min<unsigned>(blocks, (unsigned)(8 * c->num_sms));
    }
#define HCG_LAUNCH(P, T, V)                                                        \
    do {                                                                           \
        if (dirty) conv_general_listed<P, T, V, 0><<<blocks, threads, 0, st>>>(a);  \
        else if (a.kp.ktype == 0) conv_general<P, T, V, 0><<<blocks, threads, 0, st>>>(a); \
        else if (a.kp.ktype == 1) conv_general<P, T, V, 1><<<blocks, threads, 0, st>>>(a); \
        else conv_general<P, T, V, 2><<<blocks, threads, 0, st>>>(a);              \
    } while (0)
    if (out_double) {
        if (vec4) HCG_LAUNCH(true, double, true); else HCG_LAUNCH(true, double, false);
    } else if (pair_f64) {
        if (vec4) HCG_LAUNCH(true, float, true); else HCG_LAUNCH(true, float, false);
    } else {
        if (vec4) HCG_LAUNCH(false, float, true); else HCG_LAUNCH(false, float, false);
    }
#undef HCG_LAUNCH
    HCG_CUDA(c, cudaGetLastError());
    return HCGRID_OK;
}

}  // namespace hcg
