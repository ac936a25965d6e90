// hcg_conv.cuh -- what the convolution kernels (convolve.cu, convolve_gen.cu) share:
// the kernel argument block and steps (ii)+(iii) of the search.
#pragma once
#include "hcg_common.cuh"

namespace hcg {

// ------------------------------------------------------------------ shared device code
struct ConvArgs {
    const Strip* strips;
    const RingWin* wins;
    const int32_t* bin_start;
    const void* rec;            // Rec32* or Rec64*
    const float* values;        // original values [n][nchan] (multi-channel / fp64 kernels)
    void* cube;
    void* wmap;
    int32_t* counts;
    Region rg;
    KernelParams kp;
    int32_t kmax, strip_cells, tasks_per_strip, coarsen;
    int64_t ntasks;
    int32_t nchan;
    int32_t chunk;              // records per staging buffer (staged kernel)
    int32_t raw;                // 1: write the un-normalised sums (incremental gridding)
    int32_t small64;            // 1: fp64 pairs by the small-angle series (pair64_small), 0: full functions
    float qx, qy;               // radians per fixed-point unit
    double sx;                  // fixed-point units per radian (lon)
    // fix-up pass of the general kernel after the tensor-core cube kernel (convolve_mc_tc.cu): only the cells of
    // the dirty_count[0] tiles of 16 x 8 cells listed in dirty_list are recomputed (conv_general_listed)
    const int32_t* dirty_list;
    const int32_t* dirty_count;
    int32_t dirty_tiles_x, nstrip;
};

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Step (ii)+(iii): sample ranges of ring-window `w` for the cells [ix0, ix0+g-1]: [a, a+n) and, only on a region
// that spans the whole circle when the pixel window crosses the ring's first pixel, a second range [a2, a2+n2).
// (Pixel indices of such a window are reduced modulo the ring length nb, so a window on the seam costs its own
// length, not the whole ring.)
__device__ __forceinline__ void ring_segment(const RingWin& w, int ix0, int g, const Region& rg,
                                             const int32_t* __restrict__ bin_start, int& a, int& n, int& a2, int& n2) {
    a = 0; n = 0; a2 = 0; n2 = 0;
    if (w.flags == 0) return;
    long long jlo, jhi, klo = 0, khi = -1;
    if (w.flags == 2) {
        jlo = 0; jhi = (w.nb < rg.m ? w.nb : rg.m) - 1;
    } else {
        const int ixw = w.step >= 0.0 ? ix0 : ix0 + g - 1;
        const int ixe = w.step >= 0.0 ? ix0 + g - 1 : ix0;
        jlo = (long long)floor(w.a_lo + (double)ixw * w.step);
        jhi = (long long)floor(w.a_hi + (double)ixe * w.step);
        if (rg.full_circle) {
            const long long len = jhi - jlo + 1;
            if (len >= w.nb) {
                jlo = 0; jhi = w.nb - 1;
            } else {
                long long j0 = jlo % w.nb;
                if (j0 < 0) j0 += w.nb;
                jlo = j0;
                jhi = j0 + len - 1;
                if (jhi >= w.nb) { klo = 0; khi = jhi - w.nb; jhi = w.nb - 1; }
            }
        } else {
            if (jhi < 0 || jlo > rg.m - 1) return;
            if (jlo < 0) jlo = 0;
            if (jhi > rg.m - 1) jhi = rg.m - 1;
        }
    }
    const long long base = (long long)w.ring_rel * rg.m;
    a = __ldg(bin_start + base + jlo);
    n = __ldg(bin_start + base + jhi + 1) - a;
    if (khi >= klo) {
        a2 = __ldg(bin_start + base + klo);
        n2 = __ldg(bin_start + base + khi + 1) - a2;
    }
}
// the same for regions that do not span the circle (never a second range)
__device__ __forceinline__ void ring_segment(const RingWin& w, int ix0, int g, const Region& rg,
                                             const int32_t* __restrict__ bin_start, int& a, int& n) {
    int a2, n2;
    ring_segment(w, ix0, g, rg, bin_start, a, n, a2, n2);
}

struct TaskConst {
    uint32_t xc0, yc;
    float c0, c1, c2, c3, du;
    float qx, qy, h4max, k1, k2;
};

__device__ __forceinline__ TaskConst make_task_const(const ConvArgs& a, const Strip& st, int ix0) {
    TaskConst tc;
    const double u = st.u0 + (double)ix0 * st.du;
    tc.xc0 = (uint32_t)(unsigned long long)__double2ll_rn(u * a.sx);
    tc.yc = st.yi;
    tc.c0 = st.c0; tc.c1 = st.c1; tc.c2 = st.c2; tc.c3 = st.c3; tc.du = st.du_f;
    tc.qx = a.qx; tc.qy = a.qy; tc.h4max = a.kp.h4max; tc.k1 = a.kp.k1; tc.k2 = a.kp.k2;
    return tc;
}

// Step (v), one cell: fp32 pair arithmetic on exact fixed-point differences (see
// pair_update in convolve.cu for the derivation).  Returns d <= R and the kernel weight.
__device__ __forceinline__ bool pair32(const Rec32& r, const TaskConst& tc, float& w, float* e2_out = nullptr) {
    const float dx = (float)(int)(r.xi - tc.xc0) * tc.qx;
    const float dy = (float)(int)(r.yi - tc.yc) * tc.qy;
    const float u = dy * dy;
    const float u2 = u * fmaf(u, -1.0f / 12.0f, 1.0f);
    const float C = fmaf(dy, fmaf(dy, fmaf(dy, tc.c3, tc.c2), tc.c1), tc.c0);
    const float v = dx * dx;
    const float B = v * fmaf(v, -1.0f / 12.0f, 1.0f);
    const float h4 = fmaf(C, B, u2);
    const float e2 = h4 * fmaf(h4, tc.k2, tc.k1);     // -d^2 log2e / (2 sigma^2)
    if (e2_out) *e2_out = e2;
    w = ex2_approx(e2);
    return h4 <= tc.h4max;
}

// launcher of convolve_tile.cu (single channel, fp32, plate-carree targets)
int launch_conv_tile(hcgrid_ctx* c, int64_t n, float* cube, float* wmap, int32_t* counts, cudaStream_t st);

// pairs the tile kernel puts to the distance test with gx x gy tiles: candidate-stream length x cells of every tile, added to *out
int launch_tile_pairs_tested(hcgrid_ctx* c, int gx, int gy, unsigned long long* out, cudaStream_t st);

// launcher of convolve_mc.cu (many channels, fp32, plate-carree targets, nchan % 4 == 0)
int launch_conv_mc(hcgrid_ctx* c, const float* values, int nchan, float* cube, float* wmap, int32_t* counts,
                   cudaStream_t st);

// launcher of convolve_mc_tc.cu (tcgen05 / TMEM; many channels, fp32, plate-carree targets, nchan % 32 == 0);
// dirty [ceil(nchan / 256)][mc_tc_tiles] receives 1 for every tile that met a non-finite value
int launch_conv_mc_tc(hcgrid_ctx* c, const float* values, int nchan, float* cube, float* wmap, int32_t* counts,
                      int32_t* dirty, cudaStream_t st);
int mc_tc_tiles(const hcgrid_ctx* c);

// launcher of convolve_gen.cu; dirty: see ConvArgs
int launch_conv_general(hcgrid_ctx* c, const ConvArgs& a, bool pair_f64, bool out_double, cudaStream_t st,
                        const int32_t* dirty = nullptr);

}  // namespace hcg
