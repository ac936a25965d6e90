// convolve_tile.cu -- step a6, the tile kernel: single-channel fp32 gather convolution for
// plate-carree targets (Sect. 3.4 i-v; Eq. 1; kernel
// PAPER.md:186), hand-written for sm_100a.  DESIGN.md "a6 / tile kernel".
//
// One WARP owns a tile of GX x GY target cells (the paper's thread coarsening,
// PAPER.md:153, in two dimensions and at warp scope); its 32 lanes stride over the
// candidate samples of the tile, so each lane holds one sample and GX*GY partial sums.
//   step (i)    rings of the tile = union of its rows' precomputed ring ranges (a1)
//   step (ii)   lane k turns ring k's window (fp32 RingWinF of every tile row, united) into
//               a range of lookup bins
//   step (iii)  two reads of the per-pixel table give the sample range [S_start, S_end)
//   step (iv)   the ranges of all rings form one candidate stream: a 32-entry table
//               (end position, address offset) per warp in shared memory lets every lane
//               walk the stream with a monotone ring cursor; records are read straight
//               from global memory (16-byte loads, one step ahead of the arithmetic)
//   step (v)    pair arithmetic in fp32 on exact fixed-point coordinate differences, with
//               everything that depends only on the sample's column or row offset hoisted
//               out of the GX*GY pair loop and all lengths pre-scaled by
//               sqrt(log2(e) / (2 sigma^2)), so a pair costs FFMA (distance), FSETP
//               (d <= R), MUFU.EX2, FFMA (W), FFMA (sum) [+ IADD (count)].
// The 32 partial sums per cell are combined by a transposed butterfly (each shuffle step
// halves the number of live values), in a fixed order, without atomics.
#include "hcg_tile.cuh"

namespace hcg {

constexpr int kTileWarps = 4;        // warps (= tiles) per CTA when tiles are not split
constexpr int kMaxTileWarps = 4;     // largest split: warps of one CTA on one tile

// 8-cell Gaussian tiles without the count output fit 64 registers in every series mode (8 CTAs per SM) once ptxas is
// asked to; left to itself it takes 71-72 for the series modes (0 = no request for the other variants).
template <int GX, int GY, int MODE, bool COUNTS, bool SPLIT, int KFN = 0>
__global__ void __launch_bounds__(kMaxTileWarps * 32, (!COUNTS && KFN == 0 && GX * GY == 8) ? 8 : 0)
conv1_tile_f32(const TileArgs a) {
    constexpr int NC = GX * GY;
    __shared__ unsigned long long s_tab[kMaxTileWarps][32];
    __shared__ float s_pw[SPLIT ? kMaxTileWarps : 1][NC], s_ps[SPLIT ? kMaxTileWarps : 1][NC];   // partial sums of a split tile
    __shared__ int s_pc[SPLIT ? kMaxTileWarps : 1][NC];
    const int lane = threadIdx.x & 31;
    const int wib = threadIdx.x >> 5;
    // a.split == 1: the CTA's warps own consecutive tiles.  a.split == S > 1 (few tiles, long streams):
    // the CTA is S warps on ONE tile, warp p taking the stream steps p, p + S, ...; their partial sums
    // are added in warp order through shared memory (fixed order, no atomics).
    const int S = SPLIT ? a.split : 1;                          // SPLIT = false compiles to the plain one-warp-per-tile kernel
    const int part = SPLIT ? wib : 0;
    const unsigned tile = SPLIT ? blockIdx.x : blockIdx.x * kTileWarps + wib;   // ntiles <= 2^30 (api.cu)
    if (tile >= (unsigned)a.ntiles) return;                     // the whole CTA when S > 1
    const int ty = (int)(tile / (unsigned)a.tiles_x);
    const int ix0 = (int)(tile - (unsigned)ty * (unsigned)a.tiles_x) * GX;
    const int row0 = ty * GY;
    const int ncols = min(GX, a.nx - ix0);
    const int nrows = min(GY, a.ny - row0);

    // ---- tile constants
    TileConst<GY> tc;
    int ring_lo[GY], nring[GY];
    int rmin = 0x7fffffff, rmax = -0x7fffffff;
#pragma unroll
    for (int j = 0; j < GY; ++j) {
        const int4* rp = (const int4*)(a.rows + min(row0 + j, a.ny - 1));
        const int4 r0 = __ldg(rp);
        const int4 r1 = __ldg(rp + 1);
        ring_lo[j] = r0.y;
        nring[j] = j < nrows ? r0.z : 0;
        tc.cc[j] = __int_as_float(r0.w);
        if (KFN == 2) tc.sh[j] = 0.5f * __int_as_float(r1.x) * a.isk;
        if (j == 0) {
            tc.yc0 = (uint32_t)r0.x;
            tc.cc0 = __int_as_float(r0.w);
            const float sc0 = __int_as_float(r1.x);
            const float ik = a.isk;
            tc.p1 = -sc0 * ik;
            tc.p2 = -0.5f * tc.cc0 * ik * ik;
            tc.p3 = sc0 * ik * ik * ik * (1.0f / 6.0f);
        }
        if (j < nrows) {
            rmin = min(rmin, r0.y);
            rmax = max(rmax, r0.y + r0.z - 1);
        }
    }
    tc.xc0 = (uint32_t)(unsigned long long)__double2ll_rn((a.u0 + (double)ix0 * a.du) * a.sx);
    tc.sxk = a.sxk; tc.syk = a.syk; tc.duk = a.duk; tc.dyk = a.dyk;
    tc.a12 = a.a12; tc.hmax = a.hmax;
    tc.ts1 = a.ts1; tc.tg2 = a.tg2;
    tc.ecp = a.ecp; tc.esp = a.esp; tc.erk = a.erk;

    float W[NC], S_[NC];
    int cnt[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) { W[c] = 0.f; S_[c] = 0.f; cnt[c] = 0; }

    const float fxw = (float)(a.du >= 0.0 ? ix0 : ix0 + ncols - 1);   // westmost / eastmost column of the tile
    const float fxe = (float)(a.du >= 0.0 ? ix0 + ncols - 1 : ix0);
    const Rec32* __restrict__ rec = a.rec;
    unsigned long long* tab = s_tab[wib];

    for (int rb = rmin; rb <= rmax; rb += 32) {
        // ---- steps (ii)+(iii): lane k <-> ring rb + k
        const int r = rb + lane;
        int jlo = 0x7fffffff, jhi = -1;
#pragma unroll
        for (int j = 0; j < GY; ++j) {
            const int k = r - ring_lo[j];
            if (k >= 0 && k < nring[j]) {
                const float4 w = __ldg((const float4*)(a.wins + (size_t)(row0 + j) * a.kmax + k));
                const int fl = __float_as_int(w.w);
                if (fl == 1) {
                    jlo = min(jlo, __float2int_rd(fmaf(fxw, w.z, w.x)));
                    jhi = max(jhi, __float2int_rd(fmaf(fxe, w.z, w.y)));
                } else if (fl == 2) {
                    jlo = 0; jhi = a.m - 1;
                }
            }
        }
        jlo = max(jlo, 0);
        jhi = min(jhi, a.m - 1);
        int sa = 0, sn = 0;
        if (jhi >= jlo) {
            const int32_t* bs = a.bin_start + (size_t)r * a.m;
            sa = __ldg(bs + jlo);
            sn = __ldg(bs + jhi + 1) - sa;
        }
        int incl = sn;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        const int total = __shfl_sync(0xffffffffu, incl, 31);
        __syncwarp();                                   // previous pass done with the table
        // (end of ring k in the stream, index of the record that would have stream index 0)
        tab[lane] = (unsigned long long)(unsigned)incl | ((unsigned long long)(unsigned)(sa - (incl - sn)) << 32);
        __syncwarp();
        if (total == 0) continue;

        // ---- steps (iv)+(v): the candidate stream, one record ahead.  Full steps (all 32 lanes
        // inside the stream) need no validity test; the ragged last step tests against a negative
        // threshold in the lanes past the end (they re-read the last record).
        const int last = total - 1;
        const int nfull = total >> 5;
        const int stride = 32 * S;
        uint32_t tp = smem_addr(tab);                   // ring cursor: shared address of entry k
        unsigned long long eb = lds_entry8(tp);
        int i = part * 32 + lane;
        stream_seek8(min(i, last), tp, eb);
        uint4 ra = ldg_rec8(rec, eb, min(i, last));
        int i1 = i + stride;
        stream_seek8(min(i1, last), tp, eb);
        uint4 rn = ldg_rec8(rec, eb, min(i1, last));
        tc.hm = tc.hmax;
#pragma unroll 3
        for (int it = part; it < nfull; it += S) {
            const int i2 = i1 + stride;
            const int ii = min(i2, last);
            stream_seek8(ii, tp, eb);
            const uint4 rc = ldg_rec8(rec, eb, ii);
            tile_pairs<GX, GY, MODE, COUNTS, KFN>(ra, tc, W, S_, cnt);
            ra = rn; rn = rc;
            i = i1; i1 = i2;
        }
        if ((total & 31) && (nfull & (S - 1)) == part) {  // the ragged last step belongs to one warp
            tc.hm = i <= last ? tc.hmax : -1.0f;
            tile_pairs<GX, GY, MODE, COUNTS, KFN>(ra, tc, W, S_, cnt);
        }
    }

    // ---- finish: transposed reduction, (split tiles: partial sums through shared memory), normalise, store
    TileReduce<NC, 16, float>::run(W, lane);
    TileReduce<NC, 16, float>::run(S_, lane);
    if (COUNTS) TileReduce<NC, 16, int>::run(cnt, lane);
    constexpr int SHIFT = 5 - ilog2(NC);
    const bool writer = (lane & ((1 << SHIFT) - 1)) == 0;
    const int c = lane >> SHIFT;
    float wsum = W[0], ssum = S_[0];
    int csum = cnt[0];
    if (SPLIT) {
        if (writer) { s_pw[wib][c] = wsum; s_ps[wib][c] = ssum; s_pc[wib][c] = csum; }
        __syncthreads();
        if (wib != 0) return;
        if (writer) {
            wsum = s_pw[0][c]; ssum = s_ps[0][c]; csum = s_pc[0][c];
            for (int w = 1; w < S; ++w) { wsum += s_pw[w][c]; ssum += s_ps[w][c]; csum += s_pc[w][c]; }
        }
    }
    if (writer) {
        const int gx = c % GX, gy = c / GX;
        if (gx < ncols && gy < nrows) {
            const int64_t cell = (int64_t)(row0 + gy) * a.nx + ix0 + gx;
            a.cube[cell] = a.raw ? ssum : (wsum != 0.0f ? ssum / wsum : __int_as_float(0x7fc00000));
            a.wmap[cell] = wsum;
            if (COUNTS) a.counts[cell] = csum;
        }
    }
}

// ------------------------------------------------------------------ launcher
template <int GX, int GY>
static cudaError_t launch_shape(const TileArgs& a, int mode, bool counts, cudaStream_t st) {
    const unsigned blocks = a.split > 1 ? (unsigned)a.ntiles : (unsigned)((a.ntiles + kTileWarps - 1) / kTileWarps);
    const int threads = (a.split > 1 ? a.split : kTileWarps) * 32;
#define HCG_TILE(M, C)                                                                 \
    do {                                                                               \
        if (a.split > 1) conv1_tile_f32<GX, GY, M, C, true><<<blocks, threads, 0, st>>>(a);  \
        else conv1_tile_f32<GX, GY, M, C, false><<<blocks, threads, 0, st>>>(a);       \
    } while (0)
    switch (mode * 2 + (counts ? 1 : 0)) {
        case 0: HCG_TILE(0, false); break;
        case 1: HCG_TILE(0, true); break;
        case 2: HCG_TILE(1, false); break;
        case 3: HCG_TILE(1, true); break;
        case 4: HCG_TILE(2, false); break;
        default: HCG_TILE(2, true); break;
    }
#undef HCG_TILE
    return cudaGetLastError();
}

// Tapered sinc (KFN 1) and elliptical Gaussian (KFN 2): series mode 2 only (valid wherever the tile kernel is),
// three shapes.
template <int GX, int GY, int KFN>
static cudaError_t launch_shape_kfn(const TileArgs& a, bool counts, cudaStream_t st) {
    const unsigned blocks = a.split > 1 ? (unsigned)a.ntiles : (unsigned)((a.ntiles + kTileWarps - 1) / kTileWarps);
    const int threads = (a.split > 1 ? a.split : kTileWarps) * 32;
    if (counts) {
        if (a.split > 1) conv1_tile_f32<GX, GY, 2, true, true, KFN><<<blocks, threads, 0, st>>>(a);
        else conv1_tile_f32<GX, GY, 2, true, false, KFN><<<blocks, threads, 0, st>>>(a);
    } else {
        if (a.split > 1) conv1_tile_f32<GX, GY, 2, false, true, KFN><<<blocks, threads, 0, st>>>(a);
        else conv1_tile_f32<GX, GY, 2, false, false, KFN><<<blocks, threads, 0, st>>>(a);
    }
    return cudaGetLastError();
}

static const int kShapes[][2] = {{1, 1}, {2, 1}, {4, 1}, {8, 1}, {2, 2}, {4, 2}, {8, 2}, {4, 4}};
static bool kfn_shape_built(int gx, int gy) { return (gx == 1 && gy == 1) || (gx == 2 && gy == 2) || (gx == 4 && gy == 2); }

// Instruction-count model of one tile: warp instructions per cell.
static double shape_cost(int gx, int gy, int mode, bool counts, double cw, double ch, double two_r,
                         double ring_sp, double cand_per_cell, int kfn = 0) {
    const double infl = (two_r + (gx - 1) * cw) / two_r * (two_r + 2.0 * ring_sp + (gy - 1) * ch) / (two_r + 2.0 * ring_sp);
    const double per_iter = 18.0 + (mode >= 1 ? 4.0 : 2.0) * gx + (mode >= 1 ? 5.0 : 3.0) * gy +
                            (5.0 + (counts ? 1.0 : 0.0) + (mode == 2 ? 2.0 : 0.0) + (kfn == 1 ? 45.0 : kfn == 2 ? 6.0 : 0.0)) * gx * gy +
                            (kfn == 2 ? 5.0 * (gx + gy) : 0.0);
    const double iters = cand_per_cell * infl / 32.0 + 0.5;
    const double overhead = 150.0 + 14.0 * gy + 8.0 * gx * gy;
    // 16-cell tiles need ~100 registers per thread; measured on B200 they run 15-25 % slower than
    // the instruction count alone predicts (configs 2, 3, 5)
    const double occ = gx * gy >= 16 ? 1.25 : 1.0;
    return occ * (iters * per_iter + overhead) / (gx * gy);
}

int tile_series_mode(const hcgrid_ctx* c) {
    const KernelParams& kp = c->kp;
    const double amax = std::max(c->dlmax, kp.radius);
    const bool need_xy = amax * amax / 12.0 > 1e-7;
    const bool need_d = kp.radius * kp.radius * kp.inv2s2 * (kp.radius * kp.radius / 12.0) > 1e-6;
    return need_d ? 2 : (need_xy ? 1 : 0);
}

void fill_tile_args(const hcgrid_ctx* c, int mode, TileArgs& a) {
    const Region& rg = c->region;
    const KernelParams& kp = c->kp;
    const double kappa = 1.4426950408889634074 * kp.inv2s2;
    const double sk = std::sqrt(kappa);
    a.rows = c->d_rowsf.as<RowF>();
    a.wins = c->d_winsf.as<RingWinF>();
    a.bin_start = c->d_bins.as<int32_t>();
    a.rec = c->d_rec.as<Rec32>();
    a.u0 = c->car_u0; a.du = c->car_du; a.sx = rg.sx32;
    a.nx = c->strip_cells; a.ny = c->nstrip; a.kmax = c->kmax; a.m = rg.m;
    a.sxk = (float)(sk / rg.sx32);
    a.syk = (float)(sk / rg.sy32);
    a.duk = (float)(sk * c->car_du);
    a.dyk = (float)(sk * c->car_dlat);
    a.isk = (float)(1.0 / sk);
    a.a12 = (float)(1.0 / (12.0 * kappa));
    a.hmax = (float)(mode == 0 ? kappa * kp.radius * kp.radius : kappa * 4.0 * kp.hav_max);
    a.split = 1;
    a.raw = c->raw_sums ? 1 : 0;
}

int launch_conv_tile(hcgrid_ctx* c, int64_t n, float* cube, float* wmap, int32_t* counts, cudaStream_t st) {
    const Region& rg = c->region;
    const KernelParams& kp = c->kp;
    const int nx = c->strip_cells, ny = c->nstrip;
    const int kfn = kp.ktype;            // 0 Gaussian, 1 tapered sinc, 2 elliptical Gaussian
    const int mode = kfn != 0 ? 2 : tile_series_mode(c);

    // tile shape: forced by the options or chosen by the instruction-count model
    int gx = c->opt_coarsen, gy = c->opt_coarsen_y;
    if (gx == 0 || gy == 0) {
        const double two_r = 2.0 * kp.radius;
        const double ring_sp = rg.wy / std::max(1, rg.nring);
        // candidates of one cell's own search: samples per unit area x bounding box of the disc
        const double dens = (double)n / std::max(1e-300, rg.wx * rg.wy);
        const double cand = dens * (2.0 * c->dlmax) * (two_r + 2.0 * ring_sp);
        double best = 1e300;
        int bx = 1, by = 1;
        for (const auto& s : kShapes) {
            if ((gx != 0 && s[0] != gx) || (gy != 0 && s[1] != gy)) continue;
            if (s[0] > nx && s[0] > 1) continue;
            if (s[1] > ny && s[1] > 1) continue;
            if (kfn != 0 && !kfn_shape_built(s[0], s[1])) continue;
            const double cost = shape_cost(s[0], s[1], mode, counts != nullptr, c->cell_width_sky,
                                           std::fabs(c->car_dlat), two_r, ring_sp, cand, kfn);
            if (cost < best) { best = cost; bx = s[0]; by = s[1]; }
        }
        if (best == 1e300)
            return fail(c, HCGRID_ERR_INVALID_ARG, "tile shape %d x %d not built", gx, gy);
        gx = bx; gy = by;
    }

    TileArgs a{};
    fill_tile_args(c, mode, a);
    a.cube = cube; a.wmap = wmap; a.counts = counts;
    a.tiles_x = (nx + gx - 1) / gx;
    a.ntiles = (int64_t)a.tiles_x * ((ny + gy - 1) / gy);
    // Few tiles with long candidate streams (the paper's own experiments: 90 x 90 cells, up to
    // 3.6e8 samples) cannot fill 148 SMs with one warp per tile: split every
    // tile's stream over S warps of one CTA until about 48 warps per SM exist, as long as each
    // warp keeps at least 8 stream steps.
    int split = c->opt_split;
    if (split == 0) {
        split = 1;
        const double two_r = 2.0 * kp.radius;
        const double ring_sp = rg.wy / std::max(1, rg.nring);
        const double dens = (double)n / std::max(1e-300, rg.wx * rg.wy);
        const double steps = dens * (2.0 * c->dlmax + (gx - 1) * std::fabs(c->car_du)) *
                             (two_r + 2.0 * ring_sp + (gy - 1) * std::fabs(c->car_dlat)) / 32.0;
        const double want = 48.0 * c->num_sms;
        while (split < kMaxTileWarps && (double)a.ntiles * split < want && steps / (2 * split) >= 8.0) split *= 2;
    }
    a.split = split;

    cudaError_t e = cudaSuccess;
    bool built = false;
    if (kfn == HCGRID_KERNEL_TAPERED_SINC) {
        a.ts1 = kp.ts1; a.tg2 = kp.tg2;
#define HCG_SHAPE(X, Y) if (gx == X && gy == Y) { built = true; e = launch_shape_kfn<X, Y, 1>(a, counts != nullptr, st); }
        HCG_SHAPE(1, 1); HCG_SHAPE(2, 2); HCG_SHAPE(4, 2);
#undef HCG_SHAPE
    } else if (kfn == HCGRID_KERNEL_ELLIPTICAL_GAUSS) {
        a.ecp = kp.ecp; a.esp = kp.esp; a.erk = (float)(kp.ell_k / kp.inv2s2);
#define HCG_SHAPE(X, Y) if (gx == X && gy == Y) { built = true; e = launch_shape_kfn<X, Y, 2>(a, counts != nullptr, st); }
        HCG_SHAPE(1, 1); HCG_SHAPE(2, 2); HCG_SHAPE(4, 2);
#undef HCG_SHAPE
    } else {
#define HCG_SHAPE(X, Y) if (gx == X && gy == Y) { built = true; e = launch_shape<X, Y>(a, mode, counts != nullptr, st); }
        HCG_SHAPE(1, 1); HCG_SHAPE(2, 1); HCG_SHAPE(4, 1); HCG_SHAPE(8, 1);
        HCG_SHAPE(2, 2); HCG_SHAPE(4, 2); HCG_SHAPE(8, 2); HCG_SHAPE(4, 4);
#undef HCG_SHAPE
    }
    if (!built)
        return fail(c, HCGRID_ERR_INVALID_ARG, "tile shape %d x %d not built", gx, gy);
    if (e != cudaSuccess) return cuda_fail(c, e, "conv1_tile_f32");
    c->stats.coarsen = gx;
    c->stats.coarsen_y = gy;
    c->stats.split = split;
    return HCGRID_OK;
}

// ------------------------------------------------------------------ profiling: pairs put to the distance test
// One thread per tile: steps (i)-(iii) exactly as conv1_tile_f32 takes them (union of the rows' ring ranges, united
// lookup-bin windows, two table reads per ring) give the length of the tile's candidate stream; every candidate is
// tested against every cell of the tile.
__global__ void __launch_bounds__(256) tile_pairs_tested_kernel(const TileArgs a, int gx, int gy, unsigned long long* out) {
    const int64_t tile = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long pairs = 0;
    if (tile < a.ntiles) {
        const int ty = (int)(tile / a.tiles_x);
        const int ix0 = (int)(tile - (int64_t)ty * a.tiles_x) * gx, row0 = ty * gy;
        const int ncols = min(gx, a.nx - ix0), nrows = min(gy, a.ny - row0);
        int rmin = 0x7fffffff, rmax = -0x7fffffff;
        for (int j = 0; j < nrows; ++j) {
            const int4 r0 = __ldg((const int4*)(a.rows + row0 + j));
            rmin = min(rmin, r0.y);
            rmax = max(rmax, r0.y + r0.z - 1);
        }
        const float fxw = (float)(a.du >= 0.0 ? ix0 : ix0 + ncols - 1), fxe = (float)(a.du >= 0.0 ? ix0 + ncols - 1 : ix0);
        long long total = 0;
        for (int r = rmin; r <= rmax; ++r) {
            int jlo = 0x7fffffff, jhi = -1;
            for (int j = 0; j < nrows; ++j) {
                const int4 r0 = __ldg((const int4*)(a.rows + row0 + j));
                const int k = r - r0.y;
                if (k >= 0 && k < r0.z) {
                    const float4 w = __ldg((const float4*)(a.wins + (size_t)(row0 + j) * a.kmax + k));
                    const int fl = __float_as_int(w.w);
                    if (fl == 1) {
                        jlo = min(jlo, __float2int_rd(fmaf(fxw, w.z, w.x)));
                        jhi = max(jhi, __float2int_rd(fmaf(fxe, w.z, w.y)));
                    } else if (fl == 2) {
                        jlo = 0; jhi = a.m - 1;
                    }
                }
            }
            jlo = max(jlo, 0);
            jhi = min(jhi, a.m - 1);
            if (jhi >= jlo) {
                const int32_t* bs = a.bin_start + (size_t)r * a.m;
                total += __ldg(bs + jhi + 1) - __ldg(bs + jlo);
            }
        }
        pairs = (unsigned long long)total * (unsigned long long)(ncols * nrows);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) pairs += __shfl_xor_sync(0xffffffffu, pairs, o);
    if ((threadIdx.x & 31) == 0 && pairs != 0) atomicAdd(out, pairs);   // integer: order-independent
}

int launch_tile_pairs_tested(hcgrid_ctx* c, int gx, int gy, unsigned long long* out, cudaStream_t st) {
    TileArgs a{};
    fill_tile_args(c, tile_series_mode(c), a);
    a.tiles_x = (a.nx + gx - 1) / gx;
    a.ntiles = (int64_t)a.tiles_x * ((a.ny + gy - 1) / gy);
    tile_pairs_tested_kernel<<<(unsigned)((a.ntiles + 255) / 256), 256, 0, st>>>(a, gx, gy, out);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e, "tile_pairs_tested_kernel");
    return HCGRID_OK;
}

}  // namespace hcg
