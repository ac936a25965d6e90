// hcg_common.cuh -- shared types of libhcgrid (context, target description, device tables).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <string>

#include "../../include/hcgrid.h"
#include "hcg_healpix.cuh"

namespace hcg {

// ---------------------------------------------------------------- device-side layouts
// One "strip" = consecutive target cells sharing a latitude with uniform longitude
// spacing: a row of a plate-carree target, or a single cell of an arbitrary target.
struct Strip {
    double u0;        // (lon of cell 0 - region lon_lo) mod 2pi, rad
    double du;        // signed lon step between cells, rad (0 for single-cell strips)
    double lat;       // rad
    double lon0_deg;  // lon of cell 0 in degrees as the caller gave it (fp64 kernel)
    double dlon_deg;  // lon step in degrees
    double lat_deg;
    int32_t ring_lo;  // first ring (relative to region ring_first) of the strip's table
    int32_t nring;    // entries used in the strip's table row (<= kmax)
    uint32_t yi;      // fixed-point latitude of the strip (Rec32 convention)
    // cos(lat_c) cos(lat_c + dy) = c0 + dy (c1 + dy (c2 + dy c3)), fp32 coefficients
    float c0, c1, c2, c3;
    float du_f;       // du rounded to fp32
    int32_t pad_;
};

// Per (strip, ring) search window, precomputed by a1 (PAPER.md:136 step i-ii): the
// lookup-bin range of the disc's longitude extent on that ring as a linear function of
// the cell index ix along the strip.
//   first bin = floor(a_lo + ix_west * step),  last bin = floor(a_hi + ix_east * step)
// flags: 0 = empty (ring band does not meet the disc), 1 = window, 2 = whole ring
struct RingWin {
    double a_lo, a_hi, step;
    int32_t ring_rel;
    int32_t flags;
    int32_t nb;       // lookup bins along this ring (whole-ring / wrap logic)
    int32_t pad_;
};

// fp32 form of RingWin for the tile kernel (convolve_tile.cu): the same window with the
// bounds rounded outwards by the worst-case fp32 evaluation error, so that
//   first bin = floor(a_lo + ix_west * step),  last bin = floor(a_hi + ix_east * step)
// evaluated in fp32 is a superset of the fp64 window.  Entry k of a strip's row is ring
// strip.ring_lo + k.  flags as in RingWin.
struct __align__(16) RingWinF {
    float a_lo, a_hi, step;
    int32_t flags;
};

// Per-strip constants of the tile kernel (32 bytes, read with two 16-byte loads).
struct __align__(16) RowF {
    uint32_t yi;      // fixed-point latitude of the row (Rec32 convention)
    int32_t ring_lo;  // first ring (relative to region ring_first) of the row's window table
    int32_t nring;    // entries used in the row's window table
    float cc;         // cos(lat_c)
    float sc;         // sin(lat_c)
    int32_t pad_[3];
};

// 16-byte packed sample S' as the fp32 convolution reads it (a5).  xi/yi are unsigned
// fixed point over the region: lon offset u in [0, wx) -> xi = u * Region::sx32 (wraps
// naturally when wx = 2 pi), lat offset -> yi.  Differences of two fixed-point
// coordinates are exact integers, which is what keeps fp32 pair arithmetic at 1e-10 rad.
struct __align__(16) Rec32 {
    uint32_t xi, yi;
    union { float v; uint32_t idx; };  // value (nchan == 1) or original sample index
    float q;                            // per-sample weight (1 if none)
};

// fp64 mode sample: caller's degrees untouched (differences are formed in degrees first)
struct __align__(16) Rec64 {
    double lon_deg, lat_deg;
    double coslat;
    uint32_t idx;
    float q;
};

struct Region {            // what of the sphere the target can reach (host + device copy)
    int32_t nside;
    int32_t subpix;        // b: 2^b lookup bins per pixel (b may be negative)
    int32_t ring_first;    // HEALPix ring number of relative ring 0
    int32_t nring;         // rings in the tables
    int32_t m;             // bins per ring in the table (table is [nring][m], +1 sentinel)
    int32_t full_circle;   // 1: the longitude window is the whole circle
    double lon_lo;         // rad, [0, 2pi)
    double wx;             // rad, longitude extent mapped onto 2^32
    double lat_lo;         // rad
    double wy;             // rad, latitude extent mapped onto 2^32
    int64_t nbins;         // nring * m
    double sx32, sy32;     // fixed-point units per radian (lon, lat): 2^32 over a span >= wx / wy (target.cu)
};

constexpr int64_t kGraphMaxN = 1 << 21;   // auto: calls of up to this many samples are replayed as a CUDA graph
constexpr double kF32RadiusMax = 0.004;   // rad: largest support radius of the fp32 pair arithmetic (target.cu)

struct KernelParams {      // per-context constants of the pair arithmetic
    double sigma, radius;              // rad
    double inv2s2;                     // 1 / (2 sigma^2)
    double hav_max;                    // sin^2(R/2)
    float h4max;                       // 4 sin^2(R/2), rounded to fp32
    float k1, k2;                      // exponent = h4 * (k1 + k2 * h4): -log2e/(2 sigma^2) * (1, 1/12)
    // kernel function (hcgrid_set_kernel): 0 Gaussian, 1 tapered sinc, 2 elliptical Gaussian
    //   sinc(d / (b sigma)) exp(-(d / (a sigma))^2),  sinc(x) = sin(pi x) / (pi x)
    int ktype;
    double inv_a2s2, pi_bs;            // 1 / (a sigma)^2,  pi / (b sigma)
    float tg2, ts1;                    // fp32 path, from t = -exponent above = d^2 log2e / (2 sigma^2):
                                       // taper = ex2(-t * tg2), tg2 = 2 / a^2; sinc argument = ts1 * sqrt(t),
                                       // ts1 = pi sqrt(2 ln 2) / b
    // 2 elliptical Gaussian (reading c21): sigma along the axis at position angle PA (from north through
    //   east), ratio * sigma across it; exponent = d^2 / (2 sigma^2) + (d sin(beta - PA))^2 * ell_k
    double ell_k;                      // 1 / (2 (ratio sigma)^2) - 1 / (2 sigma^2)
    double ell_cp, ell_sp;             // cos PA, sin PA
    float ek2, ecp, esp;               // fp32 path: -log2e * ell_k, cos PA, sin PA
};

// ---------------------------------------------------------------- host-side helpers
struct DevBuf {
    void* p = nullptr;
    size_t cap = 0;
    cudaError_t ensure(size_t bytes) {
        if (bytes <= cap) return cudaSuccess;
        if (p) cudaFree(p);
        p = nullptr; cap = 0;
        size_t want = bytes + bytes / 8 + 256;
        cudaError_t e = cudaMalloc(&p, want);
        if (e == cudaSuccess) cap = want;
        return e;
    }
    void release() { if (p) cudaFree(p); p = nullptr; cap = 0; }
    template <class T> T* as() const { return reinterpret_cast<T*>(p); }
};

}  // namespace hcg

struct hcgrid_ctx {
    int device = 0;
    int precision = HCGRID_F32;
    int nside = 0;
    int num_sms = 148;
    hcg::KernelParams kp{};
    // options
    int opt_profile = 0, opt_subpix = -1000, opt_coarsen = 0, opt_coarsen_y = 0, opt_kernel = 0, opt_warps = 0, opt_split = 0, opt_preorder = 0;
    // target
    bool has_target = false;
    bool is_car = false;
    int64_t ncell = 0;
    int32_t nstrip = 0, strip_cells = 0, kmax = 0;
    bool small_series_ok = true;    // small-angle series valid over the whole target (R, longitude half-window <= 0.05 rad)
    bool f32_series_ok = true;      // ... and the fp32 pair arithmetic resolves the support boundary to 1e-9 rad (R <= kF32RadiusMax)
    double cell_width_sky = 0.0;    // min over strips of |du| cos(lat), rad (coarsening choice)
    hcg::Region region{};
    hcg::DevBuf d_strips, d_wins, d_winsf, d_rowsf, d_cell_lon, d_cell_lat;
    double car_u0 = 0.0, car_du = 0.0;   // plate-carree target: lon offset of column 0 / column step, rad
    double car_dlat = 0.0;               // row step, rad (signed)
    // the plate-carree target as the caller gave it, and the lookup-bin refinement chosen from the sample density
    // (refine_target_for_density: auto sub-pixel bits only, -1000 = not refined)
    int car_nx = 0, car_ny = 0;
    double car_lon0_deg = 0.0, car_lat0_deg = 0.0, car_dlon_deg = 0.0, car_dlat_deg = 0.0;
    int subpix_refined = -1000;
    // Guard of the counting pre-order against piled-up input: bins beyond kLongBin samples are ordered one block per
    // bin, which is slow when a large share of the samples sits in a few bins (a staring pointing).  Large calls copy
    // the number of such bins and the longest one to the host behind themselves; once a call has seen more than 64 of
    // them or one beyond 16 kLongBin samples, the following calls on this target take the radix sort (same S').
    int32_t* h_long = nullptr;           // pinned, mapped [2]: written by order_long_kernel's last block
    int32_t* h_long_dev = nullptr;       // its device address
    cudaEvent_t ev_long = nullptr;
    bool long_pending = false, force_radix = false;
    double dlmax = 0.0;                  // widest longitude half-window of a support disc, rad
    bool tile_ok = false;                // the tile kernel's preconditions hold for this target
    // per-call scratch
    hcg::DevBuf d_keys, d_keys_out, d_idx, d_idx_out, d_sort_tmp, d_bins, d_rec, d_misc, d_long, d_dirty, d_stat;
    hcg::DevBuf d_in_lon, d_in_lat, d_in_val, d_in_wgt, d_out_cube, d_out_w, d_out_cnt;  // *_host path
    // incremental gridding (hcgrid_accumulate / hcgrid_finalize): un-normalised sums over the batches so far
    hcg::DevBuf d_acc_cube, d_acc_w, d_acc_cnt, d_tmp_cube, d_tmp_w, d_tmp_cnt;
    bool raw_sums = false;          // the convolution kernels write sums instead of sums / W
    int acc_nchan = 0;              // channels of the running accumulation (0: none yet)
    int64_t acc_batches = 0;
    // last call (debug introspection)
    const double* last_lon = nullptr;
    const double* last_lat = nullptr;
    int64_t last_n = 0;
    cudaStream_t last_stream = nullptr;
    cudaStream_t st_copy = nullptr, st_comp = nullptr;   // hcgrid_grid_host pipeline (created on first use)
    cudaEvent_t ev_chunk[16] = {};
    int opt_host_chunks = 0;
    int opt_cells_as_grid = 1;           // HCGRID_OPT_CELLS_AS_GRID
    // Replay of repeated small calls (HCGRID_OPT_GRAPH): the kernels of one hcgrid_grid call as an instantiated CUDA
    // graph, keyed by everything a launch depends on; config_gen counts option / kernel / target changes.
    int opt_graph = -1;                  // -1 auto (inputs up to kGraphMaxN samples), 0 off, 1 on for any size
    uint64_t config_gen = 0;
    struct GraphKey {
        int64_t n; const void *lon, *lat, *values, *weights, *cube, *wmap, *counts; int32_t nchan; uint64_t gen;
        bool operator==(const GraphKey& o) const {
            return n == o.n && lon == o.lon && lat == o.lat && values == o.values && weights == o.weights && cube == o.cube &&
                   wmap == o.wmap && counts == o.counts && nchan == o.nchan && gen == o.gen;
        }
    };
    GraphKey graph_key{}, graph_seen{};  // key of the instantiated graph / of the last eager call
    bool graph_valid = false, graph_seen_valid = false;
    cudaGraphExec_t graph_exec = nullptr;
    hcgrid_stats graph_stats{};
    cudaStream_t st_cap = nullptr;       // capture happens here; the graph is launched into the caller's stream
    cudaEvent_t ev[8] = {};
    bool ev_valid = false;
    bool stat_hit = false, stat_pairs = false;   // d_stat[0] / d_stat[1] hold n_hit / n_pairs_tested of the last call
    hcgrid_stats stats{};
    std::string err;
};

namespace hcg {

// stage entry points (defined in target.cu / preorder.cu / convolve*.cu)
int build_target_car(hcgrid_ctx* c, int nx, int ny, double lon0, double lat0, double dlon, double dlat);
int build_target_cells(hcgrid_ctx* c, int64_t ncell, const double* lon, const double* lat, cudaStream_t st);
// Plate-carree targets with automatic sub-pixel bits: when the call brings more than 10 samples per lookup bin (the
// radix-sort regime) and finer bins (towards 4 per bin, up to 2^6 per pixel) bring that to 10 or less, the tables are rebuilt --
// the counting pre-order then applies and the search windows tighten.  Synchronises `st` and the device when it
// rebuilds (once per target and density class); returns HCGRID_OK and *rebuilt.
int refine_target_for_density(hcgrid_ctx* c, int64_t n, cudaStream_t st, bool* rebuilt);
int run_preorder(hcgrid_ctx* c, int64_t n, const double* lon, const double* lat, const float* values,
                 int nchan, const float* weights, cudaStream_t st);
int run_convolve(hcgrid_ctx* c, int64_t n, const float* values, int nchan, bool has_weights,
                 void* cube, void* wmap, int32_t* counts, cudaStream_t st);

int run_profile_stats(hcgrid_ctx* c, int32_t* counts, cudaStream_t st);

int fail(hcgrid_ctx* c, int code, const char* fmt, ...);
int cuda_fail(hcgrid_ctx* c, cudaError_t e, const char* what);

#define HCG_CUDA(c, call)                                              \
    do {                                                               \
        cudaError_t e_ = (call);                                       \
        if (e_ != cudaSuccess) return hcg::cuda_fail((c), e_, #call);  \
    } while (0)

}  // namespace hcg
