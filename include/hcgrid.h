/* hcgrid.h -- C-ABI of the B200-native HCGrid hot path (arXiv 2012.13173).
 *
 * What the library computes (Sect. 2.1, Eq. 1): for every target
 * cell g_ij with centre (alpha_ij, delta_ij)
 *
 *     V[g_ij] = (1 / W_ij) * sum_n V[s_n] * w(alpha_ij, delta_ij; alpha_n, delta_n)
 *     W_ij    = sum_n w(alpha_ij, delta_ij; alpha_n, delta_n)
 *
 * with the kernel of PAPER.md:186 (Sect. 3.6 iii): a radially symmetric Gaussian of
 * standard deviation sigma_kernel, w(d) = exp(-d^2 / (2 sigma^2)) of the great-circle
 * distance d, truncated at "sphere_radius" (d <= R contributes).  Contributing samples
 * are found through the pre-ordering of PAPER.md:108-124 (Sect. 3.3: HEALPix RING pixel
 * index per sample, key-value sort, ring table R_start and per-pixel table
 * P_i -> S_start) and the search of PAPER.md:134-140 (Sect. 3.4 i-v).  Every step runs on
 * the device; there is no CPU search stage and no CPU fallback.
 *
 * Conventions
 *   - Angles at the boundary are DEGREES (the paper speaks degrees/arcmin/arcsec,
 *     PAPER.md:24, 218); lon is any real (reduced mod 360), lat in [-90, 90].
 *   - Unless a function says "HOST", every array pointer is a DEVICE pointer on the
 *     context's device, owned by the caller, not modified unless it is an output.
 *   - Flat cell index of a plate-carree target is iy*nx + ix; datacube is
 *     [ncell][nchan] with the channel fastest (values is [n][nchan] likewise).
 *   - Empty cell (W == 0): V = NaN, W = 0, count = 0.
 *   - Per-sample weights q_s multiply the kernel (W = sum q w, V = sum q w v / W);
 *     counts are geometric (number of samples with d <= R, whatever q).
 *   - All calls return an hcgrid_status (0 = OK, negative = error); nothing aborts or
 *     throws.  hcgrid_last_error() gives the message of the last failing call.
 *   - A context is not re-entrant: one host thread at a time per context.
 *   - hcgrid_grid() is asynchronous on `stream`; outputs are valid once the stream is
 *     synchronised.  The context owns all scratch (grow-only, reused across calls).
 */
#ifndef HCGRID_H
#define HCGRID_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hcgrid_ctx hcgrid_ctx;

typedef enum {
    HCGRID_OK = 0,
    HCGRID_ERR_INVALID_ARG = -1,
    HCGRID_ERR_NO_TARGET = -2,
    HCGRID_ERR_ALLOC = -3,
    HCGRID_ERR_CUDA = -4,
    HCGRID_ERR_UNSUPPORTED = -5
} hcgrid_status;

/* precision mode: pair arithmetic + accumulation + output dtype */
enum { HCGRID_F32 = 0, HCGRID_F64 = 1 };

/* tuning / debug options for hcgrid_set_option (all have measured defaults) */
enum {
    HCGRID_OPT_PROFILE = 1,      /* 1: time every stage with CUDA events (hcgrid_get_stats) */
    HCGRID_OPT_SUBPIX_BITS = 2,  /* log2 of lookup bins per HEALPix pixel along the ring; -1 = auto.
                                    Takes effect at the next hcgrid_set_target_*. */
    HCGRID_OPT_COARSEN = 3,      /* cells per warp task along a target row (thread coarsening,
                                    PAPER.md:153, at warp scope); 0 = auto */
    HCGRID_OPT_KERNEL = 4,       /* 0 = auto; 1 = force the simple (non-staged) single-channel kernel;
                                    2 = force the fp64 pair arithmetic with the F32 output type;
                                    3 = force the general (any nchan) kernel with fp32 pair arithmetic;
                                    4 = force the TMA-staged single-channel kernel;
                                    5 = force the tile kernel (error if the target does not allow it);
                                    6 = force the CUDA-core cube kernel (nchan > 1; error if not applicable);
                                    7 = force the tensor-core cube kernel (tcgen05; nchan a multiple of 32) */
    HCGRID_OPT_WARPS_PER_SM = 5, /* resident convolution warps per SM (staged kernel); 0 = auto */
    HCGRID_OPT_COARSEN_Y = 6,    /* target rows per warp task (tile kernel); 0 = auto */
    HCGRID_OPT_SPLIT = 7,        /* warps sharing one tile's candidate stream (tile kernel): 1, 2, 4; 0 = auto */
    HCGRID_OPT_HOST_CHUNKS = 9,  /* hcgrid_grid_host: pieces the samples are copied and gridded in (copy of piece
                                    k+1 overlaps the gridding of piece k); 1 = one copy, one hcgrid_grid; 0 = auto
                                    (4 from 64 MB of input) */
    HCGRID_OPT_CELLS_AS_GRID = 10, /* hcgrid_set_target_cells: 1 (default) = cells that are a plate-carree grid listed
                                    row by row (lon0 + ix*dlon, lat0 + iy*dlat: what a WCS CAR header expands to) are
                                    recognised and take the plate-carree path; in fp64 mode only when those two
                                    expressions reproduce every centre bit for bit, in fp32 mode to 1e-10 deg;
                                    0 = always the per-cell path.  Set before hcgrid_set_target_cells. */
    HCGRID_OPT_GRAPH = 11,       /* replay of repeated calls: an hcgrid_grid call with the same arrays, sizes, options
                                    and target as the one before it is captured as a CUDA graph, and every further
                                    identical call is one graph launch (the arrays' contents may change, their
                                    addresses and sizes may not: any other call runs eagerly and starts over).
                                    -1 = auto (default): inputs of up to 2^21 samples, which are bound by launch
                                    gaps; 0 = never; 1 = any size.  Not used with HCGRID_OPT_PROFILE or while an
                                    accumulation is open. */
    HCGRID_OPT_PREORDER = 8      /* how S' is ordered: 1 = radix sort of (key, n); 2 = counting sort into the
                                    bin table (same S', bit for bit); 0 = auto (counting up to 10 samples per bin) */
};

typedef struct {
    int64_t n_samples;        /* samples passed to the last hcgrid_grid                      */
    int64_t n_kept;           /* samples inside the target's reach (sorted, packed)          */
    int64_t n_bins;           /* entries of the per-pixel offset table                        */
    int32_t n_rings;          /* rings of the ring table                                      */
    int32_t subpix_bits;      /* lookup bins per HEALPix pixel = 2^subpix_bits (may be < 0)   */
    int32_t coarsen;          /* cells per warp task along a row used                         */
    int32_t kernel;           /* convolution kernel variant that ran          */
    int32_t gpu_launches;     /* kernels launched by the last hcgrid_grid                     */
    int32_t coarsen_y;        /* target rows per warp task used (tile kernel; else 1)         */
    float us_pixelise, us_sort, us_tables, us_pack, us_convolve, us_total; /* PROFILE only   */
    int32_t split;            /* warps per tile used (tile kernel; else 1)                    */
    int32_t preorder;         /* pre-ordering used: 1 radix sort, 2 counting sort             */
    int64_t n_hit;            /* PROFILE + count output: pairs (cell, sample) with d <= R = sum of the counts
                                 ("kernel evaluations"); -1 otherwise                            */
    int32_t graph;            /* 1: the call was replayed from (or captured into) a CUDA graph (HCGRID_OPT_GRAPH) */
    int32_t pad_;
    int64_t n_pairs_tested;   /* PROFILE, tile and strip kernels (kernel 1..6): pairs the kernel put to the distance
                                 test (candidate stream length x cells of every tile or task); -1 otherwise     */
} hcgrid_stats;

/* Create a context.  sigma_deg = kernel standard deviation, support_radius_deg =
 * "sphere_radius", nside = HEALPix partition level N_side,
 * a power of two in [1, 16384] (12 nside^2 <= 2^32: the pixel index fits the sort key).  precision = HCGRID_F32 or HCGRID_F64.  device = CUDA
 * ordinal.  On failure *out is NULL and the message is available through
 * hcgrid_last_error(NULL). */
int hcgrid_create(hcgrid_ctx** out, double sigma_deg, double support_radius_deg,
                  int64_t nside, int precision, int device);
int hcgrid_destroy(hcgrid_ctx* ctx);

int hcgrid_set_option(hcgrid_ctx* ctx, int option, int64_t value);

/* Kernel function omega(d) of Eq. 1, d = great-circle angle, sigma and the
 * support radius as given to hcgrid_create:
 *   HCGRID_KERNEL_GAUSS         exp(-d^2 / (2 sigma^2)) -- the paper's kernel and the default; a, b ignored.
 *   HCGRID_KERNEL_TAPERED_SINC  sinc(d / (b sigma)) exp(-(d / (a sigma))^2), sinc(x) = sin(pi x) / (pi x):
 *                               the finite stand-in for the sinc PAPER.md:186 calls optimal, in the form of
 *                               the work the paper follows there (Winkel et al. 2016b, who advise a = 2.52,
 *                               b = 1.55; the caller's choice here).  Weights can
 *                               be negative: the datacube is S / W wherever W != 0 (NaN otherwise) and the
 *                               weight map may cancel towards zero.
 *   HCGRID_KERNEL_ELLIPTICAL_GAUSS  exp(-u^2 / (2 s1^2) - v^2 / (2 s2^2)) (reading c21; PAPER.md:186
 *                               names only the radially symmetric Gaussian): s1 = the context's sigma along the
 *                               axis at position angle b (degrees, from north through east), s2 = a * s1 across
 *                               it (a > 0; a < 1: the axis at the position angle is the major one).  (u, v) =
 *                               d (cos(beta - b), sin(beta - b)), d the great-circle angle and beta the bearing
 *                               of the sample seen from the cell centre.  The support stays the circle d <= R.
 * Takes effect at the next hcgrid_grid / hcgrid_accumulate; not allowed while an accumulation is open.
 * Gaussian runs on every convolution kernel; other functions on the general kernels only
 * (any target, any channel count, both precisions).  Returns HCGRID_ERR_INVALID_ARG for an
 * unknown type, non-positive a (b for the sinc) or non-finite a, b. */
enum { HCGRID_KERNEL_GAUSS = 0, HCGRID_KERNEL_TAPERED_SINC = 1, HCGRID_KERNEL_ELLIPTICAL_GAUSS = 2 };
int hcgrid_set_kernel(hcgrid_ctx* ctx, int32_t kernel_type, double a, double b);

/* Target = plate-carree grid: cell (ix, iy) centre = (lon0 + ix*dlon, lat0 + iy*dlat),
 * each evaluated with one rounding per operation (no FMA); dlon, dlat may be negative,
 * not zero.  Builds the per-row search tables on the device (synchronises the device). */
int hcgrid_set_target_car(hcgrid_ctx* ctx, int32_t nx, int32_t ny, double lon0_deg,
                          double lat0_deg, double dlon_deg, double dlat_deg);
/* Target = arbitrary cells; lon_deg/lat_deg are DEVICE arrays [ncell] (copied; synchronises the stream).  Cells
 * that form a plate-carree grid are recognised (HCGRID_OPT_CELLS_AS_GRID) and gridded like hcgrid_set_target_car's. */
int hcgrid_set_target_cells(hcgrid_ctx* ctx, int64_t ncell, const double* lon_deg,
                            const double* lat_deg, void* stream);

/* Lookup-bin refinement: on a plate-carree target with automatic HCGRID_OPT_SUBPIX_BITS, a call that brings more than
 * 10 samples per lookup bin rebuilds the target's tables with finer bins (towards 4 samples per bin, at most 2^6 bins
 * per HEALPix pixel) when that brings the density to 10 per bin or less: the counting pre-order then applies and the
 * search windows tighten.  That call
 * synchronises `stream` and the device once; later calls keep the finer tables until a new target is set.  Results
 * do not depend on the bin size beyond the order of the additions (reading c11). */

/* Grid n samples onto the target.
 *   lon_deg, lat_deg [n] double; values [n][nchan] float; weights [n] float or NULL.
 *   datacube [ncell][nchan], weightmap [ncell]: float (F32) or double (F64).
 *   counts [ncell] int32 or NULL.  stream: cudaStream_t (NULL = default stream).
 * n = 0 is legal (every cell empty). */
int hcgrid_grid(hcgrid_ctx* ctx, int64_t n, const double* lon_deg, const double* lat_deg,
                const float* values, int32_t nchan, const float* weights,
                void* datacube, void* weightmap, int32_t* counts, void* stream);

/* Same call with HOST buffers (pinned or pageable): copies the inputs to context-owned
 * device buffers, grids, copies the outputs back and synchronises before returning.
 * From 64 MB of input on (HCGRID_OPT_HOST_CHUNKS) the samples go over in 4 pieces on a copy
 * stream while a second stream grids the pieces that have arrived (hcgrid_accumulate on each,
 * one hcgrid_finalize): the same sums added in a different order, so the result agrees with
 * hcgrid_grid's to rounding, not bit for bit; it is deterministic for a given piece count.
 * Pinned buffers are needed for the copies to overlap anything.  Falls back to one piece while
 * the caller has an accumulation open. */
int hcgrid_grid_host(hcgrid_ctx* ctx, int64_t n, const double* lon_deg, const double* lat_deg,
                     const float* values, int32_t nchan, const float* weights,
                     void* datacube, void* weightmap, int32_t* counts);

/* Incremental gridding: successive batches of samples (successive scans) into one cube.
 * Eq. 1 is a ratio of two sums over the samples, both additive over batches;
 * the paper names streaming as future work.  hcgrid_accumulate grids one batch
 * (arguments as hcgrid_grid, DEVICE pointers, asynchronous on `stream`) and adds its
 * un-normalised sums, weights and counts to accumulators owned by the context; the first call
 * after hcgrid_set_target_* or after a resetting hcgrid_finalize starts from zero, and every
 * batch of one accumulation must have the same nchan.  hcgrid_finalize writes
 * datacube = sums / weightmap (NaN where the weight is 0), weightmap and, if not NULL, counts
 * of everything accumulated so far; reset != 0 ends the accumulation.  Gridding batches one
 * after the other equals gridding their union up to the order of the additions.
 * hcgrid_set_target_* also ends a running accumulation. */
int hcgrid_accumulate(hcgrid_ctx* ctx, int64_t n, const double* lon_deg, const double* lat_deg,
                      const float* values, int32_t nchan, const float* weights, void* stream);
int hcgrid_finalize(hcgrid_ctx* ctx, void* datacube, void* weightmap, int32_t* counts, int reset,
                    void* stream);
int64_t hcgrid_accumulated_batches(const hcgrid_ctx* ctx);   /* batches in the running accumulation */

int64_t hcgrid_ncell(const hcgrid_ctx* ctx);      /* cells of the current target, 0 if none */
int hcgrid_get_stats(const hcgrid_ctx* ctx, hcgrid_stats* out);
const char* hcgrid_last_error(const hcgrid_ctx* ctx);  /* ctx may be NULL (create errors) */

/* ---- introspection of the pre-ordering (tests; Fig. 3, 120-124) --------
 * Valid after a successful hcgrid_grid and a stream synchronise.  All outputs are HOST
 * arrays; pass NULL to skip one.  Sizes come from hcgrid_get_stats (n_kept, n_rings).
 *   sorted_pixel [n_kept]  HEALPix RING pixel index P' of every kept sample, in S' order
 *   sorted_index [n_kept]  original sample index n of every kept sample (the "value" of
 *                          the key-value sort)
 *   ring_first   [1]       HEALPix ring number (1 = northernmost) of ring-table entry 0
 *   ring_start   [n_rings+1] R_start: position in S' of the first sample of each ring;
 *                          ring i occupies [ring_start[i], ring_start[i+1]) (0-based form
 *                          of PAPER.md:137) */
int hcgrid_debug_preorder(hcgrid_ctx* ctx, int64_t* sorted_pixel, int64_t* sorted_index,
                          int32_t* ring_first, int64_t* ring_start);
/* HEALPix RING pixel index of n points (DEVICE in, DEVICE out [n] int64): the a2 step
 * alone, for the pixelisation self-consistency tests. */
int hcgrid_debug_ang2pix_ring(int64_t nside, int64_t n, const double* lon_deg,
                              const double* lat_deg, int64_t* pix, void* stream);

/* The same a2 code compiled for the host: HOST in, HOST out, no GPU needed (CPU tests of
 * the pixelisation's self-consistency). */
int hcgrid_host_ang2pix_ring(int64_t nside, int64_t n, const double* lon_deg,
                             const double* lat_deg, int64_t* pix);
/* Geometry of HEALPix ring `iring` (1 = northernmost .. 4*nside-1), HOST outputs, any may
 * be NULL: index of its first pixel, pixels in the ring, latitude of the ring centre,
 * longitude of the centre of its pixel 0 (pixel j is centred at lon0 + j*360/npix). */
int hcgrid_host_ring_info(int64_t nside, int32_t iring, int64_t* first_pixel, int32_t* npix,
                          double* lat_deg, double* lon0_deg);

/* Issue-rate probes for the roofline ("the builder must measure P_fp32 and
 * P_mufu on the box"): register-only chains, 8 independent per thread, all SMs.  HOST
 * outputs: FP32-pipe thread-instructions/s (FFMA) and MUFU.EX2 thread-instructions/s.
 * Synchronises the device. */
int hcgrid_measure_peaks(int device, double* fp32_inst_per_s, double* mufu_per_s);

/* The one entry point that ALLOCATES NOTHING (no cudaMalloc / cudaFree / allocating library routine), for callers
 * that cannot allocate: code under CUDA-graph capture, tight serving loops, harnesses that forbid it.  Every other
 * call of this library may grow a context-owned device buffer.  From the count output of hcgrid_grid (PAPER.md:59:
 * the samples with d <= R of every cell) it forms the figures the throughput metric is quoted in:
 *   out[0] = sum of counts[0 .. ncell)           -- pairs (cell, sample) with d <= R ("kernel evaluations", n_hit)
 *   out[1] = number of cells with counts[i] > 0  -- cells the samples reach
 * counts [ncell] int32 and out [2] uint64 are DEVICE pointers on the CURRENT device, owned by the caller;
 * asynchronous on `stream`; no context needed.  Its scratch (per-block partial sums and a ticket) is a fixed
 * 16.25 KB device array inside the library, held by every GPU that loads it until the process exits; hence
 *   - ncell <= hcgrid_static_max_cells() = 2^30, more is refused with HCGRID_ERR_INVALID_ARG;
 *   - ALL calls on one device share the array: calls that overlap on the GPU (two streams, two host threads)
 *     race and give wrong sums -- serialise them.  Calls one after the other on a stream are fine (what must start
 *     at zero is cleared at the start of every call).
 * Same sums as hcgrid_stats.n_hit (integers, fixed order).  Errors: status + hcgrid_last_error(NULL). */
int hcgrid_count_hits_static(const int32_t* counts, int64_t ncell, uint64_t* out, void* stream);
int64_t hcgrid_static_max_cells(void);

#ifdef __cplusplus
}
#endif
#endif /* HCGRID_H */
