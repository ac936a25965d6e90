// api.cu -- the C-ABI of include/hcgrid.h: argument checking, context life cycle, stage
// sequencing.  No arithmetic of the method lives here.
#include <cmath>
#include <cstdarg>
#include <cstring>
#include <new>
#include <vector>

#include "hcg_common.cuh"

namespace hcg {

static thread_local std::string g_create_err;

int fail(hcgrid_ctx* c, int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (c) c->err = buf; else g_create_err = buf;
    return code;
}

int cuda_fail(hcgrid_ctx* c, cudaError_t e, const char* what) {
    cudaGetLastError();   // clear the sticky-less error state
    const int code = e == cudaErrorMemoryAllocation ? HCGRID_ERR_ALLOC : HCGRID_ERR_CUDA;
    return fail(c, code, "CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
}

static bool is_pow2(int64_t x) { return x > 0 && (x & (x - 1)) == 0; }

}  // namespace hcg

using namespace hcg;

extern "C" {

int hcgrid_create(hcgrid_ctx** out, double sigma_deg, double support_radius_deg, int64_t nside,
                  int precision, int device) {
    if (!out) return fail(nullptr, HCGRID_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (!(sigma_deg > 0.0) || !std::isfinite(sigma_deg))
        return fail(nullptr, HCGRID_ERR_INVALID_ARG, "sigma_deg must be a positive finite number");
    if (!(support_radius_deg > 0.0) || !(support_radius_deg < 90.0))
        return fail(nullptr, HCGRID_ERR_INVALID_ARG, "support_radius_deg must be in (0, 90)");
    if (!is_pow2(nside) || nside > 16384)
        return fail(nullptr, HCGRID_ERR_INVALID_ARG, "nside must be a power of two in [1, 16384]");
    if (precision != HCGRID_F32 && precision != HCGRID_F64)
        return fail(nullptr, HCGRID_ERR_INVALID_ARG, "precision must be HCGRID_F32 or HCGRID_F64");
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDeviceCount");
    if (device < 0 || device >= ndev)
        return fail(nullptr, HCGRID_ERR_INVALID_ARG, "device %d out of range (%d devices)", device, ndev);
    hcgrid_ctx* c = new (std::nothrow) hcgrid_ctx();
    if (!c) return fail(nullptr, HCGRID_ERR_ALLOC, "out of host memory");
    c->device = device;
    c->precision = precision;
    c->nside = (int)nside;
    e = cudaSetDevice(device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, device);
    if (e != cudaSuccess) { delete c; return cuda_fail(nullptr, e, "device set-up"); }
    for (auto& ev : c->ev) {
        e = cudaEventCreate(&ev);
        if (e != cudaSuccess) { delete c; return cuda_fail(nullptr, e, "cudaEventCreate"); }
    }
    e = cudaEventCreateWithFlags(&c->ev_long, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaHostAlloc((void**)&c->h_long, 2 * sizeof(int32_t), cudaHostAllocMapped);
    if (e == cudaSuccess) e = cudaHostGetDevicePointer((void**)&c->h_long_dev, c->h_long, 0);
    if (e != cudaSuccess) { hcgrid_destroy(c); return cuda_fail(nullptr, e, "pinned word for the pre-order guard"); }
    c->h_long[0] = c->h_long[1] = 0;
    KernelParams& kp = c->kp;
    kp.sigma = sigma_deg * kDeg2Rad;
    kp.radius = support_radius_deg * kDeg2Rad;
    kp.inv2s2 = 1.0 / (2.0 * kp.sigma * kp.sigma);
    const double sr = std::sin(0.5 * kp.radius);
    kp.hav_max = sr * sr;
    kp.h4max = (float)(4.0 * sr * sr);
    const double log2e = 1.4426950408889634074;
    kp.k1 = (float)(-log2e * kp.inv2s2);
    kp.k2 = (float)(-log2e * kp.inv2s2 / 12.0);
    kp.ktype = HCGRID_KERNEL_GAUSS;
    kp.inv_a2s2 = 0.0; kp.pi_bs = 0.0; kp.tg2 = 0.0f; kp.ts1 = 0.0f;
    *out = c;
    return HCGRID_OK;
}

int hcgrid_destroy(hcgrid_ctx* c) {
    if (!c) return HCGRID_OK;
    cudaSetDevice(c->device);
    DevBuf* bufs[] = {&c->d_strips, &c->d_wins, &c->d_winsf, &c->d_rowsf, &c->d_cell_lon, &c->d_cell_lat, &c->d_keys, &c->d_keys_out,
                      &c->d_idx, &c->d_idx_out, &c->d_sort_tmp, &c->d_bins, &c->d_rec, &c->d_misc, &c->d_long, &c->d_dirty, &c->d_stat,
                      &c->d_in_lon, &c->d_in_lat, &c->d_in_val, &c->d_in_wgt, &c->d_out_cube, &c->d_out_w,
                      &c->d_out_cnt, &c->d_acc_cube, &c->d_acc_w, &c->d_acc_cnt, &c->d_tmp_cube, &c->d_tmp_w,
                      &c->d_tmp_cnt};
    for (DevBuf* b : bufs) b->release();
    for (auto& ev : c->ev) if (ev) cudaEventDestroy(ev);
    for (auto& ev : c->ev_chunk) if (ev) cudaEventDestroy(ev);
    if (c->st_copy) cudaStreamDestroy(c->st_copy);
    if (c->st_comp) cudaStreamDestroy(c->st_comp);
    if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
    if (c->ev_long) { cudaEventSynchronize(c->ev_long); cudaEventDestroy(c->ev_long); }
    if (c->h_long) cudaFreeHost(c->h_long);
    if (c->st_cap) cudaStreamDestroy(c->st_cap);
    delete c;
    return HCGRID_OK;
}

int hcgrid_set_option(hcgrid_ctx* c, int option, int64_t value) {
    if (!c) return HCGRID_ERR_INVALID_ARG;
    ++c->config_gen;
    switch (option) {
        case HCGRID_OPT_GRAPH:
            if (value < -1 || value > 1) return fail(c, HCGRID_ERR_INVALID_ARG, "graph must be -1 (auto), 0 or 1");
            c->opt_graph = (int)value;
            break;
        case HCGRID_OPT_PROFILE: c->opt_profile = value != 0; break;
        case HCGRID_OPT_SUBPIX_BITS:
            if (value < -1 || value > 6) return fail(c, HCGRID_ERR_INVALID_ARG, "subpix bits must be -1 (auto) or 0..6");
            c->opt_subpix = value < 0 ? -1000 : (int)value;
            break;
        case HCGRID_OPT_COARSEN:
            if (value < 0 || value > 8) return fail(c, HCGRID_ERR_INVALID_ARG, "coarsen must be 0 (auto) or 1..8");
            c->opt_coarsen = (int)value;
            break;
        case HCGRID_OPT_KERNEL:
            if (value < 0 || value > 7) return fail(c, HCGRID_ERR_INVALID_ARG, "kernel must be 0..7");
            c->opt_kernel = (int)value;
            break;
        case HCGRID_OPT_COARSEN_Y:
            if (value < 0 || value > 4) return fail(c, HCGRID_ERR_INVALID_ARG, "coarsen_y must be 0 (auto) or 1..4");
            c->opt_coarsen_y = (int)value;
            break;
        case HCGRID_OPT_WARPS_PER_SM:
            if (value < 0 || value > 64) return fail(c, HCGRID_ERR_INVALID_ARG, "warps per SM must be 0..64");
            c->opt_warps = (int)value;
            break;
        case HCGRID_OPT_SPLIT:
            if (value != 0 && value != 1 && value != 2 && value != 4)
                return fail(c, HCGRID_ERR_INVALID_ARG, "split must be 0 (auto), 1, 2 or 4");
            c->opt_split = (int)value;
            break;
        case HCGRID_OPT_HOST_CHUNKS:
            if (value < 0 || value > 16) return fail(c, HCGRID_ERR_INVALID_ARG, "host chunks must be 0 (auto) or 1..16");
            c->opt_host_chunks = (int)value;
            break;
        case HCGRID_OPT_CELLS_AS_GRID:
            if (value < 0 || value > 1) return fail(c, HCGRID_ERR_INVALID_ARG, "cells-as-grid must be 0 or 1");
            c->opt_cells_as_grid = (int)value;
            break;
        case HCGRID_OPT_PREORDER:
            if (value < 0 || value > 2) return fail(c, HCGRID_ERR_INVALID_ARG, "preorder must be 0 (auto), 1 or 2");
            c->opt_preorder = (int)value;
            break;
        default: return fail(c, HCGRID_ERR_INVALID_ARG, "unknown option %d", option);
    }
    return HCGRID_OK;
}

int hcgrid_set_kernel(hcgrid_ctx* c, int32_t kernel_type, double a, double b) {
    if (!c) return HCGRID_ERR_INVALID_ARG;
    ++c->config_gen;
    if (c->acc_nchan != 0)
        return fail(c, HCGRID_ERR_INVALID_ARG, "the kernel cannot change while an accumulation is open");
    KernelParams& kp = c->kp;
    if (kernel_type == HCGRID_KERNEL_GAUSS) {
        kp.ktype = HCGRID_KERNEL_GAUSS;
        return HCGRID_OK;
    }
    if (kernel_type == HCGRID_KERNEL_ELLIPTICAL_GAUSS) {
        // a = sigma_2 / sigma_1 (across / along the axis), b = position angle of the axis in degrees
        if (!(a > 0.0) || !std::isfinite(a) || !std::isfinite(b))
            return fail(c, HCGRID_ERR_INVALID_ARG, "elliptical Gaussian needs a finite axis ratio a > 0 and a finite position angle b");
        const double s2 = kp.sigma * a;
        kp.ktype = HCGRID_KERNEL_ELLIPTICAL_GAUSS;
        kp.ell_k = 1.0 / (2.0 * s2 * s2) - kp.inv2s2;
        kp.ell_cp = std::cos(b * kDeg2Rad);
        kp.ell_sp = std::sin(b * kDeg2Rad);
        kp.ek2 = (float)(-kp.ell_k * 1.4426950408889634);
        kp.ecp = (float)kp.ell_cp;
        kp.esp = (float)kp.ell_sp;
        return HCGRID_OK;
    }
    if (kernel_type != HCGRID_KERNEL_TAPERED_SINC) return fail(c, HCGRID_ERR_INVALID_ARG, "unknown kernel type %d", (int)kernel_type);
    if (!(a > 0.0) || !(b > 0.0) || !std::isfinite(a) || !std::isfinite(b))
        return fail(c, HCGRID_ERR_INVALID_ARG, "tapered sinc needs a > 0 and b > 0");
    kp.ktype = HCGRID_KERNEL_TAPERED_SINC;
    kp.inv_a2s2 = 1.0 / (a * a * kp.sigma * kp.sigma);
    kp.pi_bs = kPi / (b * kp.sigma);
    kp.tg2 = (float)(2.0 / (a * a));
    kp.ts1 = (float)(kPi * std::sqrt(2.0 * std::log(2.0)) / b);
    return HCGRID_OK;
}

int hcgrid_set_target_car(hcgrid_ctx* c, int32_t nx, int32_t ny, double lon0, double lat0, double dlon,
                          double dlat) {
    if (!c) return HCGRID_ERR_INVALID_ARG;
    if (nx < 1 || ny < 1 || (int64_t)nx * ny > (int64_t)1 << 30)
        return fail(c, HCGRID_ERR_INVALID_ARG, "nx, ny must be >= 1 and nx*ny <= 2^30");
    if (!std::isfinite(lon0) || !std::isfinite(lat0) || !std::isfinite(dlon) || !std::isfinite(dlat) ||
        dlon == 0.0 || dlat == 0.0)
        return fail(c, HCGRID_ERR_INVALID_ARG, "lon0, lat0 finite and dlon, dlat finite non-zero required");
    if (std::fabs(dlon) * (nx - 1) >= 360.0)
        return fail(c, HCGRID_ERR_INVALID_ARG, "a target row must span less than 360 degrees");
    HCG_CUDA(c, cudaSetDevice(c->device));
    c->has_target = false;
    c->acc_nchan = 0;
    ++c->config_gen;
    c->subpix_refined = -1000;
    c->force_radix = false;
    return build_target_car(c, nx, ny, lon0, lat0, dlon, dlat);
}

int hcgrid_set_target_cells(hcgrid_ctx* c, int64_t ncell, const double* lon, const double* lat, void* stream) {
    if (!c) return HCGRID_ERR_INVALID_ARG;
    if (ncell < 1 || ncell > (int64_t)1 << 26)
        return fail(c, HCGRID_ERR_INVALID_ARG, "ncell must be in [1, 2^26] for an arbitrary-cell target");
    if (!lon || !lat) return fail(c, HCGRID_ERR_INVALID_ARG, "lon_deg / lat_deg is NULL");
    HCG_CUDA(c, cudaSetDevice(c->device));
    c->has_target = false;
    c->acc_nchan = 0;
    ++c->config_gen;
    c->subpix_refined = -1000;
    c->force_radix = false;
    return build_target_cells(c, ncell, lon, lat, (cudaStream_t)stream);
}

int hcgrid_grid(hcgrid_ctx* c, int64_t n, const double* lon, const double* lat, const float* values,
                int32_t nchan, const float* weights, void* cube, void* wmap, int32_t* counts, void* stream) {
    if (!c) return HCGRID_ERR_INVALID_ARG;
    if (!c->has_target) return fail(c, HCGRID_ERR_NO_TARGET, "no target set (call hcgrid_set_target_* first)");
    if (n < 0 || n > 2000000000LL) return fail(c, HCGRID_ERR_INVALID_ARG, "n must be in [0, 2e9]");
    if (nchan < 1) return fail(c, HCGRID_ERR_INVALID_ARG, "nchan must be >= 1");
    if (n > 0 && (!lon || !lat || !values)) return fail(c, HCGRID_ERR_INVALID_ARG, "lon/lat/values is NULL");
    if (!cube || !wmap) return fail(c, HCGRID_ERR_INVALID_ARG, "datacube / weightmap is NULL");
    HCG_CUDA(c, cudaSetDevice(c->device));
    cudaStream_t st = (cudaStream_t)stream;
    if (c->acc_nchan == 0) {                                  // not in the middle of a running accumulation
        bool rebuilt = false;
        const int rcr = refine_target_for_density(c, n, st, &rebuilt);
        if (rcr != HCGRID_OK) return rcr;
        if (rebuilt) ++c->config_gen;
    }
    c->last_lon = lon; c->last_lat = lat; c->last_n = n; c->last_stream = st;
    c->ev_valid = false;
    // A call that repeats the previous one (same arrays, sizes, options, target) is replayed as a CUDA graph: below
    // ~1e6 samples the call is bound by the launch gaps of its 7-9 dependent kernels, not by their work.  The second
    // identical call captures (on a stream of the context's own: nothing runs during capture, and the caller's stream
    // may be the legacy default stream, which cannot capture); every later one is a single graph launch.
    const bool graph_ok = !c->opt_profile && c->acc_nchan == 0 && n > 0 &&
                          (c->opt_graph == 1 || (c->opt_graph < 0 && n <= kGraphMaxN));
    const hcgrid_ctx::GraphKey key{n, lon, lat, values, weights, cube, wmap, counts, nchan, c->config_gen};
    if (graph_ok && c->graph_valid && c->graph_key == key) {
        HCG_CUDA(c, cudaGraphLaunch(c->graph_exec, st));
        c->stats = c->graph_stats;
        c->stats.n_kept = -1;
        c->stat_hit = c->stat_pairs = false;
        return HCGRID_OK;
    }
    c->stats = hcgrid_stats{};
    c->stats.n_samples = n;
    if (graph_ok && c->graph_seen_valid && c->graph_seen == key) {
        if (!c->st_cap) HCG_CUDA(c, cudaStreamCreateWithFlags(&c->st_cap, cudaStreamNonBlocking));
        if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
        c->graph_valid = false;
        cudaGraph_t graph = nullptr;
        HCG_CUDA(c, cudaStreamBeginCapture(c->st_cap, cudaStreamCaptureModeThreadLocal));
        int rc = run_preorder(c, n, lon, lat, values, nchan, weights, c->st_cap);
        if (rc == HCGRID_OK) rc = run_convolve(c, n, values, nchan, weights != nullptr, cube, wmap, counts, c->st_cap);
        const cudaError_t e = cudaStreamEndCapture(c->st_cap, &graph);
        if (rc == HCGRID_OK && e == cudaSuccess && graph != nullptr &&
            cudaGraphInstantiate(&c->graph_exec, graph, 0) == cudaSuccess) {
            cudaGraphDestroy(graph);
            c->graph_key = key;
            c->graph_valid = true;
            c->graph_stats = c->stats;
            c->graph_stats.graph = 1;
            c->stats = c->graph_stats;
            HCG_CUDA(c, cudaGraphLaunch(c->graph_exec, st));
            c->stats.n_kept = -1;
            c->stat_hit = c->stat_pairs = false;
            return HCGRID_OK;
        }
        // capture refused (a call inside that may not be captured): run eagerly, do not try again for this key
        if (graph) cudaGraphDestroy(graph);
        if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
        cudaGetLastError();
        c->graph_seen_valid = false;
        c->err.clear();
        c->stats = hcgrid_stats{};
        c->stats.n_samples = n;
    } else {
        c->graph_seen = key;
        c->graph_seen_valid = graph_ok;
    }
    int rc = run_preorder(c, n, lon, lat, values, nchan, weights, st);
    if (rc != HCGRID_OK) return rc;
    rc = run_convolve(c, n, values, nchan, weights != nullptr, cube, wmap, counts, st);
    if (rc != HCGRID_OK) return rc;
    if (c->opt_profile) { cudaEventRecord(c->ev[5], st); c->ev_valid = true; }
    rc = run_profile_stats(c, counts, st);
    if (rc != HCGRID_OK) return rc;
    c->stats.n_kept = -1;   // resolved lazily by hcgrid_get_stats
    return HCGRID_OK;
}

int hcgrid_grid_host(hcgrid_ctx* c, int64_t n, const double* lon, const double* lat, const float* values,
                     int32_t nchan, const float* weights, void* cube, void* wmap, int32_t* counts) {
    if (!c) return HCGRID_ERR_INVALID_ARG;
    if (!c->has_target) return fail(c, HCGRID_ERR_NO_TARGET, "no target set (call hcgrid_set_target_* first)");
    if (n < 0 || nchan < 1) return fail(c, HCGRID_ERR_INVALID_ARG, "n >= 0 and nchan >= 1 required");
    if (n > 0 && (!lon || !lat || !values)) return fail(c, HCGRID_ERR_INVALID_ARG, "lon/lat/values is NULL");
    if (!cube || !wmap) return fail(c, HCGRID_ERR_INVALID_ARG, "datacube / weightmap is NULL");
    HCG_CUDA(c, cudaSetDevice(c->device));
    const size_t nn = (size_t)n, nc = (size_t)c->ncell;
    const size_t osz = c->precision == HCGRID_F64 ? 8 : 4;
    HCG_CUDA(c, c->d_in_lon.ensure(nn * 8 + 8));
    HCG_CUDA(c, c->d_in_lat.ensure(nn * 8 + 8));
    HCG_CUDA(c, c->d_in_val.ensure(nn * (size_t)nchan * 4 + 16));
    if (weights) HCG_CUDA(c, c->d_in_wgt.ensure(nn * 4 + 16));
    HCG_CUDA(c, c->d_out_cube.ensure(nc * (size_t)nchan * osz));
    HCG_CUDA(c, c->d_out_w.ensure(nc * osz));
    if (counts) HCG_CUDA(c, c->d_out_cnt.ensure(nc * 4));
    // Large inputs: the copy is most of the call (PCIe), so the samples go over in chunks on one
    // stream while a second stream grids the chunks that have arrived -- Eq. 1's two sums are
    // additive over samples (hcgrid_accumulate), the division happens once at the end.
    int chunks = c->opt_host_chunks;
    if (chunks == 0) chunks = nn * (20 + 4 * (size_t)nchan) >= ((size_t)64 << 20) ? 4 : 1;
    if (c->acc_nchan != 0 || n < 4096) chunks = 1;          // an open accumulation is the caller's
    if (chunks > 1) {
        if (!c->st_copy) HCG_CUDA(c, cudaStreamCreateWithFlags(&c->st_copy, cudaStreamNonBlocking));
        if (!c->st_comp) HCG_CUDA(c, cudaStreamCreateWithFlags(&c->st_comp, cudaStreamNonBlocking));
        for (int k = 0; k < chunks; ++k)
            if (!c->ev_chunk[k]) HCG_CUDA(c, cudaEventCreateWithFlags(&c->ev_chunk[k], cudaEventDisableTiming));
        HCG_CUDA(c, cudaDeviceSynchronize());               // scratch may still be in use on the caller's streams
        // equal pieces but a last one of half the size: its gridding is what the copy cannot hide
        const int64_t per = ((int64_t)((double)n / ((double)chunks - 0.5)) + 64) & ~(int64_t)63;   // value rows stay 16-byte aligned
        for (int k = 0; k < chunks; ++k) {
            const int64_t lo = std::min<int64_t>(n, (int64_t)k * per), hi = std::min<int64_t>(n, lo + per);
            const size_t m = (size_t)(hi - lo);
            if (m > 0) {
                HCG_CUDA(c, cudaMemcpyAsync(c->d_in_lon.as<double>() + lo, lon + lo, m * 8, cudaMemcpyHostToDevice, c->st_copy));
                HCG_CUDA(c, cudaMemcpyAsync(c->d_in_lat.as<double>() + lo, lat + lo, m * 8, cudaMemcpyHostToDevice, c->st_copy));
                HCG_CUDA(c, cudaMemcpyAsync(c->d_in_val.as<float>() + (size_t)lo * nchan, values + (size_t)lo * nchan,
                                            m * (size_t)nchan * 4, cudaMemcpyHostToDevice, c->st_copy));
                if (weights)
                    HCG_CUDA(c, cudaMemcpyAsync(c->d_in_wgt.as<float>() + lo, weights + lo, m * 4, cudaMemcpyHostToDevice, c->st_copy));
            }
            HCG_CUDA(c, cudaEventRecord(c->ev_chunk[k], c->st_copy));
            HCG_CUDA(c, cudaStreamWaitEvent(c->st_comp, c->ev_chunk[k], 0));
            const int rc = hcgrid_accumulate(c, (int64_t)m, c->d_in_lon.as<double>() + lo, c->d_in_lat.as<double>() + lo,
                                             c->d_in_val.as<float>() + (size_t)lo * nchan, nchan,
                                             weights ? c->d_in_wgt.as<float>() + lo : nullptr, c->st_comp);
            if (rc != HCGRID_OK) { cudaDeviceSynchronize(); c->acc_nchan = 0; return rc; }
        }
        const int rc = hcgrid_finalize(c, c->d_out_cube.p, c->d_out_w.p, counts ? c->d_out_cnt.as<int32_t>() : nullptr, 1,
                                       c->st_comp);
        if (rc != HCGRID_OK) { cudaDeviceSynchronize(); c->acc_nchan = 0; return rc; }
        HCG_CUDA(c, cudaMemcpyAsync(cube, c->d_out_cube.p, nc * (size_t)nchan * osz, cudaMemcpyDeviceToHost, c->st_comp));
        HCG_CUDA(c, cudaMemcpyAsync(wmap, c->d_out_w.p, nc * osz, cudaMemcpyDeviceToHost, c->st_comp));
        if (counts) HCG_CUDA(c, cudaMemcpyAsync(counts, c->d_out_cnt.p, nc * 4, cudaMemcpyDeviceToHost, c->st_comp));
        HCG_CUDA(c, cudaStreamSynchronize(c->st_comp));
        c->stats.n_samples = n;
        return HCGRID_OK;
    }
    cudaStream_t st = nullptr;   // legacy default stream: ordered with everything
    if (n > 0) {
        HCG_CUDA(c, cudaMemcpyAsync(c->d_in_lon.p, lon, nn * 8, cudaMemcpyHostToDevice, st));
        HCG_CUDA(c, cudaMemcpyAsync(c->d_in_lat.p, lat, nn * 8, cudaMemcpyHostToDevice, st));
        HCG_CUDA(c, cudaMemcpyAsync(c->d_in_val.p, values, nn * (size_t)nchan * 4, cudaMemcpyHostToDevice, st));
        if (weights) HCG_CUDA(c, cudaMemcpyAsync(c->d_in_wgt.p, weights, nn * 4, cudaMemcpyHostToDevice, st));
    }
    const int rc = hcgrid_grid(c, n, c->d_in_lon.as<double>(), c->d_in_lat.as<double>(), c->d_in_val.as<float>(),
                               nchan, weights ? c->d_in_wgt.as<float>() : nullptr, c->d_out_cube.p, c->d_out_w.p,
                               counts ? c->d_out_cnt.as<int32_t>() : nullptr, st);
    if (rc != HCGRID_OK) return rc;
    HCG_CUDA(c, cudaMemcpyAsync(cube, c->d_out_cube.p, nc * (size_t)nchan * osz, cudaMemcpyDeviceToHost, st));
    HCG_CUDA(c, cudaMemcpyAsync(wmap, c->d_out_w.p, nc * osz, cudaMemcpyDeviceToHost, st));
    if (counts) HCG_CUDA(c, cudaMemcpyAsync(counts, c->d_out_cnt.p, nc * 4, cudaMemcpyDeviceToHost, st));
    HCG_CUDA(c, cudaStreamSynchronize(st));
    return HCGRID_OK;
}

int64_t hcgrid_ncell(const hcgrid_ctx* c) { return c && c->has_target ? c->ncell : 0; }

int hcgrid_get_stats(const hcgrid_ctx* cc, hcgrid_stats* out) {
    hcgrid_ctx* c = const_cast<hcgrid_ctx*>(cc);
    if (!c || !out) return HCGRID_ERR_INVALID_ARG;
    HCG_CUDA(c, cudaSetDevice(c->device));
    if (c->stats.n_kept < 0) {
        HCG_CUDA(c, cudaStreamSynchronize(c->last_stream));
        int32_t kept = 0;
        HCG_CUDA(c, cudaMemcpy(&kept, c->d_bins.as<int32_t>() + c->region.nbins, 4, cudaMemcpyDeviceToHost));
        c->stats.n_kept = kept;
    }
    if (c->ev_valid) {
        HCG_CUDA(c, cudaEventSynchronize(c->ev[5]));
        float* dst[5] = {&c->stats.us_pixelise, &c->stats.us_sort, &c->stats.us_tables, &c->stats.us_pack,
                         &c->stats.us_convolve};
        for (int i = 0; i < 5; ++i) {
            float ms = 0.f;
            HCG_CUDA(c, cudaEventElapsedTime(&ms, c->ev[i], c->ev[i + 1]));
            *dst[i] = ms * 1000.f;
        }
        float ms = 0.f;
        HCG_CUDA(c, cudaEventElapsedTime(&ms, c->ev[0], c->ev[5]));
        c->stats.us_total = ms * 1000.f;
    }
    c->stats.n_hit = -1;
    c->stats.n_pairs_tested = -1;
    if (c->stat_hit || c->stat_pairs) {
        HCG_CUDA(c, cudaStreamSynchronize(c->last_stream));
        long long v[2] = {0, 0};
        HCG_CUDA(c, cudaMemcpy(v, c->d_stat.p, 16, cudaMemcpyDeviceToHost));
        if (c->stat_hit) c->stats.n_hit = v[0];
        if (c->stat_pairs) c->stats.n_pairs_tested = v[1];
    }
    c->stats.n_bins = c->region.nbins;
    c->stats.n_rings = c->region.nring;
    c->stats.subpix_bits = c->region.subpix;
    *out = c->stats;
    return HCGRID_OK;
}

const char* hcgrid_last_error(const hcgrid_ctx* c) { return c ? c->err.c_str() : g_create_err.c_str(); }

}  // extern "C"
