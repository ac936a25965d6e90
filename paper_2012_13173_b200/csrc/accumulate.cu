// accumulate.cu -- incremental gridding (the paper names streaming of
// successive scans as future work).  Eq. 1 is a ratio of two sums
// over the samples, and both sums are additive over batches of samples:
//     V = (sum_b S_b) / (sum_b W_b),   S_b = sum_{n in batch b} q w v,   W_b = sum_{n in b} q w.
// hcgrid_accumulate grids one batch with the usual path, the convolution kernels writing the
// un-normalised S_b (and W_b, counts), and adds them to context-owned accumulators;
// hcgrid_finalize divides.  Gridding the batches one after the other therefore gives the
// result of gridding their union, up to the order of the floating-point additions.
#include <cstring>

#include "hcg_common.cuh"

namespace hcg {

static double __longlong_as_double_host(long long v) { double d; std::memcpy(&d, &v, 8); return d; }
static float __int_as_float_host(int v) { float f; std::memcpy(&f, &v, 4); return f; }

// acc += part for the three outputs of one batch in one launch (thread i: sum i, and cell i's
// weight and count while i < ncell).
template <typename T>
__global__ void __launch_bounds__(256)
add_batch_kernel(T* __restrict__ acc_cube, const T* __restrict__ cube, int64_t ne, T* __restrict__ acc_w,
                 const T* __restrict__ w, int32_t* __restrict__ acc_cnt, const int32_t* __restrict__ cnt, int64_t nc) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < ne) acc_cube[i] += cube[i];
    if (i < nc) { acc_w[i] += w[i]; acc_cnt[i] += cnt[i]; }
}

template <typename T>
__global__ void __launch_bounds__(256)
finalize_kernel(const T* __restrict__ acc_cube, const T* __restrict__ acc_w, const int32_t* __restrict__ acc_cnt,
                int64_t ncell, int nchan, T* __restrict__ cube, T* __restrict__ wmap, int32_t* __restrict__ counts,
                T nan) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;      // over ncell * nchan
    if (i >= ncell * nchan) return;
    const int64_t cell = i / nchan;
    const T w = acc_w[cell];
    cube[i] = w != (T)0 ? acc_cube[i] / w : nan;   // signed kernels: W may be negative
    if (i == cell * nchan) {
        wmap[cell] = w;
        if (counts) counts[cell] = acc_cnt[cell];
    }
}

template <typename T>
static int accumulate_impl(hcgrid_ctx* c, int64_t n, const double* lon, const double* lat, const float* values,
                           int nchan, const float* weights, cudaStream_t st) {
    const size_t nc = (size_t)c->ncell, ne = nc * (size_t)nchan;
    if (c->acc_nchan == 0) {
        // first batch: its un-normalised sums ARE the accumulators
        HCG_CUDA(c, c->d_acc_cube.ensure(ne * sizeof(T)));
        HCG_CUDA(c, c->d_acc_w.ensure(nc * sizeof(T)));
        HCG_CUDA(c, c->d_acc_cnt.ensure(nc * 4));
        c->raw_sums = true;
        const int rc = hcgrid_grid(c, n, lon, lat, values, nchan, weights, c->d_acc_cube.p, c->d_acc_w.p,
                                   c->d_acc_cnt.as<int32_t>(), st);
        c->raw_sums = false;
        if (rc != HCGRID_OK) return rc;
        c->acc_nchan = nchan;
        c->acc_batches = 1;
        return HCGRID_OK;
    }
    HCG_CUDA(c, c->d_tmp_cube.ensure(ne * sizeof(T)));
    HCG_CUDA(c, c->d_tmp_w.ensure(nc * sizeof(T)));
    HCG_CUDA(c, c->d_tmp_cnt.ensure(nc * 4));
    c->raw_sums = true;
    const int rc = hcgrid_grid(c, n, lon, lat, values, nchan, weights, c->d_tmp_cube.p, c->d_tmp_w.p,
                               c->d_tmp_cnt.as<int32_t>(), st);
    c->raw_sums = false;
    if (rc != HCGRID_OK) return rc;
    const int threads = 256;
    add_batch_kernel<T><<<(unsigned)((ne + threads - 1) / threads), threads, 0, st>>>(
        c->d_acc_cube.as<T>(), c->d_tmp_cube.as<T>(), (int64_t)ne, c->d_acc_w.as<T>(), c->d_tmp_w.as<T>(),
        c->d_acc_cnt.as<int32_t>(), c->d_tmp_cnt.as<int32_t>(), (int64_t)nc);
    HCG_CUDA(c, cudaGetLastError());
    c->stats.gpu_launches += 1;
    c->acc_batches += 1;
    return HCGRID_OK;
}

template <typename T>
static int finalize_impl(hcgrid_ctx* c, void* cube, void* wmap, int32_t* counts, cudaStream_t st, T nan) {
    const int64_t ne = c->ncell * (int64_t)c->acc_nchan;
    const int threads = 256;
    finalize_kernel<T><<<(unsigned)((ne + threads - 1) / threads), threads, 0, st>>>(
        c->d_acc_cube.as<T>(), c->d_acc_w.as<T>(), c->d_acc_cnt.as<int32_t>(), c->ncell, c->acc_nchan, (T*)cube,
        (T*)wmap, counts, nan);
    HCG_CUDA(c, cudaGetLastError());
    return HCGRID_OK;
}

}  // namespace hcg

using namespace hcg;

extern "C" {

int hcgrid_accumulate(hcgrid_ctx* c, int64_t n, const double* lon, const double* lat, const float* values,
                      int32_t nchan, const float* weights, void* stream) {
    if (!c) return HCGRID_ERR_INVALID_ARG;
    if (!c->has_target) return fail(c, HCGRID_ERR_NO_TARGET, "no target set (call hcgrid_set_target_* first)");
    if (nchan < 1) return fail(c, HCGRID_ERR_INVALID_ARG, "nchan must be >= 1");
    if (c->acc_nchan != 0 && c->acc_nchan != nchan)
        return fail(c, HCGRID_ERR_INVALID_ARG, "nchan %d differs from the running accumulation's %d", (int)nchan,
                    c->acc_nchan);
    HCG_CUDA(c, cudaSetDevice(c->device));
    return c->precision == HCGRID_F64
               ? accumulate_impl<double>(c, n, lon, lat, values, nchan, weights, (cudaStream_t)stream)
               : accumulate_impl<float>(c, n, lon, lat, values, nchan, weights, (cudaStream_t)stream);
}

int hcgrid_finalize(hcgrid_ctx* c, void* cube, void* wmap, int32_t* counts, int reset, void* stream) {
    if (!c) return HCGRID_ERR_INVALID_ARG;
    if (!c->has_target || c->acc_nchan == 0)
        return fail(c, HCGRID_ERR_NO_TARGET, "nothing accumulated (call hcgrid_accumulate first)");
    if (!cube || !wmap) return fail(c, HCGRID_ERR_INVALID_ARG, "datacube / weightmap is NULL");
    HCG_CUDA(c, cudaSetDevice(c->device));
    const int rc = c->precision == HCGRID_F64
                       ? finalize_impl<double>(c, cube, wmap, counts, (cudaStream_t)stream,
                                               __longlong_as_double_host(0x7ff8000000000000LL))
                       : finalize_impl<float>(c, cube, wmap, counts, (cudaStream_t)stream, __int_as_float_host(0x7fc00000));
    if (rc == HCGRID_OK && reset) c->acc_nchan = 0;
    return rc;
}

int64_t hcgrid_accumulated_batches(const hcgrid_ctx* c) { return c && c->acc_nchan != 0 ? c->acc_batches : 0; }

}  // extern "C"
