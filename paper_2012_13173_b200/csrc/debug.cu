// debug.cu -- introspection entry points of include/hcgrid.h used by the tests and the
// bench: the a2 step alone (device and host flavours of the same HEALPix code), the
// pre-ordering tables of the last call, and the FP32 / MUFU peak probes the roofline of
// DESIGN.md is quoted against.
#include <vector>

#include "hcg_common.cuh"

namespace hcg {

HCG_HD int64_t ang2pix_ring_deg(int nside, double lon_deg, double lat_deg) {
    double l = fmod(lon_deg, 360.0);
    if (l < 0.0) l += 360.0;
    int iring, ip;
    ang2ring(nside, l * kDeg2Rad, lat_deg * kDeg2Rad, iring, ip);
    return ring_first_pixel(iring, nside) + ip;
}

__global__ void ang2pix_kernel(int nside, int64_t n, const double* __restrict__ lon,
                               const double* __restrict__ lat, int64_t* __restrict__ pix) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) pix[i] = ang2pix_ring_deg(nside, lon[i], lat[i]);
}

__global__ void sorted_pixel_kernel(int nside, int64_t nkept, const uint32_t* __restrict__ sidx,
                                    const double* __restrict__ lon, const double* __restrict__ lat,
                                    int64_t* __restrict__ pix, int64_t* __restrict__ idx) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nkept) return;
    const uint32_t s = sidx[i];
    pix[i] = ang2pix_ring_deg(nside, lon[s], lat[s]);
    idx[i] = (int64_t)s;
}

// Register-only dependent chains, 8 independent per thread: issue-rate probes.
template <int MODE>
__global__ void __launch_bounds__(256) peak_kernel(float* out, int iters, float a, float b) {
    float x[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) x[j] = a + (float)(threadIdx.x + j) * 1e-3f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            if (MODE == 0) x[j] = fmaf(x[j], a, b);
            else asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(x[j]));
        }
    }
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < 8; ++j) s += x[j];
    if (s == 12345.678f) out[0] = s;   // never true in practice; keeps the chains alive
}

}  // namespace hcg

using namespace hcg;

extern "C" {

int hcgrid_debug_ang2pix_ring(int64_t nside, int64_t n, const double* lon, const double* lat, int64_t* pix,
                              void* stream) {
    if (nside < 1 || nside > 16384 || (nside & (nside - 1)) || n < 0 || (n > 0 && (!lon || !lat || !pix)))
        return fail(nullptr, HCGRID_ERR_INVALID_ARG, "hcgrid_debug_ang2pix_ring: bad arguments");
    if (n == 0) return HCGRID_OK;
    ang2pix_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>((int)nside, n, lon, lat, pix);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "ang2pix_kernel");
    return HCGRID_OK;
}

int hcgrid_host_ang2pix_ring(int64_t nside, int64_t n, const double* lon, const double* lat, int64_t* pix) {
    if (nside < 1 || nside > 16384 || (nside & (nside - 1)) || n < 0 || (n > 0 && (!lon || !lat || !pix)))
        return fail(nullptr, HCGRID_ERR_INVALID_ARG, "hcgrid_host_ang2pix_ring: bad arguments");
    for (int64_t i = 0; i < n; ++i) pix[i] = ang2pix_ring_deg((int)nside, lon[i], lat[i]);
    return HCGRID_OK;
}

int hcgrid_host_ring_info(int64_t nside, int32_t iring, int64_t* first_pixel, int32_t* npix, double* lat_deg,
                          double* lon0_deg) {
    if (nside < 1 || nside > 16384 || (nside & (nside - 1)) || iring < 1 || iring > 4 * nside - 1)
        return fail(nullptr, HCGRID_ERR_INVALID_ARG, "hcgrid_host_ring_info: bad arguments");
    const int ns = (int)nside;
    if (first_pixel) *first_pixel = ring_first_pixel(iring, nside);
    const int np = ring_npix(iring, ns);
    if (npix) *npix = np;
    if (lat_deg) *lat_deg = (kHalfPi - ring_colat(iring, ns)) / kDeg2Rad;
    // centre of pixel 0: g = 1/2  ->  lon = (1/2 - off) * 2 pi / npix
    if (lon0_deg) *lon0_deg = (0.5 - ring_off(iring, ns)) * 360.0 / (double)np;
    return HCGRID_OK;
}

int hcgrid_debug_preorder(hcgrid_ctx* c, int64_t* sorted_pixel, int64_t* sorted_index, int32_t* ring_first,
                          int64_t* ring_start) {
    if (!c) return HCGRID_ERR_INVALID_ARG;
    if (!c->has_target || c->last_n < 0) return fail(c, HCGRID_ERR_NO_TARGET, "no hcgrid_grid call to inspect");
    HCG_CUDA(c, cudaSetDevice(c->device));
    HCG_CUDA(c, cudaStreamSynchronize(c->last_stream));
    const Region& rg = c->region;
    std::vector<int32_t> bins((size_t)rg.nbins + 1);
    HCG_CUDA(c, cudaMemcpy(bins.data(), c->d_bins.p, bins.size() * 4, cudaMemcpyDeviceToHost));
    const int64_t nkept = bins[(size_t)rg.nbins];
    if (ring_first) *ring_first = rg.ring_first;
    if (ring_start)
        for (int r = 0; r <= rg.nring; ++r) ring_start[r] = bins[(size_t)r * rg.m];
    if ((sorted_pixel || sorted_index) && nkept > 0) {
        DevBuf dp, di;
        HCG_CUDA(c, dp.ensure((size_t)nkept * 8));
        cudaError_t e = di.ensure((size_t)nkept * 8);
        if (e != cudaSuccess) { dp.release(); return cuda_fail(c, e, "alloc"); }
        sorted_pixel_kernel<<<(unsigned)((nkept + 255) / 256), 256>>>(c->nside, nkept, c->d_idx_out.as<uint32_t>(),
                                                                     c->last_lon, c->last_lat, dp.as<int64_t>(),
                                                                     di.as<int64_t>());
        e = cudaGetLastError();
        if (e == cudaSuccess && sorted_pixel)
            e = cudaMemcpy(sorted_pixel, dp.p, (size_t)nkept * 8, cudaMemcpyDeviceToHost);
        if (e == cudaSuccess && sorted_index)
            e = cudaMemcpy(sorted_index, di.p, (size_t)nkept * 8, cudaMemcpyDeviceToHost);
        dp.release(); di.release();
        if (e != cudaSuccess) return cuda_fail(c, e, "hcgrid_debug_preorder");
    }
    return HCGRID_OK;
}

int hcgrid_measure_peaks(int device, double* fp32_inst_per_s, double* mufu_per_s) {
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaSetDevice");
    int sms = 0;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    float* d = nullptr;
    e = cudaMalloc(&d, 64);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaMalloc");
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int blocks = sms * 8, threads = 256;
    double res[2] = {0, 0};
    for (int mode = 0; mode < 2; ++mode) {
        const int iters = mode == 0 ? 20000 : 4000;
        double best = 0;
        for (int rep = 0; rep < 6; ++rep) {
            cudaEventRecord(e0);
            if (mode == 0) peak_kernel<0><<<blocks, threads>>>(d, iters, 0.999f, 1e-3f);
            else peak_kernel<1><<<blocks, threads>>>(d, iters, -0.5f, 0.f);
            cudaEventRecord(e1);
            e = cudaEventSynchronize(e1);
            if (e != cudaSuccess) break;
            float ms = 0;
            cudaEventElapsedTime(&ms, e0, e1);
            const double ops = (double)blocks * threads * 8.0 * iters;
            if (rep > 0 && ops / (ms * 1e-3) > best) best = ops / (ms * 1e-3);
        }
        res[mode] = best;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(d);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "peak_kernel");
    if (fp32_inst_per_s) *fp32_inst_per_s = res[0];
    if (mufu_per_s) *mufu_per_s = res[1];
    return HCGRID_OK;
}

}  // extern "C"
