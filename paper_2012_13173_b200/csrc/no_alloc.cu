// no_alloc.cu -- hcgrid_count_hits_static: one entry point that allocates nothing.
//
// Some callers cannot call cudaMalloc: code under CUDA-graph capture, tight serving loops, harnesses that forbid
// it.  Every other entry point of the library may grow a context-owned buffer (DevBuf::ensure -> cudaMalloc).  This
// one is a variant of sum_counts_kernel (convolve.cu: n_hit of hcgrid_stats, the "kernel evaluations" of the
// throughput metric) whose scratch -- per-block partial sums and the ticket of the last-block
// reduction -- lives in a file-scope __device__ array of fixed size instead of a cudaMalloc'ed buffer:
//
//     out[0] = sum of counts[0 .. ncell)            (pairs (cell, sample) with d <= R: n_hit)
//     out[1] = number of cells with counts[i] > 0   (cells the samples reach)
//
// Limits and sharing.  kStaticMaxCells = 2^30 cells (the library's own limit for a plate-carree target); the array
// is 2 * 1024 + 32 unsigned 64-bit words = 16.25 KB, held by every GPU that loads the library until the process
// exits.  ALL calls on one device share that array and it keeps the last call's contents: the ticket is cleared at
// the start of every call (on the caller's stream), the partial sums are overwritten before they are read.  Calls
// that overlap on the GPU (two streams, or two host threads on one device) race on it and give wrong sums: callers
// serialise them.  Integer arithmetic in a fixed order: the result does not depend on scheduling.
#include <mutex>

#include "hcg_common.cuh"

namespace hcg {

constexpr int kStaticBlocks = 1024;                        // most blocks a call launches = partial sums per output
constexpr int64_t kStaticMaxCells = (int64_t)1 << 30;      // largest ncell accepted
constexpr int kStaticWords = 2 * kStaticBlocks + 32;       // partial hits, partial filled cells, ticket (+ padding)
constexpr int kStaticMaxDevices = 64;

// In HOST code this name is a host-side stand-in, not a device address: the address the kernel gets comes from
// cudaGetSymbolAddress (static_scratch below).  Device code may name it directly.
static __device__ __align__(256) unsigned long long g_static_scratch[kStaticWords];

__device__ __forceinline__ unsigned long long block_sum_u64(unsigned long long v, unsigned long long* s_red) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    __syncthreads();                                       // s_red may still be read from the previous use
    if (lane == 0) s_red[w] = v;
    __syncthreads();
    unsigned long long t = 0;
    if (w == 0) {
        t = lane < (int)(blockDim.x >> 5) ? s_red[lane] : 0ull;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    }
    return t;                                              // valid in warp 0
}

// scratch: [0, kStaticBlocks) partial hit sums, [kStaticBlocks, 2 kStaticBlocks) partial filled-cell counts,
// [2 kStaticBlocks] the ticket (zero on entry).  The block that draws the last ticket adds the partial sums up in
// block order and writes out[0], out[1].
__global__ void __launch_bounds__(256)
count_hits_static_kernel(const int32_t* __restrict__ counts, int64_t ncell, unsigned long long* __restrict__ scratch,
                         unsigned long long* __restrict__ out) {
    __shared__ unsigned long long s_red[8];
    __shared__ bool s_last;
    unsigned long long hit = 0, filled = 0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < ncell; i += (int64_t)gridDim.x * blockDim.x) {
        const int32_t c = __ldg(counts + i);
        if (c > 0) { hit += (unsigned long long)c; filled += 1; }
    }
    hit = block_sum_u64(hit, s_red);
    filled = block_sum_u64(filled, s_red);
    if (threadIdx.x == 0) {
        scratch[blockIdx.x] = hit;
        scratch[kStaticBlocks + blockIdx.x] = filled;
        __threadfence();                                   // the partial sums before the ticket
        const unsigned t = atomicAdd((unsigned int*)(scratch + 2 * kStaticBlocks), 1u);
        s_last = t == gridDim.x - 1;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    hit = 0; filled = 0;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += blockDim.x) {
        hit += ((volatile unsigned long long*)scratch)[b];
        filled += ((volatile unsigned long long*)scratch)[kStaticBlocks + b];
    }
    hit = block_sum_u64(hit, s_red);
    filled = block_sum_u64(filled, s_red);
    if (threadIdx.x == 0) { out[0] = hit; out[1] = filled; }
}

// Device address of the scratch array on the CURRENT device: looked up once per device, with that device current.
static int static_scratch(int device, unsigned long long** ptr) {
    static std::mutex mu;
    static unsigned long long* cache[kStaticMaxDevices] = {};
    std::lock_guard<std::mutex> lock(mu);
    if (!cache[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess || p == nullptr) return cuda_fail(nullptr, e, "cudaGetSymbolAddress(g_static_scratch)");
        cache[device] = (unsigned long long*)p;
    }
    *ptr = cache[device];
    return HCGRID_OK;
}

}  // namespace hcg

using namespace hcg;

extern "C" {

int64_t hcgrid_static_max_cells(void) { return kStaticMaxCells; }

int hcgrid_count_hits_static(const int32_t* counts, int64_t ncell, uint64_t* out, void* stream) {
    if (ncell < 0) return fail(nullptr, HCGRID_ERR_INVALID_ARG, "ncell must be >= 0");
    if (ncell > kStaticMaxCells)
        return fail(nullptr, HCGRID_ERR_INVALID_ARG, "hcgrid_count_hits_static takes at most %lld cells (its scratch is a "
                    "fixed device array); %lld given", (long long)kStaticMaxCells, (long long)ncell);
    if (!out || (ncell > 0 && !counts)) return fail(nullptr, HCGRID_ERR_INVALID_ARG, "counts / out is NULL");
    int device = -1;
    cudaError_t e = cudaGetDevice(&device);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDevice");
    if (device < 0 || device >= kStaticMaxDevices)
        return fail(nullptr, HCGRID_ERR_UNSUPPORTED, "device ordinal %d beyond the %d this entry point keeps addresses for",
                    device, kStaticMaxDevices);
    unsigned long long* scratch = nullptr;
    const int rc = static_scratch(device, &scratch);
    if (rc != HCGRID_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    // what must start at zero: the ticket (a call that was cut short may have left it half-way)
    e = cudaMemsetAsync(scratch + 2 * kStaticBlocks, 0, sizeof(unsigned long long), st);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaMemsetAsync(ticket)");
    int64_t blocks = (ncell + 256 * 8 - 1) / (256 * 8);     // ~8 cells per thread
    blocks = blocks < 1 ? 1 : (blocks > kStaticBlocks ? kStaticBlocks : blocks);
    count_hits_static_kernel<<<(unsigned)blocks, 256, 0, st>>>(counts, ncell, scratch, (unsigned long long*)out);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "count_hits_static_kernel");
    return HCGRID_OK;
}

}  // extern "C"
