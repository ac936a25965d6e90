// preorder.cu -- steps a2..a5: the pre-ordering of PAPER.md:108-124 (Sect. 3.3), all on
// the device (the paper runs it on CPU threads).
//   a2 pixelise   HEALPix RING pixel of every sample ("get the pixel index
//                 P_n"), reduced to a sort key = (ring - ring_first) * m + bin-in-ring,
//                 where the bins refine the ring's pixels by 2^b along the ring and are
//                 counted from the target region's western edge.  Samples the target
//                 cannot reach (other rings / outside the longitude window) get the
//                 sentinel key and sort to the end.
//   a3 sort       key-value sort of (key, n), non-descending, stable (PAPER.md:120
//                 "key-value sorting of P_n and n"); CUB radix sort over the key's
//                 varying bits (the paper's fourth option is Thrust sort_by_key).
//   a4 tables     bin_start[k] = first position in S' whose key >= k: the first-level
//                 table P_i -> S_start at bin granularity; its every m-th
//                 entry is the second-level table R_start (Fig. 3).
//   a5 pack       S -> S' ("rearrange the raw data S_n as S'") as 16-byte
//                 fixed-point records (fp32 mode) or degree records (fp64 mode).  In fp32
//                 mode a4 and a5 are one kernel: one pass over the sorted pairs.
#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>

#include "hcg_common.cuh"

namespace hcg {

// kCount: the counting pre-order (below) -- idx[i] receives the sample's arrival rank within
// its bin (global atomic on the bin's counter) instead of i.
template <bool kF32, bool kCount>
__global__ void __launch_bounds__(256)
pixelise_kernel(const double* __restrict__ lon_deg, const double* __restrict__ lat_deg,
                const float* __restrict__ values, const float* __restrict__ weights,
                int nchan, int64_t n, Region rg, uint32_t* __restrict__ keys,
                uint32_t* __restrict__ idx, Rec32* __restrict__ rec, int32_t* __restrict__ bin_count) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double lo_d = lon_deg[i], la_d = lat_deg[i];
    uint32_t key = (uint32_t)rg.nbins;                       // sentinel: sorts last
    Rec32 r;
    r.xi = 0; r.yi = 0; r.idx = (uint32_t)i; r.q = 1.0f;
    if (isfinite(lo_d) && la_d >= -90.0 && la_d <= 90.0) {
        double l = lo_d - 360.0 * floor(lo_d * (1.0 / 360.0));     // lon mod 360
        if (l >= 360.0) l -= 360.0;
        if (l < 0.0) l += 360.0;
        const double lon = l * kDeg2Rad, lat = la_d * kDeg2Rad;
        int iring, ip;
        ang2ring(rg.nside, lon, lat, iring, ip);
        const int rr = iring - rg.ring_first;
        double u = lon - rg.lon_lo;
        if (u < 0.0) u += kTwoPi;
        if (u >= kTwoPi) u -= kTwoPi;
        if (rr >= 0 && rr < rg.nring && (rg.full_circle || u < rg.wx * (1.0 - 1e-9))) {
            const int bin = (int)ring_bin(iring, rg.nside, ip, lon, rg.subpix);
            const int nb = (int)ring_nbins(iring, rg.nside, rg.subpix);
            const int j0 = (int)floor(ring_bin_coord(iring, rg.nside, rg.lon_lo, rg.subpix)) - 2;   // in [-2, nb)
            int jrel = bin - j0;                                     // in (-nb, nb + 2]
            if (jrel < 0) jrel += nb;
            if (jrel >= nb) jrel -= nb;
            if (jrel < rg.m) {
                key = (uint32_t)(rr * rg.m + jrel);
                if (kF32) {
                    r.xi = (uint32_t)(unsigned long long)__double2ll_rn(u * rg.sx32);
                    r.yi = (uint32_t)(unsigned long long)__double2ll_rn((lat - rg.lat_lo) * rg.sy32);
                }
            }
        }
    }
    keys[i] = key;
    if (kCount) idx[i] = key != (uint32_t)rg.nbins ? (uint32_t)atomicAdd(bin_count + key, 1) : 0u;
    else idx[i] = (uint32_t)i;
    if (kF32) {
        if (nchan == 1) r.v = values[i];
        if (weights) r.q = weights[i];
        rec[i] = r;
    }
}

// a4 + a5 (fp32 mode) in one pass over the sorted pairs.
// a4: bin_start from the sorted keys.  Thread i owns the gap (key[i-1], key[i]]; thread n
// closes the table.  Short gaps are written by their thread; long ones (ring boundaries,
// the empty head and tail of the table) are queued in shared memory and filled by the whole
// block.  Every entry is written exactly once, no global atomics.
// a5: rec_out[i] = rec_in[sidx[i]] for the kept samples (rec_in == nullptr: tables only).
__global__ void __launch_bounds__(256)
tables_pack_kernel(const uint32_t* __restrict__ skeys, const uint32_t* __restrict__ sidx, int64_t n,
                   int32_t nbins, int32_t* __restrict__ bin_start, const Rec32* __restrict__ rec_in,
                   Rec32* __restrict__ rec_out) {
    __shared__ int s_cnt;
    __shared__ int s_lo[256], s_hi[256], s_val[256];
    const int tid = threadIdx.x;
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + tid;
    if (tid == 0) s_cnt = 0;
    __syncthreads();
    uint4 rec = make_uint4(0, 0, 0, 0);
    bool kept = false;
    if (i <= n) {
        const int prev = i == 0 ? -1 : (int)min(skeys[i - 1], (uint32_t)nbins);
        const int cur = i == n ? nbins : (int)min(skeys[i], (uint32_t)nbins);
        kept = rec_in != nullptr && i < n && cur != nbins;
        if (kept) rec = __ldg((const uint4*)(rec_in + sidx[i]));
        if (cur - prev <= 4) {
            for (int k = prev + 1; k <= cur; ++k) bin_start[k] = (int32_t)i;
        } else {
            const int slot = atomicAdd(&s_cnt, 1);          // shared-memory queue slot, order irrelevant
            s_lo[slot] = prev + 1; s_hi[slot] = cur; s_val[slot] = (int32_t)i;
        }
    }
    if (kept) *(uint4*)(rec_out + i) = rec;
    __syncthreads();
    const int ngap = s_cnt;
    for (int g = 0; g < ngap; ++g) {
        const int hi = s_hi[g], val = s_val[g];
        for (int k = s_lo[g] + tid; k <= hi; k += 256) bin_start[k] = val;
    }
}

// ---- counting pre-order: a3..a5 without the multi-pass radix sort -------------------
// The keys are bin numbers of a table that is built anyway, so the sort of PAPER.md:120 is a
// counting sort: pixelise_kernel<.., true> counts every bin and keeps each sample's arrival
// rank, an exclusive scan of the counts IS bin_start (a4), scatter_index_kernel puts sample i
// at bin_start[key] + rank, and order_pack_kernel moves every index to its place in ascending
// order inside its bin -- arrival order is whatever the atomics made it; ascending index is what
// the stable sort gives, so S' is identical to the radix path's, bit for bit -- gathering the
// record on the way (a5).

constexpr int kLongBin = 1024;           // bins longer than this are ordered by the block-sort kernel
constexpr int64_t kGuardMinN = 1 << 20;  // calls from this size on report their count of such bins to the host
constexpr uint32_t kStartFlag = 0x80000000u, kIdxMask = 0x7fffffffu;   // n <= 2e9 < 2^31 (hcgrid_grid)

// sidx_raw[bin_start[key] + rank] = i, with the top bit set on rank 0: the sample that arrived
// first sits at its bin's first position and so marks where the bin begins.  The one sample
// with rank == kLongBin (there is exactly one iff the bin is longer) queues its bin for the
// block-sort kernel.
__global__ void __launch_bounds__(256)
scatter_index_kernel(const uint32_t* __restrict__ keys, const uint32_t* __restrict__ rank, int64_t n,
                     int32_t nbins, const int32_t* __restrict__ bin_start, uint32_t* __restrict__ sidx_raw,
                     int32_t* __restrict__ long_count, int32_t* __restrict__ long_list) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t key = keys[i];
    if (key >= (uint32_t)nbins) return;
    const uint32_t r = rank[i];
    sidx_raw[(int64_t)__ldg(bin_start + key) + r] = (uint32_t)i | (r == 0 ? kStartFlag : 0u);
    if (r == (uint32_t)kLongBin) long_list[atomicAdd(long_count, 1)] = (int32_t)key;
}

// Ascending sort of a[0, L) by the whole block, in place in global memory: the bitonic
// network in its all-ascending form (first sub-stage of every stage mirrors, the others
// shift), so the virtual padding to a power of two sits at the top and is never touched.
__device__ __forceinline__ void cmp_swap(uint32_t* a, int i, int j, int L) {
    if (j < L) {
        const uint32_t x = a[i], y = a[j];
        if (x > y) { a[i] = y; a[j] = x; }
    }
}

__device__ void block_sort_u32(uint32_t* a, int L, int tid, int nthr) {
    int P = 1;
    while (P < L) P <<= 1;
    for (int k = 2; k <= P; k <<= 1) {
        for (int t = tid; t < P / 2; t += nthr) {
            const int l = t & (k / 2 - 1), base = (t - l) * 2;
            cmp_swap(a, base + l, base + k - 1 - l, L);
        }
        __syncthreads();
        for (int j = k >> 2; j >= 1; j >>= 1) {
            for (int t = tid; t < P / 2; t += nthr) {
                const int l = t & (j - 1), i = (t - l) * 2 + l;
                cmp_swap(a, i, i + j, L);
            }
            __syncthreads();
        }
    }
}

// a3 (order inside the bins) + a5 in one pass, one thread per position p of the arrival-ordered
// index array: the thread walks left to its bin's start flag and right to the next one, counting
// on the way how many of the bin's indices are smaller than its own -- that count is its place in
// ascending order, which is the stable sort's order -- and writes its index (and, kPack, the
// gathered record) there.  The walks are neighbouring loads the warp has in L1 anyway; the kernel
// stays bound by the random record gather.  Bins longer than kLongBin are left to order_long_kernel.
template <bool kPack>
__global__ void __launch_bounds__(256)
order_pack_kernel(const uint32_t* __restrict__ sidx_raw, int64_t n, const int32_t* __restrict__ nkept_ptr,
                  uint32_t* __restrict__ sidx, const Rec32* __restrict__ rec_in, Rec32* __restrict__ rec_out) {
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t nkept = nkept_ptr[0];
    if (p >= n || p >= nkept) return;
    const uint32_t raw = sidx_raw[p];
    const uint32_t v = raw & kIdxMask;
    int below = 0;
    int64_t s = p;
    uint32_t x = raw;
    while (!(x & kStartFlag)) {
        if (p - s >= kLongBin) return;                       // a long bin
        --s;
        x = sidx_raw[s];
        below += (x & kIdxMask) < v;
    }
    int64_t e = p + 1;
    while (e < nkept) {
        x = sidx_raw[e];
        if (x & kStartFlag) break;
        if (e - s >= kLongBin) return;                       // a long bin (every member sees the same length)
        below += (x & kIdxMask) < v;
        ++e;
    }
    const int64_t d = s + below;
    sidx[d] = v;
    if (kPack) *(uint4*)(rec_out + d) = __ldg((const uint4*)(rec_in + v));
}

// The queued long bins, one block at a time: copy the indices, sort them (block_sort_u32), gather.
template <bool kPack>
__global__ void __launch_bounds__(256)
order_long_kernel(const uint32_t* __restrict__ sidx_raw, const int32_t* __restrict__ bin_start,
                  int32_t* __restrict__ long_count, const int32_t* __restrict__ long_list, uint32_t* sidx,
                  const Rec32* __restrict__ rec_in, Rec32* __restrict__ rec_out, volatile int32_t* __restrict__ host_report) {
    const int nlong = long_count[0];
    for (int g = blockIdx.x; g < nlong; g += gridDim.x) {
        const int key = long_list[g];
        const int s = bin_start[key], len = bin_start[key + 1] - s;
        if (threadIdx.x == 0) atomicMax(long_count + 1, len);   // the longest bin, for the host's guard (run_preorder)
        for (int k = threadIdx.x; k < len; k += 256) sidx[s + k] = sidx_raw[s + k] & kIdxMask;
        __syncthreads();
        block_sort_u32(sidx + s, len, threadIdx.x, 256);    // ends with a barrier
        if (kPack)
            for (int k = threadIdx.x; k < len; k += 256)
                *(uint4*)(rec_out + s + k) = __ldg((const uint4*)(rec_in + sidx[s + k]));
        __syncthreads();
    }
    // the last block to leave tells the host (a mapped pinned word pair: no copy on the stream) how many bins came
    // here and how long the longest was: run_preorder's guard against piled-up input reads it at a later call
    if (host_report && threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(long_count + 2, 1) == (int)gridDim.x - 1) {
            host_report[0] = nlong;
            host_report[1] = ((volatile int32_t*)long_count)[1];
        }
    }
}

__global__ void __launch_bounds__(256)
pack64_kernel(const uint32_t* __restrict__ sidx, int64_t n, const int32_t* __restrict__ nkept,
              const double* __restrict__ lon_deg, const double* __restrict__ lat_deg,
              const float* __restrict__ weights, Rec64* __restrict__ rec_out) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n || i >= (int64_t)nkept[0]) return;          // nkept = bin_start[nbins]
    const uint32_t s = sidx[i];
    Rec64 r;
    r.lon_deg = lon_deg[s];
    r.lat_deg = lat_deg[s];
    r.coslat = cos(r.lat_deg * kDeg2Rad);
    r.idx = s;
    r.q = weights ? weights[s] : 1.0f;
    rec_out[i] = r;
}

int run_preorder(hcgrid_ctx* c, int64_t n, const double* lon, const double* lat, const float* values,
                 int nchan, const float* weights, cudaStream_t st) {
    const Region& rg = c->region;
    const bool f32 = c->precision == HCGRID_F32 && c->f32_series_ok && c->opt_kernel != 2;
    // counting pre-order unless the samples pile up (long bins to order), the table is far
    // larger than the input (its O(bins) passes), or the option says otherwise; the result is
    // the same S' either way
    const int64_t nbins64 = (int64_t)rg.nbins;
    // what an earlier large call on this target reported behind itself: bins too long for the counting path
    // (event queries are not allowed while the thread captures a stream: the replay path asks later)
    cudaStreamCaptureStatus capturing = cudaStreamCaptureStatusNone;
    HCG_CUDA(c, cudaStreamIsCapturing(st, &capturing));
    if (capturing != cudaStreamCaptureStatusNone || !c->long_pending) {
        // nothing to read now
    } else if (cudaEventQuery(c->ev_long) != cudaSuccess) {
        cudaGetLastError();                                          // not ready: not an error
    } else {
        c->long_pending = false;
        // a few bins of a few thousand samples are fine where they are; many, or a very long one, are not
        if (c->h_long[0] > 64 || c->h_long[1] > 16 * kLongBin) c->force_radix = true;
    }
    const bool counting = n > 0 && (c->opt_preorder == 2 ||
                                    (c->opt_preorder == 0 && !c->force_radix && n <= 10 * nbins64 &&
                                     (nbins64 <= 16 * n || nbins64 <= ((int64_t)1 << 22))));
    const size_t nn = (size_t)(n > 0 ? n : 1);
    HCG_CUDA(c, c->d_keys.ensure(nn * 4));
    HCG_CUDA(c, c->d_idx.ensure(nn * 4));
    HCG_CUDA(c, c->d_idx_out.ensure(nn * 4));
    HCG_CUDA(c, c->d_bins.ensure(((size_t)rg.nbins + 4) * 4));   // + count of long bins, their largest length
    HCG_CUDA(c, c->d_rec.ensure(nn * (f32 ? sizeof(Rec32) : sizeof(Rec64)) + 64));
    if (f32) HCG_CUDA(c, c->d_misc.ensure(nn * sizeof(Rec32)));
    int end_bit = 1;
    while (end_bit < 32 && ((uint64_t)1 << end_bit) <= (uint64_t)rg.nbins) ++end_bit;
    size_t tmp_bytes = 0;
    HCG_CUDA(c, c->d_keys_out.ensure(nn * 4));
    if (counting) {
        HCG_CUDA(c, c->d_long.ensure((nn / kLongBin + 2) * 4));
        HCG_CUDA(c, cub::DeviceScan::ExclusiveSum(nullptr, tmp_bytes, c->d_bins.as<int32_t>(), c->d_bins.as<int32_t>(),
                                                  (int64_t)rg.nbins + 1, st));
    } else {
        HCG_CUDA(c, cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, c->d_keys.as<uint32_t>(),
                                                    c->d_keys_out.as<uint32_t>(), c->d_idx.as<uint32_t>(),
                                                    c->d_idx_out.as<uint32_t>(), (int64_t)nn, 0, end_bit, st));
    }
    HCG_CUDA(c, c->d_sort_tmp.ensure(tmp_bytes + 16));

    const int threads = 256;
    const unsigned nb = (unsigned)((nn + threads - 1) / threads);
    int launches = 0;
    c->stats.preorder = counting ? 2 : 1;
    if (c->opt_profile) cudaEventRecord(c->ev[0], st);
    if (counting) {
        int32_t* bins = c->d_bins.as<int32_t>();
        uint32_t* keys = c->d_keys.as<uint32_t>();
        uint32_t* rank = c->d_idx.as<uint32_t>();
        uint32_t* sidx_raw = c->d_keys_out.as<uint32_t>();   // arrival order, start-of-bin flags
        uint32_t* sidx = c->d_idx_out.as<uint32_t>();        // ascending inside every bin: the sorted "value" column
        HCG_CUDA(c, cudaMemsetAsync(bins, 0, ((size_t)rg.nbins + 4) * 4, st));
        if (f32)
            pixelise_kernel<true, true><<<nb, threads, 0, st>>>(lon, lat, values, weights, nchan, n, rg, keys, rank,
                                                                c->d_misc.as<Rec32>(), bins);
        else
            pixelise_kernel<false, true><<<nb, threads, 0, st>>>(lon, lat, values, weights, nchan, n, rg, keys, rank,
                                                                 nullptr, bins);
        HCG_CUDA(c, cudaGetLastError());
        if (c->opt_profile) cudaEventRecord(c->ev[1], st);
        HCG_CUDA(c, cub::DeviceScan::ExclusiveSum(c->d_sort_tmp.p, tmp_bytes, bins, bins, (int64_t)rg.nbins + 1, st));
        int32_t* long_count = bins + rg.nbins + 1;           // spare entry of the table, zeroed with it
        int32_t* long_list = c->d_long.as<int32_t>();
        scatter_index_kernel<<<nb, threads, 0, st>>>(keys, rank, n, (int32_t)rg.nbins, bins, sidx_raw, long_count,
                                                     long_list);
        HCG_CUDA(c, cudaGetLastError());
        if (c->opt_profile) { cudaEventRecord(c->ev[2], st); cudaEventRecord(c->ev[3], st); }
        const unsigned nlb = (unsigned)(4 * c->num_sms);
        // large calls report their long bins to the host behind themselves (never inside a stream capture: the event is
        // queried by a later call)
        volatile int32_t* report = nullptr;
        if (n >= kGuardMinN && c->opt_preorder == 0 && !c->long_pending && c->h_long_dev &&
            capturing == cudaStreamCaptureStatusNone)
            report = c->h_long_dev;
        if (f32) {
            order_pack_kernel<true><<<nb, threads, 0, st>>>(sidx_raw, n, bins + rg.nbins, sidx, c->d_misc.as<Rec32>(),
                                                            c->d_rec.as<Rec32>());
            order_long_kernel<true><<<nlb, threads, 0, st>>>(sidx_raw, bins, long_count, long_list, sidx,
                                                             c->d_misc.as<Rec32>(), c->d_rec.as<Rec32>(), report);
        } else {
            order_pack_kernel<false><<<nb, threads, 0, st>>>(sidx_raw, n, bins + rg.nbins, sidx, nullptr, nullptr);
            order_long_kernel<false><<<nlb, threads, 0, st>>>(sidx_raw, bins, long_count, long_list, sidx, nullptr,
                                                              nullptr, report);
        }
        HCG_CUDA(c, cudaGetLastError());
        launches = 6;                        // pixelise, scan (2 kernels), scatter, order + pack, long bins
        if (report) {
            HCG_CUDA(c, cudaEventRecord(c->ev_long, st));
            c->long_pending = true;
        }
    } else {
        if (n > 0) {
            if (f32)
                pixelise_kernel<true, false><<<nb, threads, 0, st>>>(lon, lat, values, weights, nchan, n, rg,
                                                                     c->d_keys.as<uint32_t>(), c->d_idx.as<uint32_t>(),
                                                                     c->d_misc.as<Rec32>(), nullptr);
            else
                pixelise_kernel<false, false><<<nb, threads, 0, st>>>(lon, lat, values, weights, nchan, n, rg,
                                                                      c->d_keys.as<uint32_t>(), c->d_idx.as<uint32_t>(),
                                                                      nullptr, nullptr);
            ++launches;
            HCG_CUDA(c, cudaGetLastError());
        }
        if (c->opt_profile) cudaEventRecord(c->ev[1], st);
        if (n > 0) {
            HCG_CUDA(c, cub::DeviceRadixSort::SortPairs(c->d_sort_tmp.p, tmp_bytes, c->d_keys.as<uint32_t>(),
                                                        c->d_keys_out.as<uint32_t>(), c->d_idx.as<uint32_t>(),
                                                        c->d_idx_out.as<uint32_t>(), n, 0, end_bit, st));
            launches += 2 + (end_bit + 7) / 8;   // CUB onesweep: histogram + scan + one pass per digit
        }
        if (c->opt_profile) cudaEventRecord(c->ev[2], st);
        {
            // a4 (+ a5 in fp32 mode: the gather rides on the same pass over the sorted pairs)
            const unsigned nb2 = (unsigned)((nn + 1 + threads - 1) / threads);
            tables_pack_kernel<<<nb2, threads, 0, st>>>(c->d_keys_out.as<uint32_t>(), c->d_idx_out.as<uint32_t>(), n,
                                                        (int32_t)rg.nbins, c->d_bins.as<int32_t>(),
                                                        f32 && n > 0 ? c->d_misc.as<Rec32>() : nullptr,
                                                        c->d_rec.as<Rec32>());
            ++launches;
            HCG_CUDA(c, cudaGetLastError());
        }
        if (c->opt_profile) cudaEventRecord(c->ev[3], st);
    }
    if (n > 0 && !f32) {
        pack64_kernel<<<nb, threads, 0, st>>>(c->d_idx_out.as<uint32_t>(), n, c->d_bins.as<int32_t>() + rg.nbins, lon,
                                              lat, weights, c->d_rec.as<Rec64>());
        ++launches;
        HCG_CUDA(c, cudaGetLastError());
    }
    if (c->opt_profile) cudaEventRecord(c->ev[4], st);
    c->stats.gpu_launches = launches;
    return HCGRID_OK;
}

}  // namespace hcg
