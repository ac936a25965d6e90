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

#include "hcg_common.cuh"

namespace hcg {

template <bool kF32>
__global__ void __launch_bounds__(256)
pixelise_kernel(const double* __restrict__ lon_deg, const double* __restrict__ lat_deg,
                const float* __restrict__ values, const float* __restrict__ weights,
                int nchan, int64_t n, Region rg, uint32_t* __restrict__ keys,
                uint32_t* __restrict__ idx, Rec32* __restrict__ rec) {
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
    idx[i] = (uint32_t)i;
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

__global__ void __launch_bounds__(256)
pack64_kernel(const uint32_t* __restrict__ skeys, const uint32_t* __restrict__ sidx, int64_t n,
              uint32_t sentinel, const double* __restrict__ lon_deg, const double* __restrict__ lat_deg,
              const float* __restrict__ weights, Rec64* __restrict__ rec_out) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    if (skeys[i] == sentinel) return;
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
    const size_t nn = (size_t)(n > 0 ? n : 1);
    HCG_CUDA(c, c->d_keys.ensure(nn * 4));
    HCG_CUDA(c, c->d_keys_out.ensure(nn * 4));
    HCG_CUDA(c, c->d_idx.ensure(nn * 4));
    HCG_CUDA(c, c->d_idx_out.ensure(nn * 4));
    HCG_CUDA(c, c->d_bins.ensure(((size_t)rg.nbins + 2) * 4));
    HCG_CUDA(c, c->d_rec.ensure(nn * (f32 ? sizeof(Rec32) : sizeof(Rec64)) + 64));
    if (f32) HCG_CUDA(c, c->d_misc.ensure(nn * sizeof(Rec32)));
    int end_bit = 1;
    while (end_bit < 32 && ((uint64_t)1 << end_bit) <= (uint64_t)rg.nbins) ++end_bit;
    size_t tmp_bytes = 0;
    HCG_CUDA(c, cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, c->d_keys.as<uint32_t>(),
                                                c->d_keys_out.as<uint32_t>(), c->d_idx.as<uint32_t>(),
                                                c->d_idx_out.as<uint32_t>(), (int64_t)nn, 0, end_bit, st));
    HCG_CUDA(c, c->d_sort_tmp.ensure(tmp_bytes + 16));

    const int threads = 256;
    const unsigned nb = (unsigned)((nn + threads - 1) / threads);
    int launches = 0;
    if (c->opt_profile) cudaEventRecord(c->ev[0], st);
    if (n > 0) {
        if (f32)
            pixelise_kernel<true><<<nb, threads, 0, st>>>(lon, lat, values, weights, nchan, n, rg,
                                                          c->d_keys.as<uint32_t>(), c->d_idx.as<uint32_t>(),
                                                          c->d_misc.as<Rec32>());
        else
            pixelise_kernel<false><<<nb, threads, 0, st>>>(lon, lat, values, weights, nchan, n, rg,
                                                           c->d_keys.as<uint32_t>(), c->d_idx.as<uint32_t>(),
                                                           nullptr);
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
    if (n > 0 && !f32) {
        pack64_kernel<<<nb, threads, 0, st>>>(c->d_keys_out.as<uint32_t>(), c->d_idx_out.as<uint32_t>(), n,
                                              (uint32_t)rg.nbins, lon, lat, weights, c->d_rec.as<Rec64>());
        ++launches;
        HCG_CUDA(c, cudaGetLastError());
    }
    if (c->opt_profile) cudaEventRecord(c->ev[4], st);
    c->stats.gpu_launches = launches;
    return HCGRID_OK;
}

}  // namespace hcg
