// convolve.cu -- step a6: the gather-style convolution (Sect. 3.4 i-v;
// Eq. 1; kernel PAPER.md:186), hand-written for sm_100a.
//
// Organisation: one WARP owns a task = G consecutive cells of a strip
// (the paper's thread coarsening, at warp scope) and its 32 lanes stride
// over the candidate samples, so every load is a contiguous slice of S' and every cell
// gets 32 partial sums that are combined with shuffles -- no atomics anywhere.
//   step (i)   ring range of the disc: the strip's precomputed RingWin row (a1)
//   step (ii)  per ring, lane k turns the disc's longitude extent into a bin range
//   step (iii) two per-pixel-table reads give the sample range [S_start, S_end)
//   step (iv)  the ranges of all rings are concatenated into one candidate stream; in the
//              staged kernel each lane issues ONE bulk async copy (cp.async.bulk, the
//              TMA engine) of its ring's slice into the warp's shared-memory buffer, so
//              the stream is flattened by the copy engine, double-buffered on mbarriers
//   step (v)   pair arithmetic on exact fixed-point coordinate differences in fp32.
#include <cstdarg>
#include <cstring>

#include "hcg_conv.cuh"

namespace hcg {

template <int G>
struct Acc32 {
    float W[G], S[G];
    int cnt[G];
};

// Step (v) for one candidate against the G cells of the task.  Coordinates: exact integer
// differences of the fixed-point positions -> fp32 radians; 4 hav(d) from the small-angle
// series h4 = u(1-u/12) + cos(phi_c)cos(phi_s) v(1-v/12), u = dphi^2, v = dlam^2; accept
// iff h4 <= 4 sin^2(R/2); d^2 = h4(1+h4/12); w = 2^(-d^2 log2e / 2 sigma^2).
template <int G, bool HASQ>
__device__ __forceinline__ void pair_update(const Rec32& r, const TaskConst& tc, Acc32<G>& acc) {
    const float dx0 = (float)(int)(r.xi - tc.xc0) * tc.qx;
    const float dy = (float)(int)(r.yi - tc.yc) * tc.qy;
    const float u = dy * dy;
    const float u2 = u * fmaf(u, -1.0f / 12.0f, 1.0f);
    const float C = fmaf(dy, fmaf(dy, fmaf(dy, tc.c3, tc.c2), tc.c1), tc.c0);
#pragma unroll
    for (int g = 0; g < G; ++g) {
        const float dx = fmaf((float)g, -tc.du, dx0);
        const float v = dx * dx;
        const float B = v * fmaf(v, -1.0f / 12.0f, 1.0f);
        const float h4 = fmaf(C, B, u2);
        const float e = h4 * fmaf(h4, tc.k2, tc.k1);
        float w = ex2_approx(e);
        if (HASQ) w *= r.q;
        if (h4 <= tc.h4max) {
            acc.W[g] += w;
            acc.S[g] = fmaf(w, r.v, acc.S[g]);
            acc.cnt[g] += 1;
        }
    }
}

template <int G>
__device__ __forceinline__ void task_finish(Acc32<G>& acc, int lane, int64_t cell0, int ncells,
                                            float* __restrict__ cube, float* __restrict__ wmap,
                                            int32_t* __restrict__ counts) {
#pragma unroll
    for (int g = 0; g < G; ++g) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            acc.W[g] += __shfl_xor_sync(0xffffffffu, acc.W[g], o);
            acc.S[g] += __shfl_xor_sync(0xffffffffu, acc.S[g], o);
            acc.cnt[g] += __shfl_xor_sync(0xffffffffu, acc.cnt[g], o);
        }
    }
#pragma unroll
    for (int g = 0; g < G; ++g) {
        if (lane == g && g < ncells) {
            const float W = acc.W[g];
            cube[cell0 + g] = W > 0.0f ? acc.S[g] / W : __int_as_float(0x7fc00000);
            wmap[cell0 + g] = W;
            if (counts) counts[cell0 + g] = acc.cnt[g];
        }
    }
}

// ------------------------------------------------------------------ kernel A: simple
// Warp per task, candidates read straight from global memory ring by ring.  Kept as the
// plainly-correct reference organisation (HCGRID_OPT_KERNEL = 1) and for kmax > 32.
template <int G, bool HASQ>
__global__ void __launch_bounds__(256)
conv1_simple_f32(const ConvArgs a) {
    const int lane = threadIdx.x & 31;
    const int64_t task = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (task >= a.ntasks) return;
    const int s = (int)(task / a.tasks_per_strip);
    const int ix0 = (int)(task % a.tasks_per_strip) * G;
    const int ncells = min(G, a.strip_cells - ix0);
    const Strip st = a.strips[s];
    const TaskConst tc = make_task_const(a, st, ix0);
    const Rec32* __restrict__ rec = (const Rec32*)a.rec;
    Acc32<G> acc;
#pragma unroll
    for (int g = 0; g < G; ++g) { acc.W[g] = 0.f; acc.S[g] = 0.f; acc.cnt[g] = 0; }
    for (int k = 0; k < st.nring; ++k) {
        const RingWin w = a.wins[(size_t)s * a.kmax + k];
        int sa, sn, sa2, sn2;
        ring_segment(w, ix0, ncells, a.rg, a.bin_start, sa, sn, sa2, sn2);
        for (int seg = 0; seg < 2; ++seg) {
            for (int i = lane; i < sn; i += 32) {
                const uint4 raw = __ldg((const uint4*)(rec + sa + i));
                Rec32 r;
                r.xi = raw.x; r.yi = raw.y; r.idx = raw.z; r.q = __uint_as_float(raw.w);
                pair_update<G, HASQ>(r, tc, acc);
            }
            sa = sa2; sn = sn2;     // second range: only where the window crosses the seam of a full-circle region
            if (sn == 0) break;
        }
    }
    task_finish<G>(acc, lane, (int64_t)s * a.strip_cells + ix0, ncells, (float*)a.cube, (float*)a.wmap, a.counts);
}

// ------------------------------------------------------------------ kernel B: staged (TMA)
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "W_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra D_%=;\n\t"
        "bra W_%=;\n\t"
        "D_%=:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

// Persistent warps; each warp walks tasks  warp_id, warp_id + nwarps, ...  Every task is a
// stream of `total` candidates cut into chunks of a.chunk records; chunk j+1 (possibly the
// first chunk of the NEXT task) is in flight while chunk j is computed.
template <int G, bool HASQ>
__global__ void __launch_bounds__(128)
conv1_staged_f32(const ConvArgs a) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int lane = threadIdx.x & 31;
    const int wib = threadIdx.x >> 5;
    const int nwib = blockDim.x >> 5;
    const int64_t nwarps = (int64_t)gridDim.x * nwib;
    const int64_t warp_id = (int64_t)blockIdx.x * nwib + wib;
    const int CH = a.chunk;
    Rec32* buf0 = (Rec32*)(smem + (size_t)wib * 2 * CH * sizeof(Rec32));
    Rec32* buf1 = buf0 + CH;
    uint64_t* bars = (uint64_t*)(smem + (size_t)nwib * 2 * CH * sizeof(Rec32)) + wib * 2;
    const uint32_t bar0 = smem_u32(bars), bar1 = smem_u32(bars + 1);
    if (lane == 0) {
        mbar_init(bar0, 1);
        mbar_init(bar1, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
    const Rec32* __restrict__ rec = (const Rec32*)a.rec;

    // per-lane segment state of a task: lane k owns ring k of the strip's table row
    struct Segs { int a, n, p, total; int s, ix0, ncells; };
    auto prepare = [&](int64_t task, Segs& sg) {
        sg.s = (int)(task / a.tasks_per_strip);
        sg.ix0 = (int)(task % a.tasks_per_strip) * G;
        sg.ncells = min(G, a.strip_cells - sg.ix0);
        const int nring = a.strips[sg.s].nring;
        sg.a = 0; sg.n = 0;
        if (lane < nring) {
            const RingWin w = a.wins[(size_t)sg.s * a.kmax + lane];
            ring_segment(w, sg.ix0, sg.ncells, a.rg, a.bin_start, sg.a, sg.n);
        }
        int incl = sg.n;                       // inclusive prefix sum over lanes
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        sg.p = incl - sg.n;
        sg.total = __shfl_sync(0xffffffffu, incl, 31);
    };
    auto issue = [&](const Segs& sg, int chunk, Rec32* buf, uint32_t bar) {
        const int c0 = chunk * CH;
        const int c1 = min(c0 + CH, sg.total);
        const int lo = max(sg.p, c0), hi = min(sg.p + sg.n, c1);
        if (lane == 0) mbar_expect_tx(bar, (uint32_t)(c1 - c0) * (uint32_t)sizeof(Rec32));
        __syncwarp();
        if (hi > lo)
            bulk_g2s(smem_u32(buf + (lo - c0)), rec + sg.a + (lo - sg.p), (uint32_t)(hi - lo) * (uint32_t)sizeof(Rec32), bar);
    };

    int64_t task = warp_id;
    if (task >= a.ntasks) return;
    Segs cur, nxt;
    prepare(task, cur);
    int chunk = 0;                 // chunk of `cur` that sits (or is arriving) in buffer `b`
    int b = 0;
    uint32_t ph0 = 0, ph1 = 0;     // phase parity of the two barriers
    if (cur.total > 0) issue(cur, 0, buf0, bar0);
    Acc32<G> acc;
#pragma unroll
    for (int g = 0; g < G; ++g) { acc.W[g] = 0.f; acc.S[g] = 0.f; acc.cnt[g] = 0; }
    TaskConst tc = make_task_const(a, a.strips[cur.s], cur.ix0);

    while (true) {
        const int nchunks = (cur.total + CH - 1) / CH;
        const bool have_chunk = chunk < nchunks;
        const bool last = chunk + 1 >= nchunks;
        // the chunk that follows goes to the other buffer (or to this one if it is unused)
        const int nb = have_chunk ? (b ^ 1) : b;
        bool have_next_task = false;
        if (!last) {
            issue(cur, chunk + 1, nb ? buf1 : buf0, nb ? bar1 : bar0);
        } else {
            const int64_t t2 = task + nwarps;
            if (t2 < a.ntasks) {
                have_next_task = true;
                prepare(t2, nxt);                  // empty tasks still have outputs to write
                if (nxt.total > 0) issue(nxt, 0, nb ? buf1 : buf0, nb ? bar1 : bar0);
            }
        }
        if (have_chunk) {
            const Rec32* buf = b ? buf1 : buf0;
            mbar_wait(b ? bar1 : bar0, b ? ph1 : ph0);
            if (b) ph1 ^= 1; else ph0 ^= 1;
            const int cnt = min(CH, cur.total - chunk * CH);
            for (int i = lane; i < cnt; i += 32) {
                const uint4 raw = *(const uint4*)(buf + i);
                Rec32 r;
                r.xi = raw.x; r.yi = raw.y; r.idx = raw.z; r.q = __uint_as_float(raw.w);
                pair_update<G, HASQ>(r, tc, acc);
            }
            __syncwarp();
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        }
        b = nb;
        if (!last) { ++chunk; continue; }
        task_finish<G>(acc, lane, (int64_t)cur.s * a.strip_cells + cur.ix0, cur.ncells,
                       (float*)a.cube, (float*)a.wmap, a.counts);
        if (!have_next_task) break;
        task += nwarps;
        cur = nxt;
        chunk = 0;
#pragma unroll
        for (int g = 0; g < G; ++g) { acc.W[g] = 0.f; acc.S[g] = 0.f; acc.cnt[g] = 0; }
        tc = make_task_const(a, a.strips[cur.s], cur.ix0);
    }
}


// ------------------------------------------------------------------ launcher
template <int G>
static int launch_f32(hcgrid_ctx* c, ConvArgs& a, bool hasq, bool staged, cudaStream_t st) {
    a.coarsen = G;
    a.tasks_per_strip = (a.strip_cells + G - 1) / G;
    a.ntasks = (int64_t)a.tasks_per_strip * c->nstrip;
    if (a.ntasks == 0) return HCGRID_OK;
    if (!staged) {
        const unsigned blocks = (unsigned)((a.ntasks + 7) / 8);
        if (hasq) conv1_simple_f32<G, true><<<blocks, 256, 0, st>>>(a);
        else conv1_simple_f32<G, false><<<blocks, 256, 0, st>>>(a);
    } else {
        const int wpb = 4;
        const int warps_sm = c->opt_warps > 0 ? c->opt_warps : 32;
        const int blocks_sm = (warps_sm + wpb - 1) / wpb;
        // two staging buffers per warp, sized so blocks_sm blocks fit the SM's shared memory
        int chunk = (int)((200 * 1024 / blocks_sm - 64) / (wpb * 2 * sizeof(Rec32)));
        chunk = chunk > 512 ? 512 : chunk & ~31;
        if (chunk < 32) chunk = 32;
        a.chunk = chunk;
        const size_t smem = (size_t)wpb * 2 * chunk * sizeof(Rec32) + wpb * 2 * sizeof(uint64_t);
        int64_t blocks = (int64_t)blocks_sm * c->num_sms;
        const int64_t need = (a.ntasks + wpb - 1) / wpb;
        if (blocks > need) blocks = need;
        auto k = hasq ? conv1_staged_f32<G, true> : conv1_staged_f32<G, false>;
        HCG_CUDA(c, cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        k<<<(unsigned)blocks, wpb * 32, smem, st>>>(a);
    }
    HCG_CUDA(c, cudaGetLastError());
    return HCGRID_OK;
}

// n_hit of hcgrid_stats: the sum of the count output (profiling only)
__global__ void __launch_bounds__(256) sum_counts_kernel(const int32_t* __restrict__ counts, int64_t ncell, unsigned long long* out) {
    long long s = 0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < ncell; i += (int64_t)gridDim.x * blockDim.x) s += counts[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0 && s != 0) atomicAdd(out, (unsigned long long)s);   // integer: order-independent
}

// the lookup tables and constants every strip kernel takes (no input or output arrays yet)
static ConvArgs lookup_args(const hcgrid_ctx* c) {
    const Region& rg = c->region;
    ConvArgs a{};
    a.strips = c->d_strips.as<Strip>();
    a.wins = c->d_wins.as<RingWin>();
    a.bin_start = c->d_bins.as<int32_t>();
    a.rec = c->d_rec.p;
    a.rg = rg; a.kp = c->kp;
    a.kmax = c->kmax; a.strip_cells = c->strip_cells;
    a.raw = c->raw_sums ? 1 : 0;
    a.small64 = c->small_series_ok ? 1 : 0;   // R and the longitude half-window <= 0.05 rad, no pole in reach
    a.qx = (float)(1.0 / rg.sx32);
    a.qy = (float)(1.0 / rg.sy32);
    a.sx = rg.sx32;
    return a;
}

// pairs the strip kernels (simple, staged, general) put to the distance test: every task of g cells tests each sample
// of its ring ranges against each of its cells; added to *out
__global__ void __launch_bounds__(256) strip_pairs_tested_kernel(const ConvArgs a, int g, unsigned long long* out) {
    const int64_t task = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long pairs = 0;
    if (task < a.ntasks) {
        const int s = (int)(task / a.tasks_per_strip);
        const int ix0 = (int)(task % a.tasks_per_strip) * g;
        const int ncells = min(g, a.strip_cells - ix0);
        const int nring = a.strips[s].nring;
        long long total = 0;
        for (int k = 0; k < nring; ++k) {
            int sa, sn, sa2, sn2;
            ring_segment(a.wins[(size_t)s * a.kmax + k], ix0, ncells, a.rg, a.bin_start, sa, sn, sa2, sn2);
            total += sn + sn2;
        }
        pairs = (unsigned long long)total * (unsigned long long)ncells;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) pairs += __shfl_xor_sync(0xffffffffu, pairs, o);
    if ((threadIdx.x & 31) == 0 && pairs) atomicAdd(out, pairs);
}

// The profiling-only figures of hcgrid_stats, after the timed stages: n_hit (sum of the count output) and, for the tile
// and the strip kernels, n_pairs_tested.
int run_profile_stats(hcgrid_ctx* c, int32_t* counts, cudaStream_t st) {
    c->stat_hit = c->stat_pairs = false;
    if (!c->opt_profile) return HCGRID_OK;
    HCG_CUDA(c, c->d_stat.ensure(16));
    HCG_CUDA(c, cudaMemsetAsync(c->d_stat.p, 0, 16, st));
    if (counts && !c->raw_sums) {
        sum_counts_kernel<<<4 * c->num_sms, 256, 0, st>>>(counts, c->ncell, c->d_stat.as<unsigned long long>());
        HCG_CUDA(c, cudaGetLastError());
        c->stat_hit = true;
    }
    if (c->stats.kernel == 6) {
        const int rc = launch_tile_pairs_tested(c, c->stats.coarsen, c->stats.coarsen_y, c->d_stat.as<unsigned long long>() + 1, st);
        if (rc != HCGRID_OK) return rc;
        c->stat_pairs = true;
    } else if (c->stats.kernel >= 1 && c->stats.kernel <= 5) {
        ConvArgs a = lookup_args(c);
        const int g = c->stats.coarsen > 0 ? c->stats.coarsen : 1;
        a.tasks_per_strip = (c->strip_cells + g - 1) / g;
        a.ntasks = (int64_t)a.tasks_per_strip * c->nstrip;
        if (a.ntasks > 0) {
            strip_pairs_tested_kernel<<<(unsigned)((a.ntasks + 255) / 256), 256, 0, st>>>(a, g, c->d_stat.as<unsigned long long>() + 1);
            HCG_CUDA(c, cudaGetLastError());
        }
        c->stat_pairs = true;
    }
    return HCGRID_OK;
}

int run_convolve(hcgrid_ctx* c, int64_t n, const float* values, int nchan, bool has_weights, void* cube,
                 void* wmap, int32_t* counts, cudaStream_t st) {
    const Region& rg = c->region;
    ConvArgs a = lookup_args(c);
    a.values = values;
    a.cube = cube; a.wmap = wmap; a.counts = counts;
    a.nchan = nchan;
    const bool f32 = c->precision == HCGRID_F32 && c->f32_series_ok && c->opt_kernel != 2;
    int rc;
    c->stats.coarsen_y = 1;
    c->stats.split = 1;
    if (c->kp.ktype != 0) {
        // kernel functions other than the paper's Gaussian: the tile kernel (one channel, plate-carree
        // target, fp32 mode) and the general kernels
        if (c->opt_kernel != 0 && c->opt_kernel != 2 && c->opt_kernel != 3 && c->opt_kernel != 5)
            return fail(c, HCGRID_ERR_UNSUPPORTED, "only the tile and the general kernels (HCGRID_OPT_KERNEL 0, 2, 3, "
                        "5) evaluate kernel functions other than the Gaussian");
        if (f32 && nchan == 1 && c->tile_ok && (c->opt_kernel == 0 || c->opt_kernel == 5)) {
            rc = launch_conv_tile(c, n, (float*)cube, (float*)wmap, counts, st);
            c->stats.kernel = 6;
            if (rc == HCGRID_OK) c->stats.gpu_launches += 1;
            return rc;
        }
        if (c->opt_kernel == 5)
            return fail(c, HCGRID_ERR_UNSUPPORTED, "the tile kernel needs fp32 mode, one channel and a plate-carree "
                        "target whose reach is a plain longitude window");
        rc = launch_conv_general(c, a, !f32, c->precision == HCGRID_F64, st);
        c->stats.coarsen = 1;
        c->stats.kernel = f32 ? 3 : (c->precision == HCGRID_F64 ? 5 : 4);
        if (rc == HCGRID_OK) c->stats.gpu_launches += 1;
        return rc;
    }
    if (c->opt_kernel == 5 && !(f32 && nchan == 1 && c->tile_ok))
        return fail(c, HCGRID_ERR_UNSUPPORTED, "the tile kernel needs fp32 mode, one channel and a plate-carree "
                    "target whose reach is a plain longitude window");
    const bool mc_ok = f32 && nchan > 1 && c->tile_ok && nchan % 4 == 0 && ((uintptr_t)values & 15) == 0 &&
                       ((uintptr_t)cube & 15) == 0;
    if (c->opt_kernel == 6 && !mc_ok)
        return fail(c, HCGRID_ERR_UNSUPPORTED, "the cube kernel needs fp32 mode, nchan a multiple of 4 (> 1), 16-byte "
                    "aligned values and datacube and a plate-carree target whose reach is a plain longitude window");
    // tensor-core cube kernel: channel blocks the MMA shapes allow (N a multiple of 32)
    const bool tc_ok = mc_ok && nchan % 32 == 0;
    if (c->opt_kernel == 7 && !tc_ok)
        return fail(c, HCGRID_ERR_UNSUPPORTED, "the tensor-core cube kernel needs what the cube kernel needs and nchan a "
                    "multiple of 32");
    if (tc_ok && (c->opt_kernel == 7 || (c->opt_kernel == 0 && nchan >= 64))) {
        const size_t nd = (size_t)mc_tc_tiles(c) * (size_t)((nchan + 255) / 256);
        HCG_CUDA(c, c->d_dirty.ensure((nd + (size_t)mc_tc_tiles(c) + 1) * 4));   // flags, list of flagged tiles, their count
        rc = launch_conv_mc_tc(c, values, nchan, (float*)cube, (float*)wmap, counts, c->d_dirty.as<int32_t>(), st);
        // tiles that met a non-finite value (0 * inf would poison all their cells) are redone cell by cell
        if (rc == HCGRID_OK) {
            a.counts = counts;
            rc = launch_conv_general(c, a, false, false, st, c->d_dirty.as<int32_t>());
        }
        c->stats.kernel = 8;
        if (rc == HCGRID_OK) c->stats.gpu_launches += 2;   // the list of flagged tiles and the pass over it
    } else if (mc_ok && (c->opt_kernel == 0 || c->opt_kernel == 6)) {
        rc = launch_conv_mc(c, values, nchan, (float*)cube, (float*)wmap, counts, st);
        c->stats.kernel = 7;
    } else if (f32 && nchan == 1 && c->tile_ok && (c->opt_kernel == 0 || c->opt_kernel == 5)) {
        rc = launch_conv_tile(c, n, (float*)cube, (float*)wmap, counts, st);
        c->stats.kernel = 6;
    } else if (f32 && nchan == 1 && c->opt_kernel != 3 && !c->raw_sums) {
        // the staged kernel keeps one sample range per ring: full-circle regions (two ranges on the seam) take the simple one
        const bool staged = c->opt_kernel != 1 && c->kmax <= 32 && !rg.full_circle;
        int G = c->opt_coarsen;
        if (G == 0) G = c->strip_cells >= 4 ? 2 : 1;
        if (G > c->strip_cells) G = 1;
        if (rg.full_circle) G = 1;   // longitude differences are taken modulo the circle: one cell per task
        switch (G) {
            case 1: rc = launch_f32<1>(c, a, has_weights, staged, st); break;
            case 2: rc = launch_f32<2>(c, a, has_weights, staged, st); break;
            case 4: rc = launch_f32<4>(c, a, has_weights, staged, st); break;
            case 8: rc = launch_f32<8>(c, a, has_weights, staged, st); break;
            default: return fail(c, HCGRID_ERR_INVALID_ARG, "coarsen %d not built (1,2,4,8)", G);
        }
        c->stats.coarsen = G;
        c->stats.kernel = staged ? 2 : 1;
    } else {
        rc = launch_conv_general(c, a, !f32, c->precision == HCGRID_F64, st);
        c->stats.coarsen = 1;
        c->stats.kernel = f32 ? 3 : (c->precision == HCGRID_F64 ? 5 : 4);
    }
    if (rc == HCGRID_OK) c->stats.gpu_launches += 1;
    return rc;
}

}  // namespace hcg
