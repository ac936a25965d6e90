// convolve_mc_tc.cu -- step a6 for spectral cubes on the 5th-generation tensor cores (tcgen05 + TMEM):
// Eq. 1 applied per channel with one kernel weight and one weight map for all channels
// (the paper lists multi-channel gridding as "underway"; reading c7 of DESIGN.md), the
// contributing samples found by the search of PAPER.md:134-140 (Sect. 3.4 i-v).  SURVEY.md 8f NEXT-1.
//
// For a tile of 128 target cells the weighted sums are a matrix product
//     S[cell][chan] = sum_k  A[cell][k] * B[k][chan],   A = q_k w(d(cell, k)),  B = spectrum of candidate k,
// over the K candidates that can reach the tile.  One CTA owns a tile of 16 x 8 cells (M = 128) and a
// block of up to 256 channels (N):
//   * one warp builds the candidate stream of the tile (ring table, lookup-bin windows: steps i-iii, as
//     in convolve_tile.cu) and keeps the candidates whose distance to the tile's rectangle of cell
//     centres is within R: compaction in stream order into a FIFO of 16-candidate groups, each entry
//     with a 4-bit mask of the 8 x 4-cell quarters of the tile the candidate can reach;
//   * 8 compute warps evaluate A per stage (= group) of 16 candidates: thread = cell, a warp = one
//     quarter of the tile, which visits only the candidates that can reach it, two at a time; the tile
//     kernel's fp32 pair arithmetic on exact fixed-point differences; every weight is split
//     w = hi + lo (hi = w rounded to TF32) and both go to the UMMA K-major core-matrix layout;
//   * 2 warps copy the candidates' spectrum rows IN PLACE from `values` (never moved: a5) with cp.async
//     into the UMMA MN-major SWIZZLE_128B_BASE32B layout, two stages ahead, and write
//     lo = v - trunc_tf32(v) beside them (the tensor core itself ignores the low 13 bits of v);
//   * one thread issues, per 8 candidates, three tcgen05.mma.kind::tf32 (hi*v, lo*v, hi*lo_v: 3xTF32,
//     product error <= ~3e-6 relative) into a 128 x 256 fp32 accumulator in TMEM;
//   * the tensor core adds with round-toward-zero (measured: -3.4e-8 relative per update), so the
//     TMEM accumulator only ever holds a CHUNK of 8 stages (48 updates) -- two accumulators alternate,
//     and the compute warps add every finished chunk into fp32 registers (round-to-nearest, 128
//     channels x 1 cell per thread), which also makes the epilogue a plain divide and store.
// W and the counts are summed on the CUDA cores from the same weights.  No atomics in the sums; the
// order of the additions is fixed by the stream order, so results are bit-wise reproducible.
// Odd tile rows walk the rings south to north, so vertically adjacent tiles, which run at the same
// time, meet the spectrum rows they share at about the same time (L2 instead of HBM).
// A non-finite value would poison a whole tile through 0 * inf; tiles whose sums came out non-finite
// are flagged and recomputed cell by cell by conv_general, which keeps reading c8 exact.
#include "hcg_tile.cuh"

namespace hcg {

struct McTcArgs {
    TileArgs t;            // tiles_x / ntiles count tiles of 16 x 8 cells
    const float* values;   // [n][nchan], channel fastest, in input order
    int32_t nchan;
    int32_t* dirty;        // [gridDim.y][ntiles]: 1 where the sums came out non-finite
};

constexpr int kTcTX = 16, kTcTY = 8;           // tile = 128 cells = MMA M
constexpr int kTcCW = 8;                       // compute warps
constexpr int kTcCT = kTcCW * 32;              // compute threads
constexpr int kTcThreads = kTcCT + 128;        // + the service warpgroup: MMA issuer, stream builder, two spectrum-row warps
constexpr int kTcBW = 2;                       // spectrum-row (B) warps
constexpr int kTcNS = 4;                       // pipeline stages
constexpr int kTcP = 2;                        // stages the spectrum rows are requested ahead
constexpr int kTcCH = 8;                       // stages per TMEM accumulator chunk
constexpr int kTcGroups = 64;                  // FIFO: groups of 16 candidates (one group = one stage)
constexpr int kTcFifo = kTcGroups * 16;
constexpr int kTcRings = 128;                  // ring-table entries per pass
constexpr int kOffAhi = 0, kOffAlo = 8192, kOffBraw = 16384, kOffBlo = 32768, kStageBytes = 49152;
constexpr int kOffFifoC = kTcNS * kStageBytes;             // uint4 [kTcFifo]: xi, yi, cos(lat_s), q
constexpr int kOffFifoI = kOffFifoC + kTcFifo * 16;        // uint32 [kTcFifo]: sample index
constexpr int kOffFifoM = kOffFifoI + kTcFifo * 4;         // uint8 [kTcFifo]: quarters of the tile within reach
constexpr int kOffTabBase = kOffFifoM + kTcFifo;           // u64 [kTcRings]
constexpr int kOffTabEnd = kOffTabBase + kTcRings * 8;     // int [kTcRings]
constexpr int kOffGrpN = kOffTabEnd + kTcRings * 4;        // uint32 [kTcGroups]: candidates in the group | 0x80 (last group of the tile)
constexpr int kOffBars = kOffGrpN + kTcGroups * 4;         // u64: full[NS], empty[NS], dfull[2], dempty[2], cfull[G], cempty[G]
constexpr int kOffMisc = kOffBars + 8 * (2 * kTcNS + 4 + 2 * kTcGroups);
constexpr int kTcSmem = kOffMisc + 64;

// ---- PTX wrappers
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// Bounded: a wait that outlasts any legitimate one (seconds) is a broken pipeline -- fail loudly, do not hang.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    for (uint32_t spins = 0;; ++spins) {
        uint32_t ok;
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (ok) return;
        if (spins > (1u << 22)) __trap();
    }
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void umma_tf32(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t addr, uint32_t (&v)[32]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "
                 "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
                 "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                   "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
                   "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
                   "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
                 : "r"(addr) : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void bar_compute() { asm volatile("bar.sync 1, %0;" ::"n"(kTcCT) : "memory"); }
__device__ __forceinline__ void cp_async16_cg(uint32_t dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ uint4 lds_u4(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ uint2 lds_u2(uint32_t addr) {
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t lds_u1(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void sts_u4(uint32_t addr, uint4 v) {
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
// keep a loop-invariant value in its register (ptxas otherwise recomputes it from the thread index every iteration)
#define HCG_PIN(x) asm volatile("" : "+r"(x))

// UMMA shared-memory matrix descriptor: start address, leading / stride byte offsets (all >> 4), version 1,
// layout type (0: no swizzle, 1: SWIZZLE_128B_BASE32B -- the only MN-major layout of 32-bit operands)
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo, uint32_t layout) {
    return (uint64_t)((saddr >> 4) & 0x3fffu) | ((uint64_t)((lbo >> 4) & 0x3fffu) << 16) |
           ((uint64_t)((sbo >> 4) & 0x3fffu) << 32) | ((uint64_t)1 << 46) | ((uint64_t)(layout & 7u) << 61);
}
// instruction descriptor: fp32 accumulate, TF32 x TF32, A K-major, B MN-major, M = 128, N
__device__ __forceinline__ uint32_t umma_idesc_tf32(int n) {
    return (1u << 4) | (2u << 7) | (2u << 10) | (0u << 15) | (1u << 16) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
}

template <int MODE, bool COUNTS>
__global__ void __launch_bounds__(kTcThreads, 1)
conv_mc_tc_f32(const McTcArgs m) {
    const TileArgs& a = m.t;
    extern __shared__ __align__(1024) unsigned char s_tc[];
    const uint32_t s_base = smem_addr(s_tc);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t b_full = s_base + kOffBars, b_empty = b_full + 8 * kTcNS, b_dfull = b_empty + 8 * kTcNS, b_dempty = b_dfull + 16;
    const uint32_t b_cfull = b_dempty + 16, b_cempty = b_cfull + 8 * kTcGroups;
    volatile uint32_t* s_flag = (volatile uint32_t*)(s_tc + kOffMisc);   // [NS] stage flags
    uint32_t* s_tmem = (uint32_t*)(s_tc + kOffMisc + 4 * kTcNS);
    int* s_bad = (int*)(s_tmem + 1);

    const int tile = blockIdx.x;
    const int ch0 = blockIdx.y * 256;
    const int nch = min(256, m.nchan - ch0);                        // channels of this block (multiple of 32)
    const int ty = tile / a.tiles_x;
    const int ix0 = (tile - ty * a.tiles_x) * kTcTX;
    const int row0 = ty * kTcTY;
    const int ncols = min(kTcTX, a.nx - ix0);
    const int nrows = min(kTcTY, a.ny - row0);

    if (warp == kTcCW) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_addr(s_tmem)), "r"(512u));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::);
        if (lane == 0) {
            for (int s = 0; s < kTcNS; ++s) { mbar_init(b_full + 8 * s, kTcCW + kTcBW); mbar_init(b_empty + 8 * s, 1); }
            for (int b = 0; b < 2; ++b) { mbar_init(b_dfull + 8 * b, 1); mbar_init(b_dempty + 8 * b, kTcCW); }
            for (int j = 0; j < kTcGroups; ++j) { mbar_init(b_cfull + 8 * j, 1); mbar_init(b_cempty + 8 * j, kTcCW + kTcBW); }
            *s_bad = 0;
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tm = *s_tmem;

    if (warp >= kTcCW) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 64;");       // the whole service warpgroup, one instruction
        if (warp == kTcCW) {
            // ============================================================ MMA issuer (lane 0 issues; the warp stays converged)
            const uint32_t idesc = umma_idesc_tf32(nch);
            const uint64_t a_hi0 = umma_desc(s_base + kOffAhi, 2048, 128, 0), a_lo0 = umma_desc(s_base + kOffAlo, 2048, 128, 0);
            const uint64_t b_rw0 = umma_desc(s_base + kOffBraw, 1024, 512, 1), b_lo0 = umma_desc(s_base + kOffBlo, 1024, 512, 1);
            for (int s = 0;; ++s) {
                const int slot = s % kTcNS;
                mbar_wait(b_full + 8 * slot, (uint32_t)(s / kTcNS) & 1u);
                const uint32_t flag = s_flag[slot];
                tc_fence_after();
                if (!(flag & 2u)) {
                    const int chunk = s / kTcCH, buf = chunk & 1;
                    const bool first = s % kTcCH == 0;
                    if (first && chunk >= 2) {
                        mbar_wait(b_dempty + 8 * buf, (uint32_t)((chunk >> 1) - 1) & 1u);
                        tc_fence_after();
                    }
                    if (lane == 0) {
                        const uint32_t d = tm + (uint32_t)buf * 256u;
                        const uint64_t so = (uint64_t)((uint32_t)slot * (kStageBytes >> 4));
#pragma unroll
                        for (int ks = 0; ks < 2; ++ks) {
                            const uint64_t ah = a_hi0 + so + (uint64_t)(ks * (4096 >> 4)), al = a_lo0 + so + (uint64_t)(ks * (4096 >> 4));
                            const uint64_t br = b_rw0 + so + (uint64_t)(ks * (8192 >> 4)), bl = b_lo0 + so + (uint64_t)(ks * (8192 >> 4));
                            umma_tf32(d, ah, br, idesc, (first && ks == 0) ? 0u : 1u);
                            umma_tf32(d, al, br, idesc, 1u);
                            umma_tf32(d, ah, bl, idesc, 1u);
                        }
                        tc_commit(b_empty + 8 * slot);
                        if (s % kTcCH == kTcCH - 1 || (flag & 1u)) tc_commit(b_dfull + 8 * buf);
                    }
                    __syncwarp();
                }
                if (flag & 1u) break;
            }
        } else if (warp == kTcCW + 1) {
            // ============================================================ stream builder: steps (i)-(iii) + compaction
            // Everything relative to a cell in the middle of the tile (the fixed-point differences are good for +- 8
            // columns / rows plus the support radius: target.cu).
            uint32_t xc0 = 0, yc0 = 0;
            float cc0 = 0.f, p1 = 0.f, p2 = 0.f, p3 = 0.f, ccmin = 2.0f;
            float bxlo[2], bxhi[2], bylo[2], byhi[2];                // extents of the cell centres of the four 8 x 4 quarters
            int rmin = 0x7fffffff, rmax = -0x7fffffff;
            const float sxk = a.sxk, syk = a.syk, a12 = a.a12;
            {
                const int ic = ncols >> 1, jc = nrows >> 1;
                for (int j = 0; j < nrows; ++j) {
                    const int4 r0 = __ldg((const int4*)(a.rows + row0 + j));
                    ccmin = fminf(ccmin, __int_as_float(r0.w));
                    rmin = min(rmin, r0.y);
                    rmax = max(rmax, r0.y + r0.z - 1);
                    if (j == jc) {
                        const int4 r1 = __ldg((const int4*)(a.rows + row0 + j) + 1);
                        yc0 = (uint32_t)r0.x;
                        cc0 = __int_as_float(r0.w);
                        const float sc0 = __int_as_float(r1.x), ik = a.isk;
                        p1 = -sc0 * ik;
                        p2 = -0.5f * cc0 * ik * ik;
                        p3 = sc0 * ik * ik * ik * (1.0f / 6.0f);
                    }
                }
                xc0 = (uint32_t)(unsigned long long)__double2ll_rn((a.u0 + (double)(ix0 + ic) * a.du) * a.sx);
                const float pad = 1e-3f * sqrtf(a.hmax);             // slack for the fp32 rounding of the extents
#pragma unroll
                for (int b = 0; b < 2; ++b) {
                    // columns 8 b .. min(8 b + 7, ncols - 1), rows 4 b .. min(4 b + 3, nrows - 1); an empty quarter reaches nothing
                    const int c0 = 8 * b, c1 = min(8 * b + 7, ncols - 1), r0 = 4 * b, r1 = min(4 * b + 3, nrows - 1);
                    const float xa = (float)(c0 - ic) * a.duk, xb = (float)(c1 - ic) * a.duk;
                    const float ya = (float)(r0 - jc) * a.dyk, yb = (float)(r1 - jc) * a.dyk;
                    bxlo[b] = c1 >= c0 ? fminf(xa, xb) - pad : 1e30f; bxhi[b] = c1 >= c0 ? fmaxf(xa, xb) + pad : -1e30f;
                    bylo[b] = r1 >= r0 ? fminf(ya, yb) - pad : 1e30f; byhi[b] = r1 >= r0 ? fmaxf(ya, yb) + pad : -1e30f;
                }
                ccmin *= 0.999f;
            }
            const float fxw = (float)(a.du >= 0.0 ? ix0 : ix0 + ncols - 1);
            const float fxe = (float)(a.du >= 0.0 ? ix0 + ncols - 1 : ix0);
            const bool flip = (ty & 1) != 0;                          // odd tile rows walk the rings south to north
            const Rec32* __restrict__ rec = a.rec;
            unsigned long long* tab_base = (unsigned long long*)(s_tc + kOffTabBase);
            int* tab_end = (int*)(s_tc + kOffTabEnd);
            uint4* fifo_c = (uint4*)(s_tc + kOffFifoC);
            uint32_t* fifo_i = (uint32_t*)(s_tc + kOffFifoI);
            unsigned char* fifo_m = s_tc + kOffFifoM;
            volatile uint32_t* grp_n = (volatile uint32_t*)(s_tc + kOffGrpN);
            const float hlim = a.hmax * 1.0001f;

            auto fetch = [&](int i, int total) -> uint4 {            // record number i of this pass's stream
                if (i >= total) return make_uint4(0, 0, 0, 0);
                int lo = 0, hi = kTcRings - 1;                        // first ring whose end is beyond i
                while (lo < hi) {
                    const int mid = (lo + hi) >> 1;
                    if (tab_end[mid] > i) hi = mid; else lo = mid + 1;
                }
                return ldg_rec(tab_base[lo], i);
            };

            int gpos = 0, published = 0;                              // candidates kept so far (FIFO position, unwrapped); groups published
            for (int pass = 0; rmin + pass * kTcRings <= rmax; ++pass) {
                // ---- ring table of this pass: lane l of sub-pass t <-> ring number 32 t + l
                int run = 0;
                for (int t = 0; t < kTcRings / 32; ++t) {
                    const int ro = pass * kTcRings + 32 * t + lane;
                    const int r = flip ? rmax - ro : rmin + ro;
                    int sa = 0, sn = 0;
                    if (r >= rmin && r <= rmax) {
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
                            sa = __ldg(bs + jlo);
                            sn = __ldg(bs + jhi + 1) - sa;
                        }
                    }
                    int incl = sn;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const int v = __shfl_up_sync(0xffffffffu, incl, o);
                        if (lane >= o) incl += v;
                    }
                    incl += run;
                    tab_end[32 * t + lane] = incl;
                    tab_base[32 * t + lane] = (unsigned long long)(uintptr_t)(rec + ((long long)sa - (incl - sn)));
                    run = __shfl_sync(0xffffffffu, incl, 31);
                }
                __syncwarp();
                const int total = run;
                // ---- the stream of this pass in blocks of 32, the next block's records in flight
                uint4 nxt = fetch(lane, total);
                for (int base = 0; base < total; base += 32) {
                    const uint4 raw = nxt;
                    nxt = fetch(base + 32 + lane, total);
                    unsigned reach = 0;
                    float cs = 0.f;
                    if (base + lane < total) {
                        const float X = (float)(int)(raw.x - xc0) * sxk;
                        const float Y = (float)(int)(raw.y - yc0) * syk;
                        cs = fmaf(Y, fmaf(Y, fmaf(Y, p3, p2), p1), cc0);
                        const float cmin = ccmin * cs;
                        float vx[2], uy[2];
#pragma unroll
                        for (int b = 0; b < 2; ++b) {
                            const float ex = fmaxf(fmaxf(bxlo[b] - X, X - bxhi[b]), 0.0f), ey = fmaxf(fmaxf(bylo[b] - Y, Y - byhi[b]), 0.0f);
                            vx[b] = ex * ex; uy[b] = ey * ey;
                            if (MODE >= 1) { vx[b] = vx[b] * fmaf(vx[b], -a12, 1.0f); uy[b] = uy[b] * fmaf(uy[b], -a12, 1.0f); }
                        }
#pragma unroll
                        for (int qq = 0; qq < 4; ++qq) reach |= fmaf(cmin, vx[qq & 1], uy[qq >> 1]) <= hlim ? 1u << qq : 0u;
                    }
                    const unsigned mk = __ballot_sync(0xffffffffu, reach != 0);
                    const int nk = __popc(mk);
                    if (nk == 0) continue;
                    // groups this block writes into for the first time must have been released by the compute warps
                    const int g_first = (gpos + 15) >> 4, g_last = (gpos + nk - 1) >> 4;
                    for (int gi = g_first; gi <= g_last; ++gi)
                        if (gi >= kTcGroups) mbar_wait(b_cempty + 8 * (gi % kTcGroups), (uint32_t)(gi / kTcGroups - 1) & 1u);
                    if (reach != 0) {
                        const int p = (gpos + __popc(mk & ((1u << lane) - 1u))) & (kTcFifo - 1);
                        fifo_c[p] = make_uint4(raw.x, raw.y, __float_as_uint(cs), raw.w);
                        fifo_i[p] = raw.z;
                        fifo_m[p] = (unsigned char)reach;
                    }
                    __syncwarp();
                    gpos += nk;
                    // publish the complete groups that are known not to be the last one (a later candidate exists)
                    const int p_end = (gpos - 1) >> 4;
                    if (lane == 0)
                        for (int gi = published; gi < p_end; ++gi) {
                            grp_n[gi % kTcGroups] = 16u;
                            mbar_arrive(b_cfull + 8 * (gi % kTcGroups));
                        }
                    published = max(published, p_end);
                }
            }
            // ---- the last group (1 .. 16 candidates; none at all: an empty group 0) carries the end-of-tile mark
            __syncwarp();
            if (lane == 0) {
                const int gi = gpos > 0 ? (gpos - 1) >> 4 : 0;
                grp_n[gi % kTcGroups] = (uint32_t)(gpos - 16 * gi) | 0x80u;
                mbar_arrive(b_cfull + 8 * (gi % kTcGroups));
            }
        } else {
            // ============================================================ spectrum rows (B): 64 threads, one 16-byte unit per row each
            const int t2 = (warp - kTcCW - 2) * 32 + lane;           // 0 .. 63
            const int upr = nch >> 2;                                 // 16-byte units per row (<= 64)
            const bool on = t2 < upr;
            uint32_t off_u[4];                                        // offset of unit t2 in a K-step's B region, by row & 3
#pragma unroll
            for (int k3 = 0; k3 < 4; ++k3)
                off_u[k3] = (uint32_t)((t2 >> 3) * 1024 + k3 * 128 + (((((t2 & 7) >> 1) ^ k3) << 5) | ((t2 & 1) << 4)));
            const unsigned long long vsrc = (unsigned long long)(uintptr_t)(m.values + ch0 + 4 * (on ? t2 : 0));
            const uint32_t vstride = (uint32_t)m.nchan * 4u;          // bytes per row
            const uint32_t fifo_i_s = s_base + kOffFifoI, grp_n_s = s_base + kOffGrpN;
            int nst = 0x7fffffff, pf = 0;
            for (int k = 0;; ++k) {
                // request the rows of the stages up to k + P (zeros for the missing rows of the last stage)
                while (pf <= k + kTcP) {
                    if (pf < nst) {
                        const int grp = pf % kTcGroups, slot = pf % kTcNS;
                        mbar_wait(b_cfull + 8 * grp, (uint32_t)(pf / kTcGroups) & 1u);
                        const uint32_t info = lds_u1(grp_n_s + 4u * (uint32_t)grp);
                        const int n = (int)(info & 31u);
                        if (info & 0x80u) nst = n > 0 ? pf + 1 : pf;
                        if (pf < nst) {
                            if (pf >= kTcNS) mbar_wait(b_empty + 8 * slot, (uint32_t)(pf / kTcNS - 1) & 1u);
                            const uint32_t sb = s_base + (uint32_t)slot * kStageBytes + kOffBraw;
                            if (on) {
                                uint32_t idx[16];
#pragma unroll
                                for (int r = 0; r < 16; ++r) idx[r] = lds_u1(fifo_i_s + (uint32_t)grp * 64u + 4u * r);
#pragma unroll
                                for (int r = 0; r < 16; ++r) {
                                    const uint32_t dst = sb + (uint32_t)((r >> 3) * 8192 + ((r >> 2) & 1) * 512) + off_u[r & 3];
                                    if (r < n) cp_async16_cg(dst, (const void*)(uintptr_t)(vsrc + (unsigned long long)idx[r] * vstride));
                                    else sts_u4(dst, make_uint4(0, 0, 0, 0));
                                }
                            }
                            __syncwarp();
                            if (lane == 0) mbar_arrive(b_cempty + 8 * grp);   // done with the group's sample indices
                        }
                    }
                    cp_commit();
                    ++pf;
                }
                if (k >= nst) {
                    if (nst == 0 && lane == 0) mbar_arrive(b_full);   // empty tile: the compute warps release the MMA warp through stage 0
                    break;
                }
                // the rows of stage k have landed (each thread reads back its own bytes): lo = v - trunc_tf32(v)
                cp_wait<kTcP>();
                const int slot = k % kTcNS;
                const uint32_t sb = s_base + (uint32_t)slot * kStageBytes + kOffBraw;
                if (on) {
#pragma unroll
                    for (int r0 = 0; r0 < 16; r0 += 4) {
                        uint4 v[4];
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            const int r = r0 + j;
                            v[j] = lds_u4(sb + (uint32_t)((r >> 3) * 8192 + ((r >> 2) & 1) * 512) + off_u[r & 3]);
                        }
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            const int r = r0 + j;
                            uint4 l;
                            l.x = __float_as_uint(__uint_as_float(v[j].x) - __uint_as_float(v[j].x & 0xffffe000u));
                            l.y = __float_as_uint(__uint_as_float(v[j].y) - __uint_as_float(v[j].y & 0xffffe000u));
                            l.z = __float_as_uint(__uint_as_float(v[j].z) - __uint_as_float(v[j].z & 0xffffe000u));
                            l.w = __float_as_uint(__uint_as_float(v[j].w) - __uint_as_float(v[j].w & 0xffffe000u));
                            sts_u4(sb + (uint32_t)(kOffBlo - kOffBraw + (r >> 3) * 8192 + ((r >> 2) & 1) * 512) + off_u[r & 3], l);
                        }
                    }
                }
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                __syncwarp();
                if (lane == 0) mbar_arrive(b_full + 8 * slot);
            }
            cp_wait<0>();
        }
    } else {
        // ================================================================ producers of A and B, accumulators
        asm volatile("setmaxnreg.inc.sync.aligned.u32 216;");
        // MMA row (= TMEM lane) 32 q + l  <->  cell (8 (q & 1) + (l & 7), 4 (q >> 1) + (l >> 3)): a warp owns an
        // 8 x 4-cell quarter of the tile; g selects the K-step of a stage (A) and the channel half (drain).
        const int q = warp & 3, g = warp >> 2;
        const int cell = q * 32 + lane;
        const int cix = 8 * (q & 1) + (lane & 7), ciy = 4 * (q >> 1) + (lane >> 3);
        const bool cell_ok = cix < ncols && ciy < nrows;
        uint32_t xc, yc;
        float cc;
        {
            const int4 r0 = __ldg((const int4*)(a.rows + min(row0 + ciy, a.ny - 1)));
            yc = (uint32_t)r0.x;
            cc = __int_as_float(r0.w);
            xc = (uint32_t)(unsigned long long)__double2ll_rn((a.u0 + (double)(ix0 + min(cix, ncols - 1)) * a.du) * a.sx);
        }
        float hm = cell_ok ? a.hmax : -1.0f;
        const float sxk = a.sxk, syk = a.syk, a12 = a.a12;
        HCG_PIN(xc); HCG_PIN(yc);
        asm volatile("" : "+f"(cc), "+f"(hm));
        const uint32_t fifo_c_s = s_base + kOffFifoC, fifo_m_s = s_base + kOffFifoM;
        const uint32_t grp_n_s = s_base + kOffGrpN;

        // ---- A: this thread owns the 8 candidates of K-step g of a stage for its cell (rows of 8 weights: two 16-byte halves)
        uint32_t a_off = (uint32_t)(g * 4096 + (cell >> 3) * 128 + (cell & 7) * 16);
        HCG_PIN(a_off);

        float acc[128];
#pragma unroll
        for (int j = 0; j < 128; ++j) acc[j] = 0.0f;
        float wsum = 0.0f;
        int csum = 0;

        auto drain = [&](int j) {
            const int buf = j & 1;
            mbar_wait(b_dfull + 8 * buf, (uint32_t)(j >> 1) & 1u);
            tc_fence_after();
            const uint32_t ta = tm + ((uint32_t)(q * 32) << 16) + (uint32_t)(buf * 256 + g * 128);
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                uint32_t v[32];
                tmem_ld32(ta + 32 * h, v);
                tmem_ld_wait();
#pragma unroll
                for (int c = 0; c < 32; ++c) acc[32 * h + c] += __uint_as_float(v[c]);
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(b_dempty + 8 * buf);
        };

        // one candidate of the group against this thread's cell: q w(d) where d <= R, else 0
        auto pair_weight = [&](const uint4 e) -> float {
            const float dy = (float)(int)(e.y - yc) * syk;
            const float dx = (float)(int)(e.x - xc) * sxk;
            float u = dy * dy, v = dx * dx;
            if (MODE >= 1) { u = u * fmaf(u, -a12, 1.0f); v = v * fmaf(v, -a12, 1.0f); }
            const float h = fmaf(cc * __uint_as_float(e.z), v, u);
            const float ee = MODE == 2 ? h * fmaf(h, a12, 1.0f) : h;
            const float w = ex2_approx(-ee) * __uint_as_float(e.w);
            const bool hit = h <= hm;
            if (COUNTS) csum += hit ? 1 : 0;
            return hit ? w : 0.0f;
        };
        auto store_weight = [&](uint32_t ad, int j, float ws) {     // slot j of the K-step: hi and lo parts
            const float hi = __uint_as_float((__float_as_uint(ws) + 0x1000u) & 0xffffe000u);
            const uint32_t p = ad + (uint32_t)((j >> 2) * 2048 + (j & 3) * 4);
            asm volatile("st.shared.f32 [%0], %1;" ::"r"(p + kOffAhi), "f"(hi) : "memory");
            asm volatile("st.shared.f32 [%0], %1;" ::"r"(p + kOffAlo), "f"(ws - hi) : "memory");
        };

        int k = 0, jd = 0, nst = 0x7fffffff;
        for (;;) {
            if (k >= nst) break;                                     // the last group has been seen
            mbar_wait(b_cfull + 8 * (k % kTcGroups), (uint32_t)(k / kTcGroups) & 1u);
            const uint32_t info = lds_u1(grp_n_s + 4u * (uint32_t)(k % kTcGroups));
            const int ng = (int)(info & 31u);
            if (info & 0x80u) nst = ng > 0 ? k + 1 : k;
            if (k >= nst) break;
            const int slot = k % kTcNS;
            if (k >= kTcNS) mbar_wait(b_empty + 8 * slot, (uint32_t)(k / kTcNS - 1) & 1u);
            const uint32_t ad = s_base + (uint32_t)slot * kStageBytes + a_off;

            // ---- A: the candidates of K-step g that can reach this warp's quarter, two at a time; zeros elsewhere
            {
                const uint32_t e0 = (uint32_t)(k % kTcGroups) * 16u + (uint32_t)g * 8u;   // FIFO index of the first
                const uint2 mk = lds_u2(fifo_m_s + e0);
                sts_u4(ad + kOffAhi, make_uint4(0, 0, 0, 0));
                sts_u4(ad + kOffAhi + 2048, make_uint4(0, 0, 0, 0));
                sts_u4(ad + kOffAlo, make_uint4(0, 0, 0, 0));
                sts_u4(ad + kOffAlo + 2048, make_uint4(0, 0, 0, 0));
                // bit j: candidate j of the K-step reaches quarter q (reach masks are bytes: bit q of byte j)
                const uint32_t sel = 0x01010101u << q;
                uint32_t live = 0;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    live |= ((mk.x & sel) >> (8 * j + q) & 1u) << j;
                    live |= ((mk.y & sel) >> (8 * j + q) & 1u) << (4 + j);
                }
                const int nk = ng - g * 8;                            // candidates present in this K-step (may be <= 0 or >= 8)
                live &= nk >= 8 ? 0xffu : (nk <= 0 ? 0u : (1u << nk) - 1u);
                while (live) {                                        // warp-uniform
                    const int j0 = __ffs(live) - 1;
                    live &= live - 1;
                    const bool two = live != 0;
                    const int j1 = two ? __ffs(live) - 1 : j0;
                    live &= live - 1;
                    const uint4 ea = lds_u4(fifo_c_s + (e0 + j0) * 16u), eb = lds_u4(fifo_c_s + (e0 + j1) * 16u);
                    const float wa = pair_weight(ea);
                    const float wb = two ? pair_weight(eb) : 0.0f;
                    wsum += wa;
                    wsum += wb;
                    store_weight(ad, j0, wa);
                    if (two) store_weight(ad, j1, wb);
                }
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            if (tid == 0) s_flag[slot] = k == nst - 1 ? 1u : 0u;
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(b_cempty + 8 * (k % kTcGroups));          // this warp is done with the group's FIFO entries
                mbar_arrive(b_full + 8 * slot);
            }
            if (k >= (jd + 1) * kTcCH + kTcNS) { drain(jd); ++jd; }
            ++k;
        }
        if (nst == 0) {                                              // nothing can reach this tile: release the MMA warp
            if (tid == 0) s_flag[0] = 3u;
            __syncwarp();
            if (lane == 0) mbar_arrive(b_full);
        }
        for (const int nchunk = (nst + kTcCH - 1) / kTcCH; jd < nchunk; ++jd) drain(jd);

        // ---- finish: W and counts over the two K-step halves of a cell (fixed order), normalise, store
        bar_compute();                                               // every warp is done with the FIFO: reuse it
        float* s_w = (float*)(s_tc + kOffFifoC);
        int* s_c = (int*)(s_w + 2 * 128);
        s_w[g * 128 + cell] = wsum;
        if (COUNTS) s_c[g * 128 + cell] = csum;
        // 0 * inf = NaN reaches every cell of the tile: non-finite sums flag the tile for the cell-by-cell pass
        float chk = 0.0f;
#pragma unroll
        for (int j = 0; j < 128; ++j) chk = fmaf(acc[j], 0.0f, chk);
        if (__any_sync(0xffffffffu, chk != 0.0f) && lane == 0) atomicOr(s_bad, 1);
        bar_compute();
        const float wtot = s_w[cell] + s_w[128 + cell];
        if (cell_ok) {
            const int64_t gc = (int64_t)(row0 + ciy) * a.nx + ix0 + cix;
            if (g == 0 && blockIdx.y == 0) {
                a.wmap[gc] = wtot;
                if (COUNTS) a.counts[gc] = s_c[cell] + s_c[128 + cell];
            }
            float* o = a.cube + (size_t)gc * m.nchan + ch0 + g * 128;
            const float nan = __int_as_float(0x7fc00000);
            const bool filled = wtot > 0.0f;
#pragma unroll
            for (int j = 0; j < 128; j += 4) {
                if (g * 128 + j < nch) {
                    float4 f;
                    f.x = a.raw ? acc[j] : (filled ? acc[j] / wtot : nan);
                    f.y = a.raw ? acc[j + 1] : (filled ? acc[j + 1] / wtot : nan);
                    f.z = a.raw ? acc[j + 2] : (filled ? acc[j + 2] / wtot : nan);
                    f.w = a.raw ? acc[j + 3] : (filled ? acc[j + 3] / wtot : nan);
                    *(float4*)(o + j) = f;
                }
            }
        }
        if (tid == 0 && m.dirty) m.dirty[(size_t)blockIdx.y * a.ntiles + tile] = *s_bad;
    }

    tc_fence_before();
    __syncthreads();
    if (warp == kTcCW) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tm), "r"(512u));
}

int launch_conv_mc_tc(hcgrid_ctx* c, const float* values, int nchan, float* cube, float* wmap, int32_t* counts,
                      int32_t* dirty, cudaStream_t st) {
    const int mode = tile_series_mode(c);
    McTcArgs m{};
    fill_tile_args(c, mode, m.t);
    m.t.cube = cube; m.t.wmap = wmap; m.t.counts = counts;
    m.t.tiles_x = (m.t.nx + kTcTX - 1) / kTcTX;
    m.t.ntiles = (int64_t)m.t.tiles_x * ((m.t.ny + kTcTY - 1) / kTcTY);
    m.values = values;
    m.nchan = nchan;
    m.dirty = dirty;
    const dim3 grid((unsigned)m.t.ntiles, (unsigned)((nchan + 255) / 256));
#define HCG_MCTC(M, C)                                                                                      \
    do {                                                                                                    \
        HCG_CUDA(c, cudaFuncSetAttribute(conv_mc_tc_f32<M, C>, cudaFuncAttributeMaxDynamicSharedMemorySize, kTcSmem)); \
        conv_mc_tc_f32<M, C><<<grid, kTcThreads, kTcSmem, st>>>(m);                                         \
    } while (0)
    switch (mode * 2 + (counts ? 1 : 0)) {
        case 0: HCG_MCTC(0, false); break;
        case 1: HCG_MCTC(0, true); break;
        case 2: HCG_MCTC(1, false); break;
        case 3: HCG_MCTC(1, true); break;
        case 4: HCG_MCTC(2, false); break;
        default: HCG_MCTC(2, true); break;
    }
#undef HCG_MCTC
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e, "conv_mc_tc_f32");
    c->stats.coarsen = kTcTX;
    c->stats.coarsen_y = kTcTY;
    return HCGRID_OK;
}

int mc_tc_tiles(const hcgrid_ctx* c) {
    return ((c->strip_cells + kTcTX - 1) / kTcTX) * ((c->nstrip + kTcTY - 1) / kTcTY);
}

}  // namespace hcg
