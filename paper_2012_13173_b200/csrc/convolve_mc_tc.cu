// convolve_mc_tc.cu -- step a6 for spectral cubes on the 5th-generation tensor cores (tcgen05 + TMEM):
// Eq. 1 applied per channel with one kernel weight and one weight map for all channels
// (the paper lists multi-channel gridding as "underway"; reading c7 of DESIGN.md), the
// contributing samples found by the search of PAPER.md:134-140 (Sect. 3.4 i-v).  SURVEY.md 8f NEXT-1.
//
// For a tile of 128 target cells the weighted sums are a matrix product
//     S[cell][chan] = sum_k  A[cell][k] * B[k][chan],   A = q_k w(d(cell, k)),  B = spectrum of candidate k,
// over the K candidates that can reach the tile.  One CTA owns a tile of 16 x 8 cells (M = 128) and a
// block of up to 256 channels (N); its warps are specialised:
//   * stream warp: builds the candidate stream of the tile (ring table, lookup-bin windows: steps i-iii,
//     as in convolve_tile.cu) and keeps the candidates whose distance to the tile's rectangle of cell
//     centres is within R: compaction in stream order into a FIFO of 32-candidate groups (= pipeline
//     stages).  A candidate's fixed-point offset from the tile centre is stored as two floats each
//     (multiple of 4096 + remainder, both exact), so the cell - candidate differences are formed with
//     three fp32 additions and carry the same single rounding as the tile kernel's integer difference;
//   * 8 compute warps evaluate A: thread = cell (= MMA row = TMEM lane), all 16 candidates of its two
//     K-steps of a stage, two candidates per instruction (packed fma.rn.f32x2 / add / mul), with the
//     tile kernel's scaled pair arithmetic; every weight is split w = hi + lo (hi = w rounded to TF32)
//     and stored straight into TENSOR MEMORY (tcgen05.st), from where the MMA reads its A operand -- no
//     shared-memory round trip and no proxy fence on this path;
//   * 4 spectrum-row warps copy the candidates' spectrum rows IN PLACE from `values` (never moved: a5)
//     with cp.async into the UMMA MN-major SWIZZLE_128B_BASE32B layout, a stage ahead, and write
//     v_lo = v - trunc_tf32(v) in bf16 into half-size MN-major SWIZZLE_128B tiles beside them (the tensor
//     core itself ignores the low 13 bits of v);
//   * MMA warp: one thread issues, per 8 candidates, two tcgen05.mma.kind::tf32 (w_hi * v, w_lo * v) and,
//     per 16 candidates, one kind::f16 on bf16 operands (w * v_lo: a 2^-11 term, for which 2^-9 of itself
//     is accuracy enough) into a 128 x 256 fp32 accumulator in TMEM: product error <= ~3e-6 relative.
// The tensor core adds with round-toward-zero (measured: -3.4e-8 relative per update), so the TMEM
// accumulator only ever holds a CHUNK of 8 stages (80 updates, bias <= 2.7e-6): the compute warps add every
// finished chunk into fp32 registers (round-to-nearest, 128 channels x 1 cell per thread), which also makes
// the epilogue a plain scale and store.  (4 stages per chunk: 1.6e-6 and 10 % slower; 10 and more: no faster.)
// W and the counts are summed on the CUDA cores from the same
// weights.  No atomics in the sums; the order of the additions is fixed by the stream order, so results
// are bit-wise reproducible.
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
constexpr int kTcCW = 8;                       // compute warps (warps 0 .. 7)
constexpr int kTcCT = kTcCW * 32;              // compute threads
constexpr int kTcBW = 4;                       // spectrum-row warps (warps 8 .. 11)
constexpr int kTcSW = 3;                       // stream-builder warps
constexpr int kTcThreads = kTcCT + 32 * kTcBW + 128;   // + the service warpgroup: MMA issuer, three stream builders
constexpr int kTcKS = 4;                       // K-steps (of 8 candidates) per pipeline stage
constexpr int kTcSC = 8 * kTcKS;               // candidates per stage = per FIFO group
constexpr int kTcNS = 3;                       // pipeline stages (B in shared memory, A in tensor memory)
constexpr int kTcBD = 1;                       // stages the spectrum rows are requested ahead of their split
constexpr int kTcCH = 8;                       // stages per TMEM accumulator chunk (10 MMA updates per stage)
constexpr int kTcGroups = 16;                  // FIFO groups
constexpr int kTcFifo = kTcGroups * kTcSC;     // FIFO entries
constexpr int kTcRings = 128;                  // ring-table entries per pass
constexpr int kBrawBytes = kTcKS * 8192;       // spectrum rows of a stage: kTcKS K-steps x 8 rows x 1 KB
// ... and their low parts v - trunc_tf32(v) in bf16, one 8 KB tile (16 rows x 256 channels) per pair of K-steps
constexpr int kBloBytes = (kTcKS / 2) * 8192;
constexpr int kOffBraw = 0, kOffBlo = kBrawBytes, kStageBytes = kBrawBytes + kBloBytes;
constexpr int kTmemA = 256;                    // TMEM columns: accumulator 0 .. 255, A ring from 256
constexpr int kTmemAStage = 16 * kTcKS + 8 * (kTcKS / 2);   // per stage: hi kTcKS x 8 columns, lo kTcKS x 8, then the weights in bf16: kTcKS / 2 x 8
static_assert(kTmemA + kTcNS * kTmemAStage <= 512, "TMEM columns");
// FIFO: per pair of candidates three float4: (Xh_a, Xh_b, Xl_a, Xl_b), (Yh_a, Yh_b, Yl_a, Yl_b), (cs_a, cs_b, q_a, q_b)
constexpr int kOffFifoX = kTcNS * kStageBytes;
constexpr int kOffFifoY = kOffFifoX + kTcFifo * 8;
constexpr int kOffFifoC = kOffFifoY + kTcFifo * 8;
constexpr int kOffFifoI = kOffFifoC + kTcFifo * 8;         // uint32 [kTcFifo]: sample index
constexpr int kOffTabBase = kOffFifoI + kTcFifo * 4;       // u64 [kTcRings]
constexpr int kOffTabEnd = kOffTabBase + kTcRings * 8;     // int [kTcRings]
constexpr int kOffGrpN = kOffTabEnd + kTcRings * 4;        // uint32 [kTcGroups]: candidates in the group | 0x80 (last group of the tile)
constexpr int kOffBars = kOffGrpN + kTcGroups * 4;         // u64: afull[NS], bfull[NS], empty[NS], dfull, dempty, cfull[G], cempty[G]
constexpr int kOffMisc = kOffBars + 8 * (3 * kTcNS + 2 + 2 * kTcGroups);
constexpr int kTcSmem = kOffMisc + 64 + 8 + 4 * kTcGroups;   // flags, tmem address, token, group counters
static_assert(kTcSmem <= 227 * 1024, "shared memory");

// ---- PTX wrappers
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// Bounded: a wait that outlasts any legitimate one (seconds) is a broken pipeline -- fail loudly, do not hang.
// (No suspend-time hint: with one, a wait on an already completed phase took ~700 cycles instead of ~100.)
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    for (uint32_t spins = 0;; ++spins) {
        uint32_t ok;
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (ok) return;
        if (spins > (1u << 24)) __trap();
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
__device__ __forceinline__ void tmem_ld16(uint32_t addr, uint32_t (&v)[16]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 "
                 "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                   "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
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

__device__ __forceinline__ void umma_tf32_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void tmem_st1(uint32_t addr, float v) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ void tmem_st16_zero(uint32_t addr) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1};"
                 ::"r"(addr), "r"(0u) : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

__device__ __forceinline__ unsigned long long f2_pack(float lo, float hi) {
    unsigned long long d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi));
    return d;
}
__device__ __forceinline__ void f2_unpack(unsigned long long v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ unsigned long long f2_add(unsigned long long a, unsigned long long b) {
    unsigned long long d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ unsigned long long f2_mul(unsigned long long a, unsigned long long b) {
    unsigned long long d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ unsigned long long f2_fma(unsigned long long a, unsigned long long b, unsigned long long c) {
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}

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

// the same for kind::f16 on bf16 operands (A K-major from tensor memory, B MN-major)
__device__ __forceinline__ uint32_t umma_idesc_bf16(int n) {
    return (1u << 4) | (1u << 7) | (1u << 10) | (0u << 15) | (1u << 16) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
}
__device__ __forceinline__ void umma_bf16_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(acc) : "memory");
}
// two floats rounded to bf16 and packed: `lo` in the low half
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
    uint32_t d;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
    return d;
}
__device__ __forceinline__ void sts_u2(uint32_t addr, uint32_t a, uint32_t b) {
    asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(addr), "r"(a), "r"(b) : "memory");
}

template <int MODE, bool COUNTS>
__global__ void __launch_bounds__(kTcThreads, 1)
conv_mc_tc_f32(const McTcArgs m) {
    const TileArgs& a = m.t;
    extern __shared__ __align__(1024) unsigned char s_tc[];
    const uint32_t s_base = smem_addr(s_tc);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t b_afull = s_base + kOffBars, b_bfull = b_afull + 8 * kTcNS, b_empty = b_bfull + 8 * kTcNS;
    const uint32_t b_dfull = b_empty + 8 * kTcNS, b_dempty = b_dfull + 8;
    const uint32_t b_cfull = b_dempty + 8, b_cempty = b_cfull + 8 * kTcGroups;
    volatile uint32_t* s_flag = (volatile uint32_t*)(s_tc + kOffMisc);   // [NS] stage flags
    uint32_t* s_tmem = (uint32_t*)(s_tc + kOffMisc + 4 * kTcNS);
    int* s_bad = (int*)(s_tmem + 1);
    volatile int* s_tok = (volatile int*)(s_tc + kOffMisc + 64);    // [0] next stream block to append, [1] FIFO position
    int* s_gcnt = (int*)(s_tc + kOffMisc + 72);                     // [G] candidates written into each FIFO group

    const int tile = blockIdx.x;
    const int ch0 = blockIdx.y * 256;
    const int nch = min(256, m.nchan - ch0);                        // channels of this block (multiple of 32)
    const int ty = tile / a.tiles_x;
    const int ix0 = (tile - ty * a.tiles_x) * kTcTX;
    const int row0 = ty * kTcTY;
    const int ncols = min(kTcTX, a.nx - ix0);
    const int nrows = min(kTcTY, a.ny - row0);
    constexpr int kMmaWarp = kTcCW + kTcBW, kStreamWarp = kMmaWarp + 1;
    // everything is measured from a cell in the middle of the tile (the fixed-point differences are good for +- 8
    // columns / rows plus the support radius: target.cu)
    const int ic = ncols >> 1, jc = nrows >> 1;
    const uint32_t xc0 = (uint32_t)(unsigned long long)__double2ll_rn((a.u0 + (double)(ix0 + ic) * a.du) * a.sx);
    const uint32_t yc0 = (uint32_t)__ldg((const int*)(a.rows + row0 + jc));

    if (warp == kMmaWarp) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_addr(s_tmem)), "r"(512u));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::);
        if (lane == 0) {
            for (int s = 0; s < kTcNS; ++s) {
                mbar_init(b_afull + 8 * s, kTcCW); mbar_init(b_bfull + 8 * s, kTcBW); mbar_init(b_empty + 8 * s, 1);
            }
            mbar_init(b_dfull, 1); mbar_init(b_dempty, kTcCW);
            for (int j = 0; j < kTcGroups; ++j) { mbar_init(b_cfull + 8 * j, 1); mbar_init(b_cempty + 8 * j, kTcCW + kTcBW); }
            *s_bad = 0;
            s_tok[0] = 0; s_tok[1] = 0;
            for (int j = 0; j < kTcGroups; ++j) s_gcnt[j] = 0;
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tm = *s_tmem;

    if (warp >= kMmaWarp) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");       // the whole service warpgroup, one instruction
        if (warp == kMmaWarp) {
            // ============================================================ MMA issuer (lane 0 issues; the warp stays converged)
            const uint32_t idesc = umma_idesc_tf32(nch);
            const uint32_t idesc16 = umma_idesc_bf16(nch);
            // spectrum rows: 32-bit MN-major, SWIZZLE_128B_BASE32B; their low parts: bf16 MN-major, SWIZZLE_128B (64-channel
            // segments 2048 bytes apart, the two 8-row groups of a 16-row tile 1024 bytes apart)
            const uint64_t b_rw0 = umma_desc(s_base + kOffBraw, 1024, 512, 1), b_lo0 = umma_desc(s_base + kOffBlo, 2048, 1024, 2);
            for (int s = 0;; ++s) {
                const int slot = s % kTcNS;
                const uint32_t par = (uint32_t)(s / kTcNS) & 1u;
                mbar_wait(b_afull + 8 * slot, par);
                const uint32_t flag = s_flag[slot];
                if (!(flag & 2u)) {
                    mbar_wait(b_bfull + 8 * slot, par);
                    const int chunk = s / kTcCH;
                    const bool first = s % kTcCH == 0;
                    if (first && chunk >= 1) mbar_wait(b_dempty, (uint32_t)(chunk - 1) & 1u);   // the previous chunk has been taken over
                    tc_fence_after();
                    if (lane == 0) {
                        const uint64_t so = (uint64_t)((uint32_t)slot * (kStageBytes >> 4));
#pragma unroll
                        for (int ks = 0; ks < kTcKS; ++ks) {               // w_hi * v + w_lo * v, TF32 (the unit truncates v)
                            const uint32_t ah = tm + kTmemA + (uint32_t)(slot * kTmemAStage + ks * 8), al = ah + 8 * kTcKS;
                            const uint64_t br = b_rw0 + so + (uint64_t)(ks * (8192 >> 4));
                            umma_tf32_ts(tm, ah, br, idesc, (first && ks == 0) ? 0u : 1u);
                            umma_tf32_ts(tm, al, br, idesc, 1u);
                        }
#pragma unroll
                        for (int j = 0; j < kTcKS / 2; ++j) {              // + w * v_lo: a 2^-11 term, bf16 x bf16 over 16 candidates
                            const uint32_t ab = tm + kTmemA + (uint32_t)(slot * kTmemAStage + 16 * kTcKS + j * 8);
                            umma_bf16_ts(tm, ab, b_lo0 + so + (uint64_t)(j * (8192 >> 4)), idesc16, 1u);
                        }
                        tc_commit(b_empty + 8 * slot);
                        if (s % kTcCH == kTcCH - 1 || (flag & 1u)) tc_commit(b_dfull);
                    }
                    __syncwarp();
                } else if (s % kTcCH != 0) {                          // end-of-tile mark without a stage: close the open chunk
                    if (lane == 0) tc_commit(b_dfull);
                    __syncwarp();
                }
                if (flag & 1u) {
                    break;
                }
            }
        } else {
            // ============================================================ stream builders: steps (i)-(iii) + compaction
            // Three warps share the stream: warp sw tests blocks sw, sw + 3, ... of 32 records; a token handed on in
            // block order gives every block its place in the FIFO, so the kept candidates stay in stream order.
            const int sw = warp - kStreamWarp;
            float cc0 = 0.f, p1 = 0.f, p2 = 0.f, p3 = 0.f, ccmin = 2.0f;
            float xlo, xhi, ylo, yhi;                                // extent of the tile's cell centres (scaled units)
            int rmin = 0x7fffffff, rmax = -0x7fffffff;
            const float sxk = a.sxk, syk = a.syk, a12 = a.a12;
            {
                for (int j = 0; j < nrows; ++j) {
                    const int4 r0 = __ldg((const int4*)(a.rows + row0 + j));
                    ccmin = fminf(ccmin, __int_as_float(r0.w));
                    rmin = min(rmin, r0.y);
                    rmax = max(rmax, r0.y + r0.z - 1);
                    if (j == jc) {
                        const int4 r1 = __ldg((const int4*)(a.rows + row0 + j) + 1);
                        cc0 = __int_as_float(r0.w);
                        const float sc0 = __int_as_float(r1.x), ik = a.isk;
                        p1 = -sc0 * ik;
                        p2 = -0.5f * cc0 * ik * ik;
                        p3 = sc0 * ik * ik * ik * (1.0f / 6.0f);
                    }
                }
                const float pad = 1e-3f * sqrtf(a.hmax);             // slack for the fp32 rounding of the extents
                const float xa = (float)(-ic) * a.duk, xb = (float)(ncols - 1 - ic) * a.duk;
                const float ya = (float)(-jc) * a.dyk, yb = (float)(nrows - 1 - jc) * a.dyk;
                xlo = fminf(xa, xb) - pad; xhi = fmaxf(xa, xb) + pad;
                ylo = fminf(ya, yb) - pad; yhi = fmaxf(ya, yb) + pad;
                ccmin *= 0.999f;
            }
            const float fxw = (float)(a.du >= 0.0 ? ix0 : ix0 + ncols - 1);
            const float fxe = (float)(a.du >= 0.0 ? ix0 + ncols - 1 : ix0);
            const bool flip = (ty & 1) != 0;                          // odd tile rows walk the rings south to north
            const Rec32* __restrict__ rec = a.rec;
            unsigned long long* tab_base = (unsigned long long*)(s_tc + kOffTabBase);
            volatile int* tab_end = (volatile int*)(s_tc + kOffTabEnd);
            float* fifo_x = (float*)(s_tc + kOffFifoX);
            float* fifo_y = (float*)(s_tc + kOffFifoY);
            float* fifo_c = (float*)(s_tc + kOffFifoC);
            uint32_t* fifo_i = (uint32_t*)(s_tc + kOffFifoI);
            volatile uint32_t* grp_n = (volatile uint32_t*)(s_tc + kOffGrpN);
            const float hlim = a.hmax * 1.0001f;
            auto bar_stream = [&]() { asm volatile("bar.sync 2, %0;" ::"n"(32 * kTcSW) : "memory"); };
            // entry p of the FIFO: pair p >> 1, member p & 1; high part = multiple of 4096 units, low part = the rest
            auto put = [&](int pos, int dxi, int dyi, float cs, float q, uint32_t sidx) {
                const int p = pos & (kTcFifo - 1), o = 4 * (p >> 1) + (p & 1);
                fifo_x[o] = (float)(dxi & ~0xfff); fifo_x[o + 2] = (float)(dxi & 0xfff);
                fifo_y[o] = (float)(dyi & ~0xfff); fifo_y[o + 2] = (float)(dyi & 0xfff);
                fifo_c[o] = cs; fifo_c[o + 2] = q;
                fifo_i[p] = sidx;
            };
            // record number i of this pass's stream; `cur` is this lane's ring cursor (i only grows within a pass)
            auto fetch = [&](int i, int total, int& cur) -> uint4 {
                if (i >= total) return make_uint4(0, 0, 0, 0);
                while (tab_end[cur] <= i) ++cur;
                return ldg_rec(tab_base[cur], i);
            };
            // `cnt` candidates have been written into FIFO group gi: the writer of the last ones publishes the group
            auto group_done = [&](int gi, int cnt) {
                __threadfence_block();
                const int slot = gi % kTcGroups;
                if (atomicAdd(s_gcnt + slot, cnt) + cnt == kTcSC) {
                    s_gcnt[slot] = 0;
                    __threadfence_block();
                    grp_n[slot] = (uint32_t)kTcSC;
                    mbar_arrive(b_cfull + 8 * slot);
                }
            };

            int blk0 = 0;                                             // blocks of the passes before this one
            for (int pass = 0; rmin + pass * kTcRings <= rmax; ++pass) {
                // ---- ring table of this pass (warp 0): lane l of sub-pass t <-> ring number 32 t + l
                if (sw == 0) {
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
                }
                bar_stream();
                const int total = tab_end[kTcRings - 1];
                const int nb = (total + 31) >> 5;
                // ---- this warp's blocks of the pass, the records of its next three blocks in flight
                int cur = 0;
                uint4 n0 = fetch(32 * sw + lane, total, cur), n1 = fetch(32 * (sw + kTcSW) + lane, total, cur),
                      n2 = fetch(32 * (sw + 2 * kTcSW) + lane, total, cur);
                for (int b = sw; b < nb; b += kTcSW) {
                    const uint4 raw = n0;
                    n0 = n1; n1 = n2;
                    n2 = fetch(32 * (b + 3 * kTcSW) + lane, total, cur);
                    bool keep = false;
                    float cs = 0.f;
                    const int dxi = (int)(raw.x - xc0), dyi = (int)(raw.y - yc0);
                    if (32 * b + lane < total) {
                        const float X = (float)dxi * sxk, Y = (float)dyi * syk;
                        cs = fmaf(Y, fmaf(Y, fmaf(Y, p3, p2), p1), cc0);
                        const float ex = fmaxf(fmaxf(xlo - X, X - xhi), 0.0f), ey = fmaxf(fmaxf(ylo - Y, Y - yhi), 0.0f);
                        float v = ex * ex, u = ey * ey;
                        if (MODE >= 1) { v = v * fmaf(v, -a12, 1.0f); u = u * fmaf(u, -a12, 1.0f); }
                        keep = fmaf(ccmin * cs, v, u) <= hlim;
                    }
                    const unsigned mk = __ballot_sync(0xffffffffu, keep);
                    const int nk = __popc(mk);
                    // the token: FIFO position of this block's first candidate, in block order
                    int gpos = 0;
                    if (lane == 0) {
                        while (s_tok[0] != blk0 + b) { }
                        __threadfence_block();
                        gpos = s_tok[1];
                        s_tok[1] = gpos + nk;
                        __threadfence_block();
                        s_tok[0] = blk0 + b + 1;
                    }
                    gpos = __shfl_sync(0xffffffffu, gpos, 0);
                    if (nk == 0) continue;
                    // the groups this block writes into must have been released by the readers of their previous contents
                    // (a group's first writer may be another warp that is still waiting for just that)
                    for (int gi = gpos / kTcSC; gi <= (gpos + nk - 1) / kTcSC; ++gi)
                        if (gi >= kTcGroups) mbar_wait(b_cempty + 8 * (gi % kTcGroups), (uint32_t)(gi / kTcGroups - 1) & 1u);
                    if (keep) put(gpos + __popc(mk & ((1u << lane) - 1u)), dxi, dyi, cs, __uint_as_float(raw.w), raw.z);
                    __syncwarp();
                    if (lane == 0) {
                        const int ga = gpos / kTcSC, gb = (gpos + nk - 1) / kTcSC;   // nk <= 32: at most two groups
                        if (ga == gb) group_done(ga, nk);
                        else { group_done(ga, kTcSC * gb - gpos); group_done(gb, gpos + nk - kTcSC * gb); }
                    }
                }
                bar_stream();                                         // every block of the pass has been appended
                blk0 += nb;
            }
            // ---- the end-of-tile mark: the last, partial group (its unused slots filled with candidates far outside every
            // cell's reach: weight 0, never counted), or an empty group when the stream ended on a group boundary
            if (sw == 0) {
                const int gpos = s_tok[1];
                const int gi = gpos / kTcSC, nlast = gpos - kTcSC * gi;
                if (nlast == 0 && gi >= kTcGroups) mbar_wait(b_cempty + 8 * (gi % kTcGroups), (uint32_t)(gi / kTcGroups - 1) & 1u);
                const int far = __float2int_rn((8.0f * fabsf(a.dyk) + 10.0f * sqrtf(a.hmax)) / syk);
                if (nlast > 0 && lane >= nlast) put(kTcSC * gi + lane, 0, far, 1.0f, 0.0f, 0u);
                __syncwarp();
                if (lane == 0) {
                    s_gcnt[gi % kTcGroups] = 0;
                    __threadfence_block();
                    grp_n[gi % kTcGroups] = (uint32_t)nlast | 0x80u;
                    mbar_arrive(b_cfull + 8 * (gi % kTcGroups));
                }
            }
        }
    } else if (warp >= kTcCW) {
        // ================================================================ spectrum rows (B): 128 threads
        asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        // (Measured and not kept: TMA tile::gather4 requests of 4 rows x 128 bytes land in exactly this layout with
        // CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B, but the copy engine takes ~47 cycles per request per SM -- 3 x slower
        // than the 16-byte cp.async below.)
        // thread t4: 16-byte unit u = t4 & 63 of the rows r = 2 i + (t4 >> 6), i = 0 .. kTcSC / 2 - 1, of every stage
        const int t4 = tid - kTcCT;
        const int u = t4 & 63, rp = t4 >> 6;
        const int upr = nch >> 2;                                     // 16-byte units per row (<= 64)
        const bool on = u < upr;
        // offset of unit u in a K-step's B region for a row r: by r & 3 (row in the 4-row atom), plus ((r >> 2) & 1) * 512, (r >> 3) * 8192
        uint32_t off_u[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int k3 = 2 * h + rp;                                // r & 3 for r = 2 i + rp: i even -> rp, i odd -> 2 + rp
            off_u[h] = (uint32_t)((u >> 3) * 1024 + k3 * 128 + (((((u & 7) >> 1) ^ k3) << 5) | ((u & 1) << 4)));
        }
        const unsigned long long vsrc = (unsigned long long)(uintptr_t)(m.values + ch0 + 4 * (on ? u : 0));
        const uint32_t vstride = (uint32_t)m.nchan * 4u;              // bytes per row
        const uint32_t fifo_i_s = s_base + kOffFifoI, grp_n_s = s_base + kOffGrpN;
        // row r = 2 i + rp of the stage: (r >> 3) = i >> 2, (r >> 2) & 1 = (i >> 1) & 1, r & 3 = 2 (i & 1) + rp
        auto unit_off = [&](int i) -> uint32_t { return (uint32_t)((i >> 2) * 8192 + ((i >> 1) & 1) * 512) + off_u[i & 1]; };
        // the 8 bytes (4 channels in bf16) of the same unit in the low-part tiles: row r = 2 i + rp is row k = r & 15 of tile
        // r >> 4; channels 4 u ..: segment u >> 4 (2048 bytes), 8-row group k >> 3 (1024), row k & 7 (128), 16-byte chunk
        // ((u & 15) >> 1) ^ (k & 7), half u & 1
        uint32_t off_l[4];                                            // by i & 3 (= the row's k & 7 given rp)
#pragma unroll
        for (int v = 0; v < 4; ++v) {
            const int k7 = 2 * v + rp;
            off_l[v] = (uint32_t)((u >> 4) * 2048 + k7 * 128 + ((((u & 15) >> 1) ^ k7) << 4) + (u & 1) * 8);
        }
        auto lo_off = [&](int i) -> uint32_t { return (uint32_t)((i >> 3) * 8192 + ((i >> 2) & 1) * 1024) + off_l[i & 3]; };
        constexpr int NU = kTcSC / 2;                                 // units per thread per stage
        int nst = 0x7fffffff, pf = 0;
        for (int k = 0;; ++k) {
            // request the rows of the stages up to k + BD (the missing rows of the last stage are zeros)
            while (pf <= k + kTcBD) {
                if (pf < nst) {
                    const int grp = pf % kTcGroups, slot = pf % kTcNS;
                    mbar_wait(b_cfull + 8 * grp, (uint32_t)(pf / kTcGroups) & 1u);
                    const uint32_t info = lds_u1(grp_n_s + 4u * (uint32_t)grp);
                    const int n = (int)(info & 0x7fu);
                    if (info & 0x80u) nst = n > 0 ? pf + 1 : pf;
                    if (pf < nst) {
                        if (pf >= kTcNS) mbar_wait(b_empty + 8 * slot, (uint32_t)(pf / kTcNS - 1) & 1u);
                        const uint32_t sb = s_base + (uint32_t)slot * kStageBytes + kOffBraw;
                        if (on) {
#pragma unroll
                            for (int i0 = 0; i0 < NU; i0 += 8) {
                                uint32_t idx[8];
#pragma unroll
                                for (int i = 0; i < 8; ++i) idx[i] = lds_u1(fifo_i_s + (uint32_t)(grp * kTcSC + 2 * (i0 + i) + rp) * 4u);
#pragma unroll
                                for (int i = 0; i < 8; ++i) {
                                    const uint32_t dst = sb + unit_off(i0 + i);
                                    if (2 * (i0 + i) + rp < n) cp_async16_cg(dst, (const void*)(uintptr_t)(vsrc + (unsigned long long)idx[i] * vstride));
                                    else sts_u4(dst, make_uint4(0, 0, 0, 0));
                                }
                            }
                        }
                        __syncwarp();
                        if (lane == 0) mbar_arrive(b_cempty + 8 * grp);   // done with the group's sample indices
                    }
                }
                cp_commit();
                ++pf;
            }
            if (k >= nst) break;
            // the rows of stage k have landed (each thread reads back its own bytes): lo = v - trunc_tf32(v)
            cp_wait<kTcBD>();
            const int slot = k % kTcNS;
            const uint32_t sb = s_base + (uint32_t)slot * kStageBytes + kOffBraw;
            if (on) {
                // two register buffers of 4 units take turns: the loads of one batch are in flight while the other is
                // split and stored (the shared-memory wrappers are ordered among themselves, so the overlap has to be
                // spelled out)
                auto load4 = [&](uint4 (&v)[4], int i0) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) v[j] = lds_u4(sb + unit_off(i0 + j));
                };
                auto split4 = [&](uint4 (&v)[4], int i0) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const float lx = __uint_as_float(v[j].x) - __uint_as_float(v[j].x & 0xffffe000u);
                        const float ly = __uint_as_float(v[j].y) - __uint_as_float(v[j].y & 0xffffe000u);
                        const float lz = __uint_as_float(v[j].z) - __uint_as_float(v[j].z & 0xffffe000u);
                        const float lw = __uint_as_float(v[j].w) - __uint_as_float(v[j].w & 0xffffe000u);
                        sts_u2(sb + (kOffBlo - kOffBraw) + lo_off(i0 + j), pack_bf16(lx, ly), pack_bf16(lz, lw));
                    }
                };
                uint4 va[4], vb[4];
                load4(va, 0);
#pragma unroll
                for (int i0 = 0; i0 < NU; i0 += 8) {
                    load4(vb, i0 + 4);
                    split4(va, i0);
                    if (i0 + 8 < NU) load4(va, i0 + 8);
                    split4(vb, i0 + 4);
                }
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncwarp();
            if (lane == 0) mbar_arrive(b_bfull + 8 * slot);
        }
        cp_wait<0>();
    } else {
        // ================================================================ A (kernel weights) and the accumulators
        asm volatile("setmaxnreg.inc.sync.aligned.u32 200;");
        // MMA row (= TMEM lane) 32 q + l  <->  cell (8 (q & 1) + (l & 7), 4 (q >> 1) + (l >> 3)); g selects the half
        // of a stage's K-steps (A) and the channel half (drain).
        const int q = warp & 3, g = warp >> 2;
        const int cell = q * 32 + lane;
        const int cix = 8 * (q & 1) + (lane & 7), ciy = 4 * (q >> 1) + (lane >> 3);
        const bool cell_ok = cix < ncols && ciy < nrows;
        // this cell's offset from the tile centre in fixed-point units, split like the candidates' (negated: the
        // differences are formed by additions)
        unsigned long long ncxh, ncxl, ncyh, ncyl, cc2;
        {
            const int4 r0 = __ldg((const int4*)(a.rows + min(row0 + ciy, a.ny - 1)));
            const uint32_t xc = (uint32_t)(unsigned long long)__double2ll_rn((a.u0 + (double)(ix0 + min(cix, ncols - 1)) * a.du) * a.sx);
            const int cxi = (int)(xc - xc0), cyi = (int)((uint32_t)r0.x - yc0);
            const float xh = -(float)(cxi & ~0xfff), xl = -(float)(cxi & 0xfff), yh = -(float)(cyi & ~0xfff), yl = -(float)(cyi & 0xfff);
            const float cc = __int_as_float(r0.w);
            ncxh = f2_pack(xh, xh); ncxl = f2_pack(xl, xl); ncyh = f2_pack(yh, yh); ncyl = f2_pack(yl, yl); cc2 = f2_pack(cc, cc);
        }
        float hm = cell_ok ? a.hmax : -1.0f;
        asm volatile("" : "+l"(ncxh), "+l"(ncxl), "+l"(ncyh), "+l"(ncyl), "+l"(cc2), "+f"(hm));
        const unsigned long long sxk2 = f2_pack(a.sxk, a.sxk), syk2 = f2_pack(a.syk, a.syk);
        const unsigned long long na12 = f2_pack(-a.a12, -a.a12), pa12 = f2_pack(a.a12, a.a12), one2 = f2_pack(1.0f, 1.0f);
        const uint32_t fifo_x_s = s_base + kOffFifoX, fifo_y_s = s_base + kOffFifoY, fifo_c_s = s_base + kOffFifoC;
        const uint32_t grp_n_s = s_base + kOffGrpN;
        const uint32_t t_lane = tm + ((uint32_t)(q * 32) << 16);     // this warp's TMEM lanes

        float acc[128];
#pragma unroll
        for (int j = 0; j < 128; ++j) acc[j] = 0.0f;
        unsigned long long wsum2 = 0ull;
        int csum = 0;

        // take a finished chunk over from the TMEM accumulator: channels 128 g .. 128 g + 127 of this thread's cell
        auto drain = [&](int j) {
            mbar_wait(b_dfull, (uint32_t)j & 1u);
            tc_fence_after();
#pragma unroll
            for (int h = 0; h < 8; ++h) {
                uint32_t v[16];
                tmem_ld16(t_lane + (uint32_t)(g * 128 + 16 * h), v);
                tmem_ld_wait();
#pragma unroll
                for (int c = 0; c < 16; ++c) acc[16 * h + c] += __uint_as_float(v[c]);
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(b_dempty);
        };

        int k = 0, jd = 0, nst = 0x7fffffff;
        bool term = false;
        for (;;) {
            if (k >= nst) break;                                     // the last group has been seen
            // the chunk the MMA warp has finished must be taken over before it can start the next: as soon as it is
            // complete, and at the latest when this warp would have to wait for a stage of the following chunk
            if (jd < k / kTcCH && (k == (jd + 1) * kTcCH + kTcNS - 1 || mbar_test(b_dfull, (uint32_t)jd & 1u))) { drain(jd); ++jd; 
            }
            mbar_wait(b_cfull + 8 * (k % kTcGroups), (uint32_t)(k / kTcGroups) & 1u);
            const uint32_t info = lds_u1(grp_n_s + 4u * (uint32_t)(k % kTcGroups));
            if (info & 0x80u) nst = (info & 0x7fu) > 0 ? k + 1 : k;
            if (k >= nst) { term = true; break; }                   // an empty last group: the stream ended on a group boundary
            const int slot = k % kTcNS;
            if (k >= kTcNS) {
                mbar_wait(b_empty + 8 * slot, (uint32_t)(k / kTcNS - 1) & 1u);
                tc_fence_after();
            }

            // ---- A: K-steps g * kTcKS / 2 .. of the stage x this thread's cell, two candidates per instruction
#pragma unroll
            for (int kk = 0; kk < kTcKS / 2; ++kk) {
                const int ks = g * (kTcKS / 2) + kk;
                const uint32_t pr0 = (uint32_t)((k % kTcGroups) * (kTcSC / 2) + ks * 4);   // first candidate pair of the K-step
                uint32_t hi[8], lo[8];
#pragma unroll
                for (int pp = 0; pp < 4; ++pp) {
                    const uint4 ex = lds_u4(fifo_x_s + (pr0 + pp) * 16u), ey = lds_u4(fifo_y_s + (pr0 + pp) * 16u);
                    const uint4 ec = lds_u4(fifo_c_s + (pr0 + pp) * 16u);
                    const unsigned long long xh = ((unsigned long long)ex.y << 32) | ex.x, xl = ((unsigned long long)ex.w << 32) | ex.z;
                    const unsigned long long yh = ((unsigned long long)ey.y << 32) | ey.x, yl = ((unsigned long long)ey.w << 32) | ey.z;
                    const unsigned long long cs = ((unsigned long long)ec.y << 32) | ec.x, qq = ((unsigned long long)ec.w << 32) | ec.z;
                    // exact differences of the split fixed-point offsets, one rounding in the last addition
                    const unsigned long long dx = f2_mul(f2_add(f2_add(xh, ncxh), f2_add(xl, ncxl)), sxk2);
                    const unsigned long long dy = f2_mul(f2_add(f2_add(yh, ncyh), f2_add(yl, ncyl)), syk2);
                    unsigned long long v = f2_mul(dx, dx), u = f2_mul(dy, dy);
                    if (MODE >= 1) { v = f2_mul(v, f2_fma(v, na12, one2)); u = f2_mul(u, f2_fma(u, na12, one2)); }
                    const unsigned long long h2 = f2_fma(f2_mul(cc2, cs), v, u);
                    const unsigned long long e2 = MODE == 2 ? f2_mul(h2, f2_fma(h2, pa12, one2)) : h2;
                    float ha, hb, ea, eb;
                    f2_unpack(h2, ha, hb);
                    f2_unpack(e2, ea, eb);
                    const unsigned long long w2 = f2_mul(f2_pack(ex2_approx(-ea), ex2_approx(-eb)), qq);
                    float wa, wb;
                    f2_unpack(w2, wa, wb);
                    const bool hita = ha <= hm, hitb = hb <= hm;
                    wa = hita ? wa : 0.0f;
                    wb = hitb ? wb : 0.0f;
                    if (COUNTS) csum += (hita ? 1 : 0) + (hitb ? 1 : 0);
                    const unsigned long long ws2 = f2_pack(wa, wb);
                    wsum2 = f2_add(wsum2, ws2);
                    hi[2 * pp] = (__float_as_uint(wa) + 0x1000u) & 0xffffe000u;
                    hi[2 * pp + 1] = (__float_as_uint(wb) + 0x1000u) & 0xffffe000u;
                    lo[2 * pp] = __float_as_uint(wa - __uint_as_float(hi[2 * pp]));
                    lo[2 * pp + 1] = __float_as_uint(wb - __uint_as_float(hi[2 * pp + 1]));
                }
                const uint32_t t_hi = t_lane + kTmemA + (uint32_t)(slot * kTmemAStage + ks * 8), t_lo = t_hi + 8 * kTcKS;
                // the same eight weights in bf16 for the low-part product: candidates 8 kk .. 8 kk + 7 of this thread's
                // 16-candidate tile g = columns 4 kk .. 4 kk + 3 (column c: candidate 2 c in the low half, 2 c + 1 in the high)
                const uint32_t t_bf = t_lane + kTmemA + (uint32_t)(slot * kTmemAStage + 16 * kTcKS + g * 8 + kk * 4);
                asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};"
                             ::"r"(t_bf), "r"(pack_bf16(__uint_as_float(hi[0]), __uint_as_float(hi[1]))),
                               "r"(pack_bf16(__uint_as_float(hi[2]), __uint_as_float(hi[3]))),
                               "r"(pack_bf16(__uint_as_float(hi[4]), __uint_as_float(hi[5]))),
                               "r"(pack_bf16(__uint_as_float(hi[6]), __uint_as_float(hi[7]))) : "memory");
                asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};"
                             ::"r"(t_hi), "r"(hi[0]), "r"(hi[1]), "r"(hi[2]), "r"(hi[3]), "r"(hi[4]), "r"(hi[5]), "r"(hi[6]), "r"(hi[7]) : "memory");
                asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};"
                             ::"r"(t_lo), "r"(lo[0]), "r"(lo[1]), "r"(lo[2]), "r"(lo[3]), "r"(lo[4]), "r"(lo[5]), "r"(lo[6]), "r"(lo[7]) : "memory");
            }
            tmem_st_wait();
            tc_fence_before();
            if (tid == 0) s_flag[slot] = k == nst - 1 ? 1u : 0u;
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(b_cempty + 8 * (k % kTcGroups));          // this warp is done with the group's FIFO entries
                mbar_arrive(b_afull + 8 * slot);
            }
            ++k;
        }
        if (term) {                                                  // no stage carried the end-of-tile mark: send it on its own
            const int slot = nst % kTcNS;
            if (nst >= kTcNS) mbar_wait(b_empty + 8 * slot, (uint32_t)(nst / kTcNS - 1) & 1u);
            if (tid == 0) s_flag[slot] = 3u;
            __syncwarp();
            if (lane == 0) mbar_arrive(b_afull + 8 * slot);
        }
        for (const int nchunk = (nst + kTcCH - 1) / kTcCH; jd < nchunk; ++jd) drain(jd);

        // ---- finish: W and counts over the two K-step halves of a cell (fixed order), normalise, store
        float wsa, wsb;
        f2_unpack(wsum2, wsa, wsb);
        bar_compute();                                               // every warp is done with the FIFO: reuse it
        float* s_w = (float*)(s_tc + kOffFifoX);
        int* s_c = (int*)(s_w + 2 * 128);
        s_w[g * 128 + cell] = wsa + wsb;
        if (COUNTS) s_c[g * 128 + cell] = csum;
        // 0 * inf = NaN reaches every cell of the tile: non-finite sums flag the tile for the cell-by-cell pass
        float chk = 0.0f;
#pragma unroll
        for (int j = 0; j < 128; ++j) chk = fmaf(acc[j], 0.0f, chk);
        if (__any_sync(0xffffffffu, chk != 0.0f) && lane == 0) atomicOr(s_bad, 1);
        bar_compute();
        const float wtot = s_w[cell] + s_w[128 + cell];
        // what the sums are multiplied by: 1 / W (one division per cell; a product differs from the quotient by at most
        // 1.5 ulp), NaN for a cell no sample reaches, 1 for un-normalised sums
        const float scale = a.raw ? 1.0f : (wtot > 0.0f ? 1.0f / wtot : __int_as_float(0x7fc00000));
        if (cell_ok && g == 0 && blockIdx.y == 0) {
            const int64_t gc = (int64_t)(row0 + ciy) * a.nx + ix0 + cix;
            a.wmap[gc] = wtot;
            if (COUNTS) a.counts[gc] = s_c[cell] + s_c[128 + cell];
        }
        // The sums go out through shared memory (the stage buffers are idle by now: every MMA has completed and the row
        // warps have left): a thread holds 128 channels of ONE cell, so direct stores would touch 32 cells' rows per
        // instruction; transposed, a warp writes 512 contiguous bytes of one cell per instruction.
        constexpr uint32_t kPitch = 1024 + 16;                       // bytes per cell row (+ 16: conflict-free 16-byte columns)
        static_assert(128 * kPitch <= (uint32_t)kOffFifoX, "epilogue staging");
        {
            const uint32_t so = s_base + (uint32_t)cell * kPitch + (uint32_t)g * 512u;
#pragma unroll
            for (int j = 0; j < 128; j += 4)
                sts_u4(so + 4u * j, make_uint4(__float_as_uint(acc[j] * scale), __float_as_uint(acc[j + 1] * scale),
                                               __float_as_uint(acc[j + 2] * scale), __float_as_uint(acc[j + 3] * scale)));
        }
        bar_compute();
        {
            const int nu = nch >> 2;                                  // 16-byte units per cell (<= 64)
            for (int cl = warp; cl < 128; cl += kTcCW) {              // cell 32 q' + l' of the tile
                const int ex = 8 * ((cl >> 5) & 1) + (cl & 7), ey = 4 * (cl >> 6) + ((cl & 31) >> 3);
                if (ex >= ncols || ey >= nrows) continue;             // warp-uniform
                float* o = a.cube + ((size_t)(row0 + ey) * a.nx + ix0 + ex) * m.nchan + ch0;
                const uint32_t si = s_base + (uint32_t)cl * kPitch;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int u = lane + 32 * h;
                    if (u < nu) {
                        const uint4 v = lds_u4(si + 16u * u);
                        *(uint4*)(o + 4 * u) = v;
                    }
                }
            }
        }
        if (tid == 0 && m.dirty) m.dirty[(size_t)blockIdx.y * a.ntiles + tile] = *s_bad;
    }

    tc_fence_before();
    __syncthreads();
    if (warp == kMmaWarp) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tm), "r"(512u));
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
