// convolve_mc.cu -- step a6 for spectral cubes: many channels per sample, fp32, plate-carree
// targets (Sect. 3.4 i-v; Eq. 1 PAPER.md:59 applied per channel with one
// kernel weight and one weight map for all channels -- the paper lists multi-channel
// gridding as "underway"; reading c7 of DESIGN.md).  DESIGN.md "a6 / cube kernel".
//
// A CTA of 8 warps owns 8 x 8 target cells; warp w owns the 4 x 2 sub-tile (w & 1, w >> 1) and
// all channels of a 256-channel block, lane l holding channels 8l .. 8l+7 of its 8 cells in
// 64 accumulators (32 register pairs).  Every warp walks the candidate stream of its own
// sub-tile (built as in convolve_tile.cu); the 8 warps of a CTA are neighbours on the sky,
// so the spectrum rows they share are found in L2.
//   phase 1 (per 32 candidates): lane = candidate; the 8 kernel weights of the sub-tile by
//           the tile kernel's scaled fp32 pair arithmetic; weight map / counts accumulated
//           per lane; candidates that hit at least one of the 8 cells are compacted into a
//           per-warp shared-memory list (8 weights + the row's address)
//   phase 2 (per listed candidate): the warp copies the sample's spectrum row in place
//           (values are never moved: a5) into an 8-deep shared-memory ring with cp.async.cg
//           (L2 only: going through L1 cost 30 %), seven rows ahead of the arithmetic, and
//           does 8 cells x 8 channels of FMAs as 32 packed fma.rn.f32x2.
// Sub-tile rows alternate the ring direction of the stream (north to south, then south to
// north), so vertically adjacent sub-tiles, which start together, meet their shared samples
// at about the same time.
// Reductions in a fixed order, no atomics.
#include "hcg_tile.cuh"

namespace hcg {

struct McArgs {
    TileArgs t;            // tiles_x / ntiles count CTA tiles of 8 x 8 cells
    const float* values;   // [n][nchan], channel fastest, in input order
    int32_t nchan;
};

constexpr int kMcWarps = 8;
constexpr int kMcTile = 8;         // CTA tile edge in cells
constexpr int kSX = 4, kSY = 2;    // sub-tile of one warp
constexpr int kHitStride = 12;     // floats per list entry: 8 weights + row address + pad (48 B)
constexpr int kRowDepth = 8;       // spectrum rows in flight per warp (cp.async ring)
constexpr int kMcSmemWarp = 32 * 16 + 32 * kHitStride * 4 + kRowDepth * 1024 + 2 * 1024;   // table + list + rows + W + counts

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ float4 lds128(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}

__device__ __forceinline__ unsigned long long ffma2(unsigned long long a, unsigned long long b, unsigned long long c) {
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ unsigned long long pack2(float lo, float hi) {
    unsigned long long d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi));
    return d;
}
__device__ __forceinline__ void unpack2(unsigned long long v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}

// Step (v) of phase 1: weights q * w(d) of one candidate for the 4 x 2 cells (0 where d > R).
template <int MODE>
__device__ __forceinline__ unsigned sub_tile_weights(const uint4 raw, const TileConst<kSY>& tc, float (&wq)[8]) {
    const float q = __uint_as_float(raw.w);
    const float dx0 = (float)(int)(raw.x - tc.xc0) * tc.sxk;
    const float dy0 = (float)(int)(raw.y - tc.yc0) * tc.syk;
    const float cs = fmaf(dy0, fmaf(dy0, fmaf(dy0, tc.p3, tc.p2), tc.p1), tc.cc0);
    float V[kSX], U[kSY], C[kSY];
#pragma unroll
    for (int i = 0; i < kSX; ++i) {
        const float dx = i == 0 ? dx0 : fmaf(-(float)i, tc.duk, dx0);
        const float v = dx * dx;
        V[i] = MODE >= 1 ? v * fmaf(v, -tc.a12, 1.0f) : v;
    }
#pragma unroll
    for (int j = 0; j < kSY; ++j) {
        const float dy = j == 0 ? dy0 : fmaf(-(float)j, tc.dyk, dy0);
        const float u = dy * dy;
        U[j] = MODE >= 1 ? u * fmaf(u, -tc.a12, 1.0f) : u;
        C[j] = tc.cc[j] * cs;
    }
    unsigned hits = 0;                                      // bit c: cell c is within R
#pragma unroll
    for (int j = 0; j < kSY; ++j) {
#pragma unroll
        for (int i = 0; i < kSX; ++i) {
            const float h = fmaf(C[j], V[i], U[j]);
            const float e = MODE == 2 ? h * fmaf(h, tc.a12, 1.0f) : h;
            const float w = ex2_approx(-e) * q;
            const bool hit = h <= tc.hm;
            wq[j * kSX + i] = hit ? w : 0.0f;
            hits |= hit ? 1u << (j * kSX + i) : 0u;
        }
    }
    return hits;
}

template <int MODE, bool COUNTS>
__global__ void __launch_bounds__(kMcWarps * 32, 2)
conv_mc_f32(const McArgs m) {
    const TileArgs& a = m.t;
    extern __shared__ __align__(16) unsigned char s_mc[];
    const int lane = threadIdx.x & 31;
    const int wib = threadIdx.x >> 5;
    const int cty = (int)(blockIdx.x / (unsigned)a.tiles_x);
    const int cix0 = (int)(blockIdx.x - (unsigned)cty * (unsigned)a.tiles_x) * kMcTile;
    const int crow0 = cty * kMcTile;
    const int ix0 = cix0 + kSX * (wib & 1);
    const int row0 = crow0 + kSY * (wib >> 1);
    const int ncols = min(kSX, a.nx - ix0);
    const int nrows = min(kSY, a.ny - row0);
    if (ncols <= 0 || nrows <= 0) return;                   // no CTA-wide barrier below

    // ---- sub-tile constants (as conv1_tile_f32 with GX = 4, GY = 2)
    TileConst<kSY> tc;
#pragma unroll
    for (int j = 0; j < kSY; ++j) {
        const int4* rp = (const int4*)(a.rows + min(row0 + j, a.ny - 1));
        const int4 r0 = __ldg(rp);
        tc.cc[j] = __int_as_float(r0.w);
        if (j == 0) {
            const int4 r1 = __ldg(rp + 1);
            tc.yc0 = (uint32_t)r0.x;
            tc.cc0 = __int_as_float(r0.w);
            const float sc0 = __int_as_float(r1.x);
            const float ik = a.isk;
            tc.p1 = -sc0 * ik;
            tc.p2 = -0.5f * tc.cc0 * ik * ik;
            tc.p3 = sc0 * ik * ik * ik * (1.0f / 6.0f);
        }
    }
    tc.xc0 = (uint32_t)(unsigned long long)__double2ll_rn((a.u0 + (double)ix0 * a.du) * a.sx);
    tc.sxk = a.sxk; tc.syk = a.syk; tc.duk = a.duk; tc.dyk = a.dyk;
    tc.a12 = a.a12; tc.hmax = a.hmax; tc.hm = a.hmax;

    // ---- ring range of the sub-tile
    int rmin = 0x7fffffff, rmax = -0x7fffffff;
    for (int j = 0; j < nrows; ++j) {
        const int4 r0 = __ldg((const int4*)(a.rows + row0 + j));
        rmin = min(rmin, r0.y);
        rmax = max(rmax, r0.y + r0.z - 1);
    }
    const float fxw = (float)(a.du >= 0.0 ? ix0 : ix0 + ncols - 1);
    const float fxe = (float)(a.du >= 0.0 ? ix0 + ncols - 1 : ix0);
    const Rec32* __restrict__ rec = a.rec;
    unsigned char* wsm = s_mc + (size_t)wib * kMcSmemWarp;
    ulonglong2* tab = (ulonglong2*)wsm;
    float* hitl = (float*)(wsm + 32 * 16);
    const uint32_t hit_s = smem_addr(hitl);
    const uint32_t vring = smem_addr(wsm + 32 * 16 + 32 * kHitStride * 4) + lane * 32;   // this lane's 32 B of slot 0
    // per-lane partial sums of the weight map and the counts live in shared memory (lane-private)
    float* wacc = (float*)(wsm + 32 * 16 + 32 * kHitStride * 4 + kRowDepth * 1024) + lane * 8;
    int* cacc = (int*)(wacc + 256 - lane * 8) + lane * 8;
    const int nchan = m.nchan;
    const bool flip = ((row0 / kSY) & 1) != 0;              // odd sub-tile rows walk the rings south to north

    for (int ch0 = 0; ch0 < nchan; ch0 += 256) {
        const int chl = ch0 + 8 * lane;                      // first channel of this lane
        const bool ok0 = chl < nchan, ok1 = chl + 4 < nchan; // nchan % 4 == 0 (launcher)
        unsigned long long acc[8][4];
#pragma unroll
        for (int c = 0; c < 8; ++c)
#pragma unroll
            for (int k = 0; k < 4; ++k) acc[c][k] = 0ull;
        *(float4*)wacc = make_float4(0.f, 0.f, 0.f, 0.f);
        *(float4*)(wacc + 4) = make_float4(0.f, 0.f, 0.f, 0.f);
        *(int4*)cacc = make_int4(0, 0, 0, 0);
        *(int4*)(cacc + 4) = make_int4(0, 0, 0, 0);
        const unsigned long long chl_bytes = (unsigned long long)(32 * lane);   // this lane's 8 channels of the block

        for (int rb = 0; rb <= rmax - rmin; rb += 32) {
            // ---- steps (ii)+(iii) for the sub-tile: lane k <-> ring number k of this pass
            const int r = flip ? rmax - rb - lane : rmin + rb + lane;
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
            int sa = 0, sn = 0;
            if (jhi >= jlo && r >= rmin && r <= rmax) {
                const int32_t* bs = a.bin_start + (size_t)r * a.m;
                sa = __ldg(bs + jlo);
                sn = __ldg(bs + jhi + 1) - sa;
            }
            int incl = sn;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += t;
            }
            const int total = __shfl_sync(0xffffffffu, incl, 31);
            __syncwarp();
            tab[lane] = make_ulonglong2((unsigned long long)(unsigned)incl,
                                        (unsigned long long)(uintptr_t)(rec + ((long long)sa - (incl - sn))));
            __syncwarp();
            if (total == 0) continue;

            // ---- the candidate stream in chunks of 32
            const int last = total - 1;
            const int niter = (total + 31) >> 5;
            uint32_t tp = smem_addr(tab);
            unsigned long long end, base;
            lds_entry(tp, end, base);
            int i = lane;
            stream_seek(min(i, last), tp, end, base);
            uint4 cur = ldg_rec(base, min(i, last));
            for (int it = 0; it < niter; ++it) {
                // next chunk's record, in flight during phase 2
                const int i1 = i + 32;
                const int ii = min(i1, last);
                stream_seek(ii, tp, end, base);
                const uint4 nxt = ldg_rec(base, ii);

                // phase 1
                float wq[8];
                tc.hm = i <= last ? tc.hmax : -1.0f;
                const unsigned hits = sub_tile_weights<MODE>(cur, tc, wq);
                const unsigned mask = __ballot_sync(0xffffffffu, hits != 0);
                if (hits != 0) {
                    float* e = hitl + __popc(mask & ((1u << lane) - 1u)) * kHitStride;
                    *(float4*)(e + 0) = make_float4(wq[0], wq[1], wq[2], wq[3]);
                    *(float4*)(e + 4) = make_float4(wq[4], wq[5], wq[6], wq[7]);
                    *(unsigned long long*)(e + 8) =
                        (unsigned long long)(uintptr_t)(m.values + (size_t)cur.z * nchan + ch0);
                    float4 w0 = *(float4*)wacc, w1 = *(float4*)(wacc + 4);
                    w0.x += wq[0]; w0.y += wq[1]; w0.z += wq[2]; w0.w += wq[3];
                    w1.x += wq[4]; w1.y += wq[5]; w1.z += wq[6]; w1.w += wq[7];
                    *(float4*)wacc = w0; *(float4*)(wacc + 4) = w1;
                    if (COUNTS) {
                        int4 c0 = *(int4*)cacc, c1 = *(int4*)(cacc + 4);
                        c0.x += hits & 1; c0.y += (hits >> 1) & 1; c0.z += (hits >> 2) & 1; c0.w += (hits >> 3) & 1;
                        c1.x += (hits >> 4) & 1; c1.y += (hits >> 5) & 1; c1.z += (hits >> 6) & 1; c1.w += (hits >> 7) & 1;
                        *(int4*)cacc = c0; *(int4*)(cacc + 4) = c1;
                    }
                }
                __syncwarp();

                // phase 2: explicit shared addresses, so the loop carries only e, the entry and the slot
                const int nhit = __popc(mask);
                if (nhit > 0) {
                    auto issue = [&](uint32_t ent_s, uint32_t dst) {
                        unsigned long long rp;
                        asm volatile("ld.shared.u64 %0, [%1+32];" : "=l"(rp) : "r"(ent_s));
                        rp += chl_bytes;
                        if (ok0) cp_async16(dst, (const void*)(uintptr_t)rp);
                        if (ok1) cp_async16(dst + 16, (const void*)(uintptr_t)(rp + 16));
                    };
#pragma unroll
                    for (int p = 0; p < kRowDepth - 1; ++p) {
                        if (p < nhit) issue(hit_s + p * (kHitStride * 4), vring + p * 1024);
                        cp_async_commit();
                    }
                    uint32_t ent_s = hit_s;
#pragma unroll 4
                    for (int e = 0; e < nhit; ++e, ent_s += kHitStride * 4) {
                        if (e + kRowDepth - 1 < nhit)
                            issue(ent_s + (kRowDepth - 1) * (kHitStride * 4),
                                  vring + (uint32_t)((e + kRowDepth - 1) & (kRowDepth - 1)) * 1024u);
                        cp_async_commit();
                        // the 8 weights by two broadcast loads, issued before the wait for the row so that
                        // their latency hides behind it; each weight is paired with itself in registers
                        // (duplicated pairs in shared memory cost twice the load/store-pipe cycles)
                        const float4 wlo = lds128(ent_s), whi = lds128(ent_s + 16);
                        cp_async_wait<kRowDepth - 1>();     // row e has landed (each lane reads its own bytes)
                        const uint32_t src = vring + (uint32_t)(e & (kRowDepth - 1)) * 1024u;
                        // lanes past nchan read stale shared memory: their sums are never stored
                        const float4 va = lds128(src), vb = lds128(src + 16);
                        const unsigned long long v01 = pack2(va.x, va.y), v23 = pack2(va.z, va.w);
                        const unsigned long long v45 = pack2(vb.x, vb.y), v67 = pack2(vb.z, vb.w);
                        const float wv[8] = {wlo.x, wlo.y, wlo.z, wlo.w, whi.x, whi.y, whi.z, whi.w};
#pragma unroll
                        for (int c = 0; c < 8; ++c) {
                            const unsigned long long ww = pack2(wv[c], wv[c]);
                            acc[c][0] = ffma2(v01, ww, acc[c][0]);
                            acc[c][1] = ffma2(v23, ww, acc[c][1]);
                            acc[c][2] = ffma2(v45, ww, acc[c][2]);
                            acc[c][3] = ffma2(v67, ww, acc[c][3]);
                        }
                    }
                }
                __syncwarp();                               // list is rewritten by the next chunk
                cur = nxt;
                i = i1;
            }
        }

        // ---- finish this channel block: W (and counts) across lanes, normalise, store
        float W[8];
        int cnt[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) { W[c] = wacc[c]; cnt[c] = cacc[c]; }
        TileReduce<8, 16, float>::run(W, lane);
        if (COUNTS) TileReduce<8, 16, int>::run(cnt, lane);
        const float wmine = W[0];                           // lane L holds cell L >> 2
        if (ch0 == 0 && (lane & 3) == 0) {
            const int c = lane >> 2;
            const int gx = c % kSX, gy = c / kSX;
            if (gx < ncols && gy < nrows) {
                const int64_t cell = (int64_t)(row0 + gy) * a.nx + ix0 + gx;
                a.wmap[cell] = wmine;
                if (COUNTS) a.counts[cell] = cnt[0];
            }
        }
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const float wc = __shfl_sync(0xffffffffu, wmine, 4 * c);
            const int gx = c % kSX, gy = c / kSX;
            if (gx < ncols && gy < nrows) {
                const int64_t cell = (int64_t)(row0 + gy) * a.nx + ix0 + gx;
                float* o = a.cube + (size_t)cell * nchan + chl;
                float f[8];
#pragma unroll
                for (int k = 0; k < 4; ++k) unpack2(acc[c][k], f[2 * k], f[2 * k + 1]);
                const float nan = __int_as_float(0x7fc00000);
#pragma unroll
                for (int k = 0; k < 8; ++k) f[k] = a.raw ? f[k] : (wc > 0.0f ? f[k] / wc : nan);
                if (ok0) *(float4*)o = make_float4(f[0], f[1], f[2], f[3]);
                if (ok1) *(float4*)(o + 4) = make_float4(f[4], f[5], f[6], f[7]);
            }
        }
    }
}

int launch_conv_mc(hcgrid_ctx* c, const float* values, int nchan, float* cube, float* wmap, int32_t* counts,
                   cudaStream_t st) {
    const int mode = tile_series_mode(c);
    McArgs m{};
    fill_tile_args(c, mode, m.t);
    m.t.cube = cube; m.t.wmap = wmap; m.t.counts = counts;
    m.t.tiles_x = (m.t.nx + kMcTile - 1) / kMcTile;
    m.t.ntiles = (int64_t)m.t.tiles_x * ((m.t.ny + kMcTile - 1) / kMcTile);
    m.values = values;
    m.nchan = nchan;
    const unsigned blocks = (unsigned)m.t.ntiles;
    const int threads = kMcWarps * 32;
    const int smem = kMcWarps * kMcSmemWarp;
#define HCG_MC(M, C)                                                                                   \
    do {                                                                                               \
        HCG_CUDA(c, cudaFuncSetAttribute(conv_mc_f32<M, C>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)); \
        conv_mc_f32<M, C><<<blocks, threads, smem, st>>>(m);                                           \
    } while (0)
    switch (mode * 2 + (counts ? 1 : 0)) {
        case 0: HCG_MC(0, false); break;
        case 1: HCG_MC(0, true); break;
        case 2: HCG_MC(1, false); break;
        case 3: HCG_MC(1, true); break;
        case 4: HCG_MC(2, false); break;
        default: HCG_MC(2, true); break;
    }
#undef HCG_MC
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e, "conv_mc_f32");
    c->stats.coarsen = kSX;
    c->stats.coarsen_y = kSY;
    return HCGRID_OK;
}

}  // namespace hcg
