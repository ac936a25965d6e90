// hcg_tile.cuh -- what the tile kernels (convolve_tile.cu: one channel; convolve_mc.cu: many
// channels) share: the argument block, the scaled fp32 pair arithmetic of step (v), the
// candidate stream's ring cursor of step (iv) and the transposed warp reduction.
#pragma once
#include "hcg_conv.cuh"

namespace hcg {

struct TileArgs {
    const RowF* rows;
    const RingWinF* wins;
    const int32_t* bin_start;
    const Rec32* rec;
    float* cube;
    float* wmap;
    int32_t* counts;
    double u0, du, sx;          // lon offset of column 0 (rad), column step (rad), fixed-point units per rad
    int32_t nx, ny, kmax, m;    // target shape, window-table row length, lookup bins per ring
    int32_t tiles_x;
    int32_t raw;                // 1: write the un-normalised sums (incremental gridding), 0: sums / W
    int32_t split;              // warps per tile (1, 2, 4 or 8): long candidate streams of few tiles are split
    int64_t ntiles;
    float sxk, syk;             // sqrt(kappa) * radians per fixed-point unit (lon, lat)
    float duk, dyk;             // sqrt(kappa) * column step / row step (signed)
    float isk;                  // 1 / sqrt(kappa)
    float a12;                  // 1 / (12 kappa): series coefficient in scaled units
    float hmax;                 // kappa * 4 sin^2(R/2)  (series modes)  or  kappa * R^2 (flat mode)
    float ts1, tg2;             // tapered sinc (KFN 1): sinc argument = ts1 sqrt(e), taper = ex2(-e tg2)
    float ecp, esp, erk;        // elliptical Gaussian (KFN 2): cos PA, sin PA, (sigma_1 / sigma_2)^2 - 1
};

template <int GY>
struct TileConst {
    uint32_t xc0, yc0;
    float sxk, syk, duk, dyk;
    float cc0, p1, p2, p3;      // cos(lat_s) = cc0 + dy (p1 + dy (p2 + dy p3)), dy scaled
    float cc[GY];
    float a12, hmax;
    float hm;                   // hmax, or -1 for a lane that is past the end of the stream
    float ts1, tg2;             // KFN 1 only
    float ecp, esp, erk;        // KFN 2 only
    float sh[GY];               // KFN 2 only: sin(lat_c) / (2 sqrt(kappa)) of the tile's rows
};

// Tapered sinc from e = kappa d^2 (the Gaussian's base-2 exponent): sinc(ts1 sqrt(e)) ex2(-e tg2).
// sin by hand: y = k pi + r, |r| <= pi/2 (pi split in two so that k pi is exact for the k <= ~30 the
// support radius allows), odd Taylor polynomial to r^11 (next term r^13/13! <= 5.7e-8), sign from k's parity.
__device__ __forceinline__ float tile_tapered_sinc(float e, float ts1, float tg2) {
    const float y = ts1 * sqrtf(e);
    const float kb = fmaf(y, 0.318309886f, 12582912.0f);          // 1.5 * 2^23: the integer lands in the low bits
    const float k = kb - 12582912.0f;
    float r = fmaf(k, -3.140625f, y);
    r = fmaf(k, -9.67653589793e-4f, r);
    const float r2 = r * r;
    float p = fmaf(r2, -2.50521084e-8f, 2.75573192e-6f);
    p = fmaf(r2, p, -1.98412698e-4f);
    p = fmaf(r2, p, 8.33333333e-3f);
    p = fmaf(r2, p, -1.66666667e-1f);
    p = fmaf(r2 * r, p, r);
    const float s = __uint_as_float(__float_as_uint(p) ^ (__float_as_uint(kb) << 31));
    const float sinc = y < 1e-4f ? 1.0f : __fdividef(s, y);
    return sinc * ex2_approx(-e * tg2);
}

// MODE 0 "flat": d^2 = dy^2 + cos cos dx^2 (valid while R^2/12 and dl_max^2/12 < 1e-7);
// MODE 1 "series": 4 hav(d) = u(1-u/12) + C v(1-v/12) for the test, weight from the same;
// MODE 2 "full": as 1, plus d^2 = h(1 + h/12) for the weight.
// KFN 0: Gaussian, w = ex2(-e); KFN 1: tapered sinc of the same e (hcgrid_set_kernel).
// KFN 2: elliptical Gaussian (reading c21; MODE 2 only), w = ex2(-(e + erk t^2 (1 + h / (3 kappa)))) with
//   t = sqrt(kappa) (x cos PA - y sin PA),  x = cos(lat_s) sin dx,  y = sin dy + sin(lat_c) cos(lat_s) 2 sin^2(dx / 2)
// -- x, y the sample's direction along the cell's east and north, (d sin(beta - PA))^2 = (x cos PA - y sin PA)^2
// (d / sin d)^2, (d / sin d)^2 = 1 + d^2 / 3 + ...; in the scaled units sin z = z (1 - 2 a12 z^2 + 1.2 a12^2 z^4) and
// 2 sin^2(dx / 2) = V / (2 kappa).
template <int GX, int GY, int MODE, bool COUNTS, int KFN = 0>
__device__ __forceinline__ void tile_pairs(const uint4 raw, const TileConst<GY>& tc, float (&W)[GX * GY],
                                           float (&S)[GX * GY], int (&cnt)[GX * GY]) {
    const float q = __uint_as_float(raw.w);
    const float qv = q * __uint_as_float(raw.z);
    const float dx0 = (float)(int)(raw.x - tc.xc0) * tc.sxk;
    const float dy0 = (float)(int)(raw.y - tc.yc0) * tc.syk;
    const float cs = fmaf(dy0, fmaf(dy0, fmaf(dy0, tc.p3, tc.p2), tc.p1), tc.cc0);
    float V[GX], U[GY], C[GY];
    float X[GX], Y[GY], SH[GY];                    // KFN 2: x cos PA; sin(dy) sin PA; sin(lat_c) cos(lat_s) sin PA / 2, scaled
    const float a6 = 2.0f * tc.a12, a120 = 1.2f * tc.a12 * tc.a12;
#pragma unroll
    for (int i = 0; i < GX; ++i) {
        const float dx = i == 0 ? dx0 : fmaf(-(float)i, tc.duk, dx0);
        const float v = dx * dx;
        V[i] = MODE >= 1 ? v * fmaf(v, -tc.a12, 1.0f) : v;
        if (KFN == 2) X[i] = dx * fmaf(v, fmaf(v, a120, -a6), 1.0f) * (cs * tc.ecp);
    }
#pragma unroll
    for (int j = 0; j < GY; ++j) {
        const float dy = j == 0 ? dy0 : fmaf(-(float)j, tc.dyk, dy0);
        const float u = dy * dy;
        U[j] = MODE >= 1 ? u * fmaf(u, -tc.a12, 1.0f) : u;
        C[j] = tc.cc[j] * cs;
        if (KFN == 2) {
            Y[j] = dy * fmaf(u, fmaf(u, a120, -a6), 1.0f) * tc.esp;
            SH[j] = tc.sh[j] * (cs * tc.esp);
        }
    }
#pragma unroll
    for (int j = 0; j < GY; ++j) {
#pragma unroll
        for (int i = 0; i < GX; ++i) {
            const float h = fmaf(C[j], V[i], U[j]);
            float e = MODE == 2 ? h * fmaf(h, tc.a12, 1.0f) : h;
            if (KFN == 2) {
                const float t = fmaf(-SH[j], V[i], X[i] - Y[j]);
                e = fmaf(tc.erk * (t * t), fmaf(h, 4.0f * tc.a12, 1.0f), e);
            }
            const float w = KFN == 1 ? tile_tapered_sinc(fmaxf(e, 0.0f), tc.ts1, tc.tg2) : ex2_approx(-e);
            // predicated accumulate, spelled out so the count stays one predicated add
            if (COUNTS)
                asm("{\n\t.reg .pred p;\n\t"
                    "setp.le.f32 p, %3, %4;\n\t"
                    "@p fma.rn.f32 %0, %5, %6, %0;\n\t"
                    "@p fma.rn.f32 %1, %5, %7, %1;\n\t"
                    "@p add.s32 %2, %2, 1;\n\t}"
                    : "+f"(W[j * GX + i]), "+f"(S[j * GX + i]), "+r"(cnt[j * GX + i])
                    : "f"(h), "f"(tc.hm), "f"(w), "f"(q), "f"(qv));
            else if (h <= tc.hm) {
                W[j * GX + i] = fmaf(w, q, W[j * GX + i]);
                S[j * GX + i] = fmaf(w, qv, S[j * GX + i]);
            }
        }
    }
}

// Transposed warp reduction of N (a power of two <= 32) per-lane values: after the call
// v[0] of lane L holds the sum over all 32 lanes of value number L >> (5 - log2 N).
template <int N, int SH, typename T>
struct TileReduce {
    static __device__ __forceinline__ void run(T* v, int lane) {
        if constexpr (SH >= 1) {
            if constexpr (N > 1) {
                constexpr int H = N / 2;
                const bool up = (lane & SH) != 0;
#pragma unroll
                for (int i = 0; i < H; ++i) {
                    const T keep = up ? v[i + H] : v[i];
                    const T send = up ? v[i] : v[i + H];
                    v[i] = keep + __shfl_xor_sync(0xffffffffu, send, SH);
                }
                TileReduce<H, SH / 2, T>::run(v, lane);
            } else {
                v[0] += __shfl_xor_sync(0xffffffffu, v[0], SH);
                TileReduce<1, SH / 2, T>::run(v, lane);
            }
        }
    }
};

// ---- the candidate stream's ring cursor (step iv): entry k of the per-warp table is
// (end position of ring k in the stream, record address of stream index 0 within ring k)
__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void lds_entry(uint32_t tp, unsigned long long& end, unsigned long long& base) {
    asm volatile("ld.shared.v2.u64 {%0, %1}, [%2];" : "=l"(end), "=l"(base) : "r"(tp));
}
__device__ __forceinline__ void stream_seek(int i, uint32_t& tp, unsigned long long& end, unsigned long long& base) {
    // a step of 32 usually crosses one ring boundary: one predicated advance, then the loop
    asm volatile("{\n\t.reg .pred p;\n\t"
                 "setp.ge.s32 p, %3, %4;\n\t"
                 "@p add.u32 %2, %2, 16;\n\t"
                 "@p ld.shared.v2.u64 {%0, %1}, [%2];\n\t}"
                 : "+l"(end), "+l"(base), "+r"(tp) : "r"(i), "r"((int)end));
    while (i >= (int)end) {
        tp += 16;
        lds_entry(tp, end, base);
    }
}
__device__ __forceinline__ uint4 ldg_rec(unsigned long long base, int i) {
    return __ldg((const uint4*)(uintptr_t)(base + (unsigned long long)(unsigned)i * 16ull));
}

// The same cursor with 8-byte table entries (the tile kernel): low word = end of ring k in the stream, high word =
// record index of the record that would have stream index 0 (may be negative).  One 64-bit load lands in the
// register pair that holds the entry -- no copies -- and the record address is rec + (base + i).
__device__ __forceinline__ unsigned long long lds_entry8(uint32_t tp) {
    unsigned long long eb;
    asm volatile("ld.shared.u64 %0, [%1];" : "=l"(eb) : "r"(tp));
    return eb;
}
__device__ __forceinline__ void stream_seek8(int i, uint32_t& tp, unsigned long long& eb) {
    asm volatile("{\n\t.reg .pred p;\n\t.reg .b32 e, b;\n\t"
                 "mov.b64 {e, b}, %0;\n\t"
                 "setp.ge.s32 p, %2, e;\n\t"
                 "@p add.u32 %1, %1, 8;\n\t"
                 "@p ld.shared.u64 %0, [%1];\n\t}"
                 : "+l"(eb), "+r"(tp) : "r"(i));
    while (i >= (int)(uint32_t)eb) {
        tp += 8;
        eb = lds_entry8(tp);
    }
}
__device__ __forceinline__ uint4 ldg_rec8(const Rec32* __restrict__ rec, unsigned long long eb, int i) {
    return __ldg((const uint4*)rec + ((int)(eb >> 32) + i));
}

constexpr int ilog2(int n) { return n <= 1 ? 0 : 1 + ilog2(n / 2); }

// Host side: the fields of TileArgs that depend only on the context (not on the tile shape
// or the outputs), and the series mode the tolerances need.
int tile_series_mode(const hcgrid_ctx* c);
void fill_tile_args(const hcgrid_ctx* c, int mode, TileArgs& a);

}  // namespace hcg
