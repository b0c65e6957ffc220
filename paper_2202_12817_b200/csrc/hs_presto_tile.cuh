// PRESTO-like harmonic sum (Alg. 1; eq. 4), tile kernel:
// every lane owns 16 CONSECUTIVE top bins, so that each term of eq. 4 is a compile-time offset
// into a short private row that the lane reads with vector loads.
//
// Index algebra.  Alg. 1 visits x[Round(h n / H')] for H' = 1, 2, 4, .., Hq = 2^L and
// h in {1} U {2, 4, .., H'}.  Written in 32nds the fractions h/H' are kk/32 with
//     level 0: kk = 32            level 1: 16           level 2: 8           level 3: 4, 24
//     level 4: 2, 12, 20, 28      level 5: 1, 6, 10, 14, 18, 22, 26, 30
// (the harmonic sets are nested: S_{2H'} = S_{H'} + the terms of level log2(2H')),
// and Round is round-half-up in exact integers (reading R3):  idx = (kk n + 16) >> 5.
// For n = n0 + 16 i + e  (n0 a multiple of 512, lane i, e = 0..15):
//     idx = kk n0/32 + (kk/2) i + ((kk e + 16) >> 5)            (kk even)
//     idx = n0/32 + ((i + 1) >> 1)                              (kk = 1: one element for all e)
// so lane i reads the kk/2 + 1 elements that start at (kk/2) i of the span x[kk n0/32 ..], at offsets
// known when the kernel is compiled: 147 elements for its 16 outputs instead of 17 x 16 separate loads.
//
// Data movement of a CTA tile of T = 512 W outputs (W pairs of warps):
//   * 14 spans (all fractions but kk = 32, 16 and 8) are copied into shared memory as they are by one 1-D bulk
//     async copy each (TMA engine, cp.async.bulk -> UBLKCP), completing on one mbarrier; a lane stride of
//     kk/2 words makes the vector loads LDS.128 / .64 / .32 bank-conflict free for every one of them;
//   * kk = 32 (x[n] itself) and kk = 16 would bank-conflict at lane strides of 16 / 8 words (kk = 8 joins them so that
//     the tile's shared memory drops under 27.5 KB and an SM holds 8 CTAs instead of 7), and a lane's words
//     are contiguous in global memory too: they are loaded straight into registers (LDG.256 / LDG.128) while
//     the bulk copies are in flight, which also keeps 12 B/bin off the shared-memory pipe;
//   * two warps share each 512-output warp tile (one takes outputs e < 8 of every lane's 16, the other e >= 8):
//     twice the warps for the same shared memory (occupancy is set by shared memory: 28 000 B = 27.3 KB per CTA at
//     W = 2 and H = 32, so an SM holds 8 CTAs);
//   * a lane's 8 outputs are consecutive: they are stored from registers as whole 32-byte sectors
//     (st.global.v8 -> STG.E.256): no transposition through shared memory, no barrier.
// Staging, arithmetic and stores of different tiles overlap across the 8 CTAs an SM holds (one tile per CTA: the
// kernel is not persistent, the grid has one CTA per tile and spectrum).
#pragma once
#include "hs_common.cuh"

namespace hs_tile {

constexpr int G = 16;                       // outputs per lane
constexpr int TILE = 32 * G;                // outputs per warp tile (one pair of warps)

// fraction table in enumeration order (level-major), L levels
__host__ __device__ constexpr int n_frac(int L) { return L == 0 ? 1 : L <= 2 ? L + 1 : L == 3 ? 5 : L == 4 ? 9 : 17; }
__host__ __device__ constexpr int frac_kk(int f) {
    constexpr int t[17] = {32, 16, 8, 4, 24, 2, 12, 20, 28, 1, 6, 10, 14, 18, 22, 26, 30};
    return t[f];
}
// words of shared memory of the span of fraction kk of a CTA tile of W warp tiles (+ 4: the word shared with the next tile)
__host__ __device__ constexpr int span_words(int kk, int W) { return 16 * kk * W + 4; }
// stage layout: fractions 3 .. NF-1 (kk = 4, 24, 2, ...) back to back; 0 (kk = 32), 1 (kk = 16) and 2 (kk = 8) stay in registers
constexpr int F_SMEM = 3;                   // first fraction that goes through shared memory
__host__ __device__ constexpr int span_off(int f, int W) {
    int o = 0;
    for (int g = F_SMEM; g < f; ++g) o += span_words(frac_kk(g), W);
    return o;
}
__host__ __device__ constexpr int smem_words(int L, int W) { return n_frac(L) > F_SMEM ? span_off(n_frac(L), W) : 4; }

// offset of output e in the row of fraction kk (kk even)
__host__ __device__ constexpr int row_off(int kk, int e) { return (kk * e + 16) >> 5; }

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    unsigned done = 0;
    while (!done) {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
                     : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    }
}

// t[p - LO] = row[p] for p = P .. HI: 16-, 8- or 4-byte loads, whichever is aligned (the row start is aligned to A words)
// and stays inside the range
template <int A, int LO, int P, int HI, int NW>
__device__ __forceinline__ void load_words(const float* __restrict__ row, float (&t)[NW]) {
    if constexpr (P <= HI) {
        if constexpr (A >= 4 && P % 4 == 0 && P + 3 <= HI) {
            const float4 q = *reinterpret_cast<const float4*>(row + P);
            t[P - LO] = q.x; t[P - LO + 1] = q.y; t[P - LO + 2] = q.z; t[P - LO + 3] = q.w;
            load_words<A, LO, P + 4, HI>(row, t);
        } else if constexpr (A >= 2 && P % 2 == 0 && P + 1 <= HI) {
            const float2 q = *reinterpret_cast<const float2*>(row + P);
            t[P - LO] = q.x; t[P - LO + 1] = q.y;
            load_words<A, LO, P + 2, HI>(row, t);
        } else {
            t[P - LO] = row[P];
            load_words<A, LO, P + 1, HI>(row, t);
        }
    }
}

// add the term of fraction KK to the accumulators of outputs e = E0 + u, u = 0..NE-1
// (FIRST: they are set, not added to)
template <int KK, int E0, int NE, bool FIRST>
__device__ __forceinline__ void add_terms(const float* __restrict__ row, float (&acc)[NE]) {
    if (KK == 1) {                                       // one element for the whole lane
        const float v = row[0];
#pragma unroll
        for (int u = 0; u < NE; ++u) acc[u] = FIRST ? v : __fadd_rn(acc[u], v);
        return;
    }
    constexpr int lo = row_off(KK, E0), hi = row_off(KK, E0 + NE - 1);
    constexpr int A = (KK % 8 == 0) ? 4 : (KK % 4 == 0) ? 2 : 1;     // words the row start is aligned to
    // exactly the words lo .. hi, by the widest aligned loads that stay inside them (the shared-memory pipe is the
    // kernel's busiest unit: a 16-byte load that is only half used costs its full 4 wavefronts)
    float t[hi - lo + 1];
    load_words<A, lo, lo, hi>(row, t);
#pragma unroll
    for (int u = 0; u < NE; ++u) {
        const float v = t[row_off(KK, E0 + u) - lo];
        acc[u] = FIRST ? v : __fadd_rn(acc[u], v);
    }
}

// S += add, SNR at H' = HP (once per H', reading R2), strict > keeps the first maximum (R6)
template <int HP, int NE>
__device__ __forceinline__ void close_level(const HsStats& st, float (&S)[NE], const float (&add)[NE], float (&best)[NE], int (&bh)[NE]) {
#pragma unroll
    for (int u = 0; u < NE; ++u) {
        S[u] = __fadd_rn(S[u], add[u]);
        const float snr = hs_snr(S[u], st.nmis[HP - 1], st.inv_sigma[HP - 1]);
        if (snr > best[u]) { best[u] = snr; bh[u] = HP; }
    }
}

// start of the row of lane `lane` of warp tile w in the span of fraction F
template <int F, int W>
__device__ __forceinline__ const float* row_ptr(const float* __restrict__ sm, int w, int lane) {
    constexpr int kk = frac_kk(F);
    if (kk == 1) return sm + span_off(F, W) + 16 * w + ((lane + 1) >> 1);
    return sm + span_off(F, W) + 16 * kk * w + (kk / 2) * lane;
}

// the words of 8 outputs of a lane that come straight from global memory:
// xr = x[n .. n + 8) (fraction 32/32), yr = x[i16 .. i16 + 5) (fraction 16/32: output u reads yr[(u + 1) >> 1])
// zr = x[i8 .. i8 + 3) (fraction 8/32: output u reads zr[(u + 2) >> 2])
struct Direct {
    float xr[8];
    float yr[5];
    float zr[3];
};

template <int L>
__device__ __forceinline__ void load_direct(Direct& d, const float* __restrict__ x, const float* __restrict__ x16, const float* __restrict__ x8,
                                            int N, int n, int i16, int i8, bool interior, bool al32) {   // x16, x8: the rows fractions 16/32, 8/32 read from (x itself in 1-D)
    if (interior) {
        if (al32) {
            asm volatile("ld.global.nc.L1::no_allocate.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n"
                         : "=f"(d.xr[0]), "=f"(d.xr[1]), "=f"(d.xr[2]), "=f"(d.xr[3]), "=f"(d.xr[4]), "=f"(d.xr[5]), "=f"(d.xr[6]), "=f"(d.xr[7])
                         : "l"(x + n));
        } else {                                             // rows that start on an odd 16-byte unit
            asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];\n"
                         : "=f"(d.xr[0]), "=f"(d.xr[1]), "=f"(d.xr[2]), "=f"(d.xr[3]) : "l"(x + n));
            asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];\n"
                         : "=f"(d.xr[4]), "=f"(d.xr[5]), "=f"(d.xr[6]), "=f"(d.xr[7]) : "l"(x + n + 4));
        }
        if (L >= 1) {
            asm volatile("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];\n"
                         : "=f"(d.yr[0]), "=f"(d.yr[1]), "=f"(d.yr[2]), "=f"(d.yr[3]) : "l"(x16 + i16));
            asm volatile("ld.global.nc.f32 %0, [%1];\n" : "=f"(d.yr[4]) : "l"(x16 + i16 + 4));
        }
        if (L >= 2) {
            asm volatile("ld.global.nc.v2.f32 {%0,%1}, [%2];\n" : "=f"(d.zr[0]), "=f"(d.zr[1]) : "l"(x8 + i8));
            asm volatile("ld.global.nc.f32 %0, [%1];\n" : "=f"(d.zr[2]) : "l"(x8 + i8 + 2));
        }
    } else {                                                 // the last tile of a row: element-wise, zero beyond the end
#pragma unroll
        for (int u = 0; u < 8; ++u) d.xr[u] = (n + u < N) ? __ldg(x + n + u) : 0.f;
        if (L >= 1) {
#pragma unroll
            for (int u = 0; u < 5; ++u) d.yr[u] = (i16 + u < N) ? __ldg(x16 + i16 + u) : 0.f;
        }
        if (L >= 2) {
#pragma unroll
            for (int u = 0; u < 3; ++u) d.zr[u] = (i8 + u < N) ? __ldg(x8 + i8 + u) : 0.f;
        }
    }
}

// all levels for outputs e = E0 + u, u < 8, of the lane, level by level:
// S_{2H'} = S_{H'} + (the new terms of the level, summed first)
struct NoWait { __device__ __forceinline__ void operator()() const {} };
template <int L, int E0, int W, class BeforeL5 = NoWait>
__device__ __forceinline__ void chain8(const float* __restrict__ sm, const HsStats& st, int w, int lane, const Direct& d,
                                       float (&best)[8], int (&bh)[8], BeforeL5 before_l5 = NoWait()) {
    float S[8], add[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) { S[u] = d.xr[u]; best[u] = hs_snr(S[u], st.nmis[0], st.inv_sigma[0]); bh[u] = 1; }   // H' = 1: x[n]
    if (L >= 1) {
#pragma unroll
        for (int u = 0; u < 8; ++u) add[u] = d.yr[(u + 1) >> 1];
        close_level<2, 8>(st, S, add, best, bh);
    }
    if (L >= 2) {
#pragma unroll
        for (int u = 0; u < 8; ++u) add[u] = d.zr[(u + 2) >> 2];
        close_level<4, 8>(st, S, add, best, bh);
    }
    if (L >= 3) {
        add_terms<4, E0, 8, true>(row_ptr<3, W>(sm, w, lane), add);
        add_terms<24, E0, 8, false>(row_ptr<4, W>(sm, w, lane), add);
        close_level<8, 8>(st, S, add, best, bh);
    }
    if (L >= 4) {
        add_terms<2, E0, 8, true>(row_ptr<5, W>(sm, w, lane), add);
        add_terms<12, E0, 8, false>(row_ptr<6, W>(sm, w, lane), add);
        add_terms<20, E0, 8, false>(row_ptr<7, W>(sm, w, lane), add);
        add_terms<28, E0, 8, false>(row_ptr<8, W>(sm, w, lane), add);
        close_level<16, 8>(st, S, add, best, bh);
    }
    if (L >= 5) {
        before_l5();                                        // the level-5 spans may complete on a barrier of their own
        add_terms<1, E0, 8, true>(row_ptr<9, W>(sm, w, lane), add);
        add_terms<6, E0, 8, false>(row_ptr<10, W>(sm, w, lane), add);
        add_terms<10, E0, 8, false>(row_ptr<11, W>(sm, w, lane), add);
        add_terms<14, E0, 8, false>(row_ptr<12, W>(sm, w, lane), add);
        add_terms<18, E0, 8, false>(row_ptr<13, W>(sm, w, lane), add);
        add_terms<22, E0, 8, false>(row_ptr<14, W>(sm, w, lane), add);
        add_terms<26, E0, 8, false>(row_ptr<15, W>(sm, w, lane), add);
        add_terms<30, E0, 8, false>(row_ptr<16, W>(sm, w, lane), add);
        close_level<32, 8>(st, S, add, best, bh);
    }
}

// 8 consecutive outputs of a lane, starting at bin n of the row
__device__ __forceinline__ void store8(float* __restrict__ ps, int* __restrict__ pb, int n, int n_fund, bool full, bool al32,
                                       const float (&v)[8], const int (&b)[8]) {
    if (full && al32) {
        asm volatile("st.global.cs.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};\n" :: "l"(ps), "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]),
                     "f"(v[4]), "f"(v[5]), "f"(v[6]), "f"(v[7]) : "memory");
        asm volatile("st.global.cs.v8.s32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};\n" :: "l"(pb), "r"(b[0]), "r"(b[1]), "r"(b[2]), "r"(b[3]),
                     "r"(b[4]), "r"(b[5]), "r"(b[6]), "r"(b[7]) : "memory");
    } else if (full) {                                       // rows that start on an odd 16-byte unit
        __stcs(reinterpret_cast<float4*>(ps), make_float4(v[0], v[1], v[2], v[3]));
        __stcs(reinterpret_cast<float4*>(ps + 4), make_float4(v[4], v[5], v[6], v[7]));
        __stcs(reinterpret_cast<int4*>(pb), make_int4(b[0], b[1], b[2], b[3]));
        __stcs(reinterpret_cast<int4*>(pb + 4), make_int4(b[4], b[5], b[6], b[7]));
    } else {
#pragma unroll
        for (int u = 0; u < 8; ++u)
            if (n + u < n_fund) { st_cs(ps + u, v[u]); st_cs(pb + u, b[u]); }
    }
}

}  // namespace hs_tile

// grid: (tiles of 512 W outputs, spectra); block: 64 W threads; dynamic shared memory: 4 smem_words(L, W) bytes
// TWOD (hs_plan_2d, reading R15): blockIdx.y is the row z + Z of an f-fdot plane and the term of fraction kk/32 is read
// from row Round(kk z / 32) = (kk z + 16) >> 5 (arithmetic shift = floor: half up also for negative z) -- the same
// for the whole tile, so every span is still one contiguous copy, only from its own row.
// SPLIT: the spans of levels 2-4 (issued first) and of level 5 complete on separate mbarriers, so the first 9 terms are
// added while the 8 longest spans are still landing (2.97 against 3.01 ms at H = 32; no gain below).  A warp of its own
// for the issue, and two issuing threads with a barrier each, were measured too: 2.96-3.05 ms, not kept.
template <int L, int W, bool DSTATS = false, bool TWOD = false, bool SPLIT = false>
__global__ void __launch_bounds__(64 * W)
hs_presto_tile_kernel(const __grid_constant__ HsShape sh, const __grid_constant__ HsStats st_param, HsIO io) {
    using namespace hs_tile;
    __shared__ float s_st_raw[DSTATS ? sizeof(HsStats) / 4 : 1];     // only the per-spectrum-statistics build pays for it
    HsStats& s_st = *reinterpret_cast<HsStats*>(s_st_raw);
    if (DSTATS) hs_load_dstats(s_st, io, blockIdx.y, sh.H);
    const HsStats& st = DSTATS ? s_st : st_param;
    constexpr int NF = n_frac(L);
    extern __shared__ float4 hs_tile_smem4[];
    float* sm = reinterpret_cast<float*>(hs_tile_smem4);
    __shared__ unsigned long long bar[2];
    constexpr int F5 = 9;                                   // first fraction of level 5
    const int s = blockIdx.y;
    const int N = (int)sh.n_bins, n_fund = (int)sh.n_fund;
    const int n0 = blockIdx.x * (TILE * W);
    const int b0 = blockIdx.x * (TILE * W / 32);            // n0 / 32: the span of fraction kk starts at element kk b0
    const float* x = io.x + (long long)s * sh.in_stride;                  // the row of x[n] itself (fraction 32/32)
    const int zq = s - sh.Z;                                                 // TWOD: z of this row
    auto frac_row = [&](int kk) -> const float* {                           // the row fraction kk/32 reads from
        return TWOD ? io.x + (long long)(((kk * zq + 16) >> 5) + sh.Z) * sh.in_stride : x;
    };
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (NF > F_SMEM) {
        if (threadIdx.x == 0) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" :: "r"(smem_u32(&bar[0])) : "memory");
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" :: "r"(smem_u32(&bar[1])) : "memory");
            asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        }
        __syncthreads();                                    // barrier initialised; the other warps go on to their own loads
        if (threadIdx.x == 0) {
            // A span is cut at the end of the row's allocation (in_stride is a multiple of 4 words, so the byte count
            // stays a multiple of 16): words beyond n_bins only ever feed outputs that do not exist.
            const long long lim = sh.in_stride;
            unsigned total[2] = {0, 0};
#pragma unroll
            for (int f = F_SMEM; f < NF; ++f) {
                const long long room = lim - (long long)frac_kk(f) * b0;
                total[(SPLIT && f >= F5) ? 1 : 0] += 4u * (unsigned)max(0ll, min((long long)span_words(frac_kk(f), W), room));
            }
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" :: "r"(smem_u32(&bar[0])), "r"(total[0]) : "memory");
            if (SPLIT && NF > F5)
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" :: "r"(smem_u32(&bar[1])), "r"(total[1]) : "memory");
#pragma unroll
            for (int f = F_SMEM; f < NF; ++f) {
                const int kk = frac_kk(f);
                const long long room = lim - (long long)kk * b0;
                const unsigned bytes = 4u * (unsigned)max(0ll, min((long long)span_words(kk, W), room));
                if (bytes)
                    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
                                 :: "r"(smem_u32(sm + span_off(f, W))), "l"(frac_row(kk) + kk * b0), "r"(bytes),
                                    "r"(smem_u32(&bar[(SPLIT && f >= F5) ? 1 : 0])) : "memory");
            }
        }
    }
    // lane i of warp pair w owns outputs nw + 16 i + [0, 16); this warp does the 8 that start at 8 half
    const int w = warp >> 1, half = warp & 1;
    const int nw = n0 + TILE * w;
    Direct d;
    load_direct<L>(d, x, frac_row(16), frac_row(8), N, nw + 16 * lane + 8 * half, nw / 2 + 8 * lane + 4 * half,
                   nw / 4 + 4 * lane + 2 * half, nw + TILE + 8 <= N, (reinterpret_cast<uintptr_t>(x) & 31u) == 0);
    if (NF > F_SMEM) mbar_wait(smem_u32(&bar[0]), 0);
    auto wait5 = [&]() { if (SPLIT && NF > F5) mbar_wait(smem_u32(&bar[1]), 0); };
    float best[8];
    int bh[8];
    if (half == 0) chain8<L, 0, W>(sm, st, w, lane, d, best, bh, wait5);
    else chain8<L, 8, W>(sm, st, w, lane, d, best, bh, wait5);
    const int n_out = nw + 16 * lane + 8 * half;
    const long long o = (long long)s * sh.out_stride + n_out;
    const bool oal32 = (((reinterpret_cast<uintptr_t>(io.snr + o)) | (reinterpret_cast<uintptr_t>(io.best_h + o))) & 31u) == 0;
    store8(io.snr + o, io.best_h + o, n_out, n_fund, nw + TILE <= n_fund, oal32, best, bh);
}
