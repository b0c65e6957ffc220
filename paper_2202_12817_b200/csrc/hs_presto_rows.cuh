// PRESTO-like harmonic sum (Alg. 1; eq. 4), "rows" kernel:
// every lane owns 16 CONSECUTIVE top bins, so that each term of eq. 4 is a compile-time offset
// into a short private row of shared memory that the lane reads with vector loads.
//
// Index algebra.  Alg. 1 visits x[Round(h n / H')] for H' = 1, 2, 4, .., Hq = 2^L and
// h in {1} U {2, 4, .., H'}.  Written in 32nds the fractions h/H' are kk/32 with
//     level 0: kk = 32            level 1: 16           level 2: 8           level 3: 4, 24
//     level 4: 2, 12, 20, 28      level 5: 1, 6, 10, 14, 18, 22, 26, 30
// (the harmonic sets are nested, hs_presto.cuh: S_{2H'} = S_{H'} + the terms of level log2(2H')),
// and Round is round-half-up in exact integers (reading R3):  idx = (kk n + 16) >> 5.
// For n = n0 + 16 i + e  (n0 a multiple of 512, lane i, e = 0..15):
//     idx = kk n0/32 + (kk/2) i + ((kk e + 16) >> 5)            (kk even)
//     idx = n0/32 + ((i + 1) >> 1)                              (kk = 1: one element for all e)
// so lane i reads the kk/2 + 1 elements that start at (kk/2) i of the span x[kk n0/32 ..], at offsets
// known when the kernel is compiled: 147 elements for its 16 outputs instead of 17 x 16 separate loads,
// fetched as LDS.128 / LDS.64 / LDS.32 according to the alignment (kk/2) i allows.
//
// Shared-memory layout of a CTA tile of T = 512 W outputs (W warps):
//   * 15 spans are copied as they are by one 1-D bulk async copy each (TMA engine, cp.async.bulk ->
//     UBLKCP): the lane stride kk/2 words makes their vector loads bank-conflict free;
//   * for kk = 32 and kk = 16 a lane stride of 16 / 8 words would serialise the 16-byte loads 4- / 2-fold,
//     so those two spans are stored as padded rows by coalesced 16-byte cp.async copies of the whole CTA:
//     kk = 16 with a pitch of 12 words (the 4 words of padding repeat the head of the next row), kk = 32 as
//     pairs of 16-word rows sharing one 16-byte pad (row32_off: conflict-free lane-major AND stream-major).
// The outputs of a lane are consecutive too; they go back through the warp's own kk = 32 rows
// (dead by then) so that the global stores are coalesced 16-byte streaming stores.
#pragma once
#include "hs_common.cuh"

namespace hs_rows {

constexpr int G = 16;                       // outputs per lane
constexpr int WT = 32 * G;                  // outputs per warp

// fraction table in enumeration order (level-major), L levels
__host__ __device__ constexpr int n_frac(int L) { return L == 0 ? 1 : L <= 2 ? L + 1 : L == 3 ? 5 : L == 4 ? 9 : 17; }
__host__ __device__ constexpr int frac_kk(int f) {
    constexpr int t[17] = {32, 16, 8, 4, 24, 2, 12, 20, 28, 1, 6, 10, 14, 18, 22, 26, 30};
    return t[f];
}
__host__ __device__ constexpr int frac_level(int f) { return f == 0 ? 0 : f == 1 ? 1 : f == 2 ? 2 : f <= 4 ? 3 : f <= 8 ? 4 : 5; }
__host__ __device__ constexpr bool frac_padded(int kk) { return kk == 32 || kk == 16; }
__host__ __device__ constexpr int pad_pitch(int kk) { return kk / 2 + 4; }
// kk = 32 (x[n] itself; its rows are also the transposition buffer of the output pass): row r holds exactly the 16
// words of lane r, two rows share 9 sixteen-byte units (8 of data + 1 of padding).  Both ways the rows are touched
// are then bank-conflict free: lane-major (lane i reads / writes unit c of row i: 9 (i >> 1) + 4 (i & 1) + c are
// distinct mod 8 over 8 lanes) and stream-major (consecutive lanes take consecutive units of the row pairs).
__host__ __device__ constexpr int row32_off(int r) { return 36 * (r >> 1) + 16 * (r & 1); }
// words of shared memory of one span of a CTA tile of W warps
__host__ __device__ constexpr int span_words(int kk, int W) {
    return kk == 32 ? 18 * 32 * W : frac_padded(kk) ? 32 * W * pad_pitch(kk) : 16 * kk * W + 4;
}
__host__ __device__ constexpr int span_off(int f, int W) {
    int o = 0;
    for (int g = 0; g < f; ++g) o += span_words(frac_kk(g), W);
    return o;
}
__host__ __device__ constexpr int smem_words(int L, int W) { return span_off(n_frac(L), W); }

// offset of output e in the row of fraction kk (kk even), and the range a group of 8 outputs spans
__host__ __device__ constexpr int row_off(int kk, int e) { return (kk * e + 16) >> 5; }

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

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
    constexpr int lo_al = lo & ~(A - 1);
    constexpr int nvec = (hi - lo_al) / A + 1;
    float t[nvec * A];
#pragma unroll
    for (int v = 0; v < nvec; ++v) {
        if (A == 4) {
            const float4 q = *reinterpret_cast<const float4*>(row + lo_al + 4 * v);
            t[4 * v] = q.x; t[4 * v + 1] = q.y; t[4 * v + 2] = q.z; t[4 * v + 3] = q.w;
        } else if (A == 2) {
            const float2 q = *reinterpret_cast<const float2*>(row + lo_al + 2 * v);
            t[2 * v] = q.x; t[2 * v + 1] = q.y;
        } else {
            t[v] = row[lo_al + v];
        }
    }
#pragma unroll
    for (int u = 0; u < NE; ++u) {
        const float v = t[row_off(KK, E0 + u) - lo_al];
        acc[u] = FIRST ? v : __fadd_rn(acc[u], v);
    }
}


// guarded staging of words [g, g + len) of the row into sm (zero beyond the end of the row)
template <int BLOCK>
__device__ __forceinline__ void stage_guarded(float* __restrict__ sm, const float* __restrict__ x, int g, int len4, int N) {
    float4* dst = reinterpret_cast<float4*>(sm);
#pragma unroll 1
    for (int i = threadIdx.x; i < len4; i += BLOCK) {
        const int e = g + 4 * i;
        float4 v;
        if (e + 3 < N) {
            v = __ldg(reinterpret_cast<const float4*>(x + e));
        } else {
            v.x = (e < N) ? __ldg(x + e) : 0.f;
            v.y = (e + 1 < N) ? __ldg(x + e + 1) : 0.f;
            v.z = (e + 2 < N) ? __ldg(x + e + 2) : 0.f;
            v.w = (e + 3 < N) ? __ldg(x + e + 3) : 0.f;
        }
        dst[i] = v;
    }
}

// padded rows of fraction KK (32 or 16): row r = x[g + RL r .. g + RL r + RL + 4), RL = KK/2, pitch RL + 4.
// Thread t copies float4 number t + j BLOCK of the span, j = 0 .. RL/4 - 1 (coalesced); a float4 that
// starts a row is also the 4-word tail of the row before.  INTERIOR: the span ends inside the spectrum and
// the copies are 16-byte cp.async (LDGSTS: no register round trip, waited for once by the caller).
template <int BLOCK, int KK, int W, bool INTERIOR>
__device__ __forceinline__ void stage_padded(float* __restrict__ sm, const float* __restrict__ x, int g, int N) {
    constexpr int RL = KK / 2, P = RL + 4, ROWS = 32 * W, Q = ROWS * RL / 4;      // float4s of the span proper
    static_assert(Q % BLOCK == 0, "span shape");
#pragma unroll
    for (int j = 0; j <= Q / BLOCK; ++j) {
        const int q = threadIdx.x + j * BLOCK;
        if (j == Q / BLOCK && threadIdx.x != 0) break;                 // float4 number Q: only the last row's tail
        const int e = g + 4 * q;
        const int r = (4 * q) / RL, col = (4 * q) % RL;
        if (INTERIOR) {
            if (r < ROWS)
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" :: "r"(smem_u32(sm + r * P + col)), "l"(x + e) : "memory");
            if (col == 0 && r >= 1)
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" :: "r"(smem_u32(sm + (r - 1) * P + RL)), "l"(x + e) : "memory");
        } else {
            float4 v;
            v.x = (e < N) ? __ldg(x + e) : 0.f;
            v.y = (e + 1 < N) ? __ldg(x + e + 1) : 0.f;
            v.z = (e + 2 < N) ? __ldg(x + e + 2) : 0.f;
            v.w = (e + 3 < N) ? __ldg(x + e + 3) : 0.f;
            if (r < ROWS) *reinterpret_cast<float4*>(sm + r * P + col) = v;
            if (col == 0 && r >= 1) *reinterpret_cast<float4*>(sm + (r - 1) * P + RL) = v;
        }
    }
}

// The same for a span that ends inside the spectrum, with the per-thread address arithmetic done once:
// float4 number q = t + j BLOCK lands at word (q / F4) P + 4 (q % F4), F4 = RL/4 float4s per row; BLOCK is a
// multiple of F4, so q % F4 = t % F4 for every j and the destination advances by (BLOCK / F4) P words per j.
template <int BLOCK, int KK, int W>
__device__ __forceinline__ void stage_padded_interior(float* __restrict__ sm, const float* __restrict__ src_span) {
    constexpr int RL = KK / 2, P = RL + 4, F4 = RL / 4, ROWS = 32 * W, Q = ROWS * F4, NJ = Q / BLOCK;
    static_assert(Q % BLOCK == 0 && BLOCK % F4 == 0, "span shape");
    const int t = threadIdx.x;
    const unsigned dst = smem_u32(sm + (t / F4) * P + 4 * (t % F4));
    const float* src = src_span + 4 * t;
    const bool head = (t % F4) == 0;                                   // this float4 starts a row
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" :: "r"(dst + 4u * (j * (BLOCK / F4) * P)), "l"(src + 4 * j * BLOCK) : "memory");
        if (head && (j > 0 || t > 0))                                  // ... and is the tail of the row before
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" :: "r"(dst + 4u * (j * (BLOCK / F4) * P) - 16u), "l"(src + 4 * j * BLOCK) : "memory");
    }
    if (t == 0)                                                        // the tail of the last row
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" :: "r"(dst + 4u * (ROWS * P) - 16u), "l"(src + 4 * Q) : "memory");
}

// kk = 32 rows (row32_off layout) of a tile of W warps: float4 number q of the span x[g ..] is unit q & 3 of row q >> 2
template <int BLOCK, int W, bool INTERIOR>
__device__ __forceinline__ void stage_x32(float* __restrict__ sm, const float* __restrict__ x, int g, int N) {
    constexpr int Q = 32 * W * 4, NJ = Q / BLOCK;
    static_assert(Q % BLOCK == 0 && BLOCK % 8 == 0, "span shape");
    const int t = threadIdx.x;
    float* d0 = sm + row32_off(t >> 2) + 4 * (t & 3);             // + 36 BLOCK / 8 words per j
    if (INTERIOR) {
        const unsigned dst = smem_u32(d0);
        const float* src = x + g + 4 * t;
#pragma unroll
        for (int j = 0; j < NJ; ++j)
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" :: "r"(dst + 4u * (j * (36 * BLOCK / 8))), "l"(src + 4 * j * BLOCK) : "memory");
    } else {
#pragma unroll
        for (int j = 0; j < NJ; ++j) {
            const int e = g + 4 * (t + j * BLOCK);
            float4 v;
            v.x = (e < N) ? __ldg(x + e) : 0.f;
            v.y = (e + 1 < N) ? __ldg(x + e + 1) : 0.f;
            v.z = (e + 2 < N) ? __ldg(x + e + 2) : 0.f;
            v.w = (e + 3 < N) ? __ldg(x + e + 3) : 0.f;
            *reinterpret_cast<float4*>(d0 + j * (36 * BLOCK / 8)) = v;
        }
    }
}

// start of lane `lane` of warp `w`'s row in the span of fraction F
template <int F, int W>
__device__ __forceinline__ const float* row_ptr(const float* __restrict__ sm, int w, int lane) {
    constexpr int kk = frac_kk(F);
    if (kk == 32) return sm + span_off(F, W) + row32_off(32 * w + lane);
    if (frac_padded(kk)) return sm + span_off(F, W) + (32 * w + lane) * pad_pitch(kk);
    if (kk == 1) return sm + span_off(F, W) + 16 * w + ((lane + 1) >> 1);
    return sm + span_off(F, W) + 16 * kk * w + (kk / 2) * lane;
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

// outputs e = E0 + u, u < NE, of the lane: all levels
template <int L, int W, int E0, int NE>
__device__ __forceinline__ void level_chain(const float* __restrict__ sm, const HsStats& st, int w, int lane,
                                            float (&res_snr)[G], int (&res_bh)[G]) {
    float S[NE], best[NE], add[NE];
    int bh[NE];
    add_terms<32, E0, NE, true>(row_ptr<0, W>(sm, w, lane), S);             // H' = 1: x[n]
#pragma unroll
    for (int u = 0; u < NE; ++u) { best[u] = hs_snr(S[u], st.nmis[0], st.inv_sigma[0]); bh[u] = 1; }
    if (L >= 1) {
        add_terms<16, E0, NE, true>(row_ptr<1, W>(sm, w, lane), add);
        close_level<2, NE>(st, S, add, best, bh);
    }
    if (L >= 2) {
        add_terms<8, E0, NE, true>(row_ptr<2, W>(sm, w, lane), add);
        close_level<4, NE>(st, S, add, best, bh);
    }
    if (L >= 3) {
        add_terms<4, E0, NE, true>(row_ptr<3, W>(sm, w, lane), add);
        add_terms<24, E0, NE, false>(row_ptr<4, W>(sm, w, lane), add);
        close_level<8, NE>(st, S, add, best, bh);
    }
    if (L >= 4) {
        add_terms<2, E0, NE, true>(row_ptr<5, W>(sm, w, lane), add);
        add_terms<12, E0, NE, false>(row_ptr<6, W>(sm, w, lane), add);
        add_terms<20, E0, NE, false>(row_ptr<7, W>(sm, w, lane), add);
        add_terms<28, E0, NE, false>(row_ptr<8, W>(sm, w, lane), add);
        close_level<16, NE>(st, S, add, best, bh);
    }
    if (L >= 5) {
        add_terms<1, E0, NE, true>(row_ptr<9, W>(sm, w, lane), add);
        add_terms<6, E0, NE, false>(row_ptr<10, W>(sm, w, lane), add);
        add_terms<10, E0, NE, false>(row_ptr<11, W>(sm, w, lane), add);
        add_terms<14, E0, NE, false>(row_ptr<12, W>(sm, w, lane), add);
        add_terms<18, E0, NE, false>(row_ptr<13, W>(sm, w, lane), add);
        add_terms<22, E0, NE, false>(row_ptr<14, W>(sm, w, lane), add);
        add_terms<26, E0, NE, false>(row_ptr<15, W>(sm, w, lane), add);
        add_terms<30, E0, NE, false>(row_ptr<16, W>(sm, w, lane), add);
        close_level<32, NE>(st, S, add, best, bh);
    }
#pragma unroll
    for (int u = 0; u < NE; ++u) { res_snr[E0 + u] = best[u]; res_bh[E0 + u] = bh[u]; }
}

}  // namespace hs_rows

// NE = 16 / 8: a warp does the 16 outputs of its lanes at once / as two groups of 8.
// NE = -8 ("pair"): TWO warps share a 512-output tile, one takes outputs e < 8 of every lane's 16, the
// other e >= 8: twice the warps for the same shared memory (the kernel's occupancy is set by shared memory).
template <int L, int W, bool BULK, int NE>
__global__ void __launch_bounds__(NE < 0 ? 64 * W : 32 * W, 12 / W)
hs_presto_rows_kernel(const __grid_constant__ HsShape sh, const __grid_constant__ HsStats st, HsIO io) {
    using namespace hs_rows;
    constexpr bool PAIR = NE < 0;
    constexpr int BLOCK = PAIR ? 64 * W : 32 * W;
    constexpr int T = WT * W;                           // outputs per CTA
    constexpr int NF = n_frac(L);
    extern __shared__ float4 hs_rows_smem4[];
    float* sm = reinterpret_cast<float*>(hs_rows_smem4);
    __shared__ unsigned long long bar;

    const int s = blockIdx.y;
    const int N = (int)sh.n_bins;
    const int n_fund = (int)sh.n_fund;
    const int n0 = blockIdx.x * T;
    const int b0 = blockIdx.x * (T / 32);               // n0 / 32: span of fraction kk starts at element kk b0
    const float* x = io.x + (long long)s * sh.in_stride;
    asm volatile("" : "+l"(x));                                  // one materialised row pointer for all the copies

    // ---- stage ----
    const bool interior = BULK && (n0 + T + 4 <= N);    // every span (the longest is kk = 32) ends inside the row
    if (interior) {
        if (threadIdx.x == 0) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" :: "r"(smem_u32(&bar)) : "memory");
            asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
            unsigned total = 0;
#pragma unroll
            for (int f = 0; f < NF; ++f) if (!frac_padded(frac_kk(f))) total += 4u * span_words(frac_kk(f), W);
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" :: "r"(smem_u32(&bar)), "r"(total) : "memory");
#pragma unroll
            for (int f = 0; f < NF; ++f) {
                constexpr int dummy = 0; (void)dummy;
                const int kk = frac_kk(f);
                if (!frac_padded(kk)) {
                    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
                                 :: "r"(smem_u32(sm + span_off(f, W))), "l"(x + kk * b0), "r"(4u * span_words(kk, W)),
                                    "r"(smem_u32(&bar)) : "memory");
                }
            }
        }
    } else {
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            const int kk = frac_kk(f);
            if (!frac_padded(kk)) stage_guarded<BLOCK>(sm + span_off(f, W), x, kk * b0, span_words(kk, W) / 4, N);
        }
    }
    if (interior) {
        stage_x32<BLOCK, W, true>(sm + span_off(0, W), x, 32 * b0, N);
        if (L >= 1) stage_padded_interior<BLOCK, 16, W>(sm + span_off(1, W), x + 16 * b0);
        asm volatile("cp.async.commit_group;\n cp.async.wait_group 0;\n" ::: "memory");
    } else {
        stage_x32<BLOCK, W, false>(sm + span_off(0, W), x, 32 * b0, N);
        if (L >= 1) stage_padded<BLOCK, 16, W, false>(sm + span_off(1, W), x, 16 * b0, N);
    }
    __syncthreads();
    if (interior) {
        unsigned done = 0;
        while (!done) {
            asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n selp.u32 %0, 1, 0, p;\n}\n"
                         : "=r"(done) : "r"(smem_u32(&bar)) : "memory");
        }
    }

    // ---- compute: lane i of warp w owns outputs n0 + 512 w + 16 i + [0, 16) ----
    const int lane = threadIdx.x & 31;
    const int w = PAIR ? (threadIdx.x >> 6) : (threadIdx.x >> 5);
    const int half = PAIR ? ((threadIdx.x >> 5) & 1) : 0;
    float res_snr[G];
    int res_bh[G];
    if (PAIR) {
        if (half == 0) {
            level_chain<L, W, 0, 8>(sm, st, w, lane, res_snr, res_bh);
        } else {
            level_chain<L, W, 8, 8>(sm, st, w, lane, res_snr, res_bh);
#pragma unroll
            for (int u = 0; u < 8; ++u) { res_snr[u] = res_snr[8 + u]; res_bh[u] = res_bh[8 + u]; }   // registers 0..7 either way
        }
    } else if (NE == 16) {
        level_chain<L, W, 0, 16>(sm, st, w, lane, res_snr, res_bh);
    } else {
        level_chain<L, W, 0, 8>(sm, st, w, lane, res_snr, res_bh);
        level_chain<L, W, 8, 8>(sm, st, w, lane, res_snr, res_bh);
    }

    // ---- store: transpose through the tile's own kk = 32 rows (32 rows x pitch 20, no longer read) ----
    float* stg = sm + span_off(0, W) + row32_off(32 * w);
    int* stgi = reinterpret_cast<int*>(stg);
    const long long orow = (long long)s * sh.out_stride;
    const int nw = n0 + WT * w;
    constexpr int V0 = 0, NV = PAIR ? 2 : 4;            // float4s of a row this warp writes / stream quarters it reads
    const int vbase = PAIR ? 2 * half : V0;
    auto sync_tile = [&]() { if (PAIR) __syncthreads(); else __syncwarp(); };
    const bool full = n0 + T <= n_fund;                   // every output of the tile exists: no per-store checks
    sync_tile();
#pragma unroll
    for (int v = 0; v < NV; ++v) {
        const int col = PAIR ? 8 * half + 4 * v : 4 * v;
        *reinterpret_cast<float4*>(stg + row32_off(lane) + col) =
            make_float4(res_snr[4 * v], res_snr[4 * v + 1], res_snr[4 * v + 2], res_snr[4 * v + 3]);
    }
    sync_tile();
    // float4 number q = lane + 32 (vbase + k) of the tile's output stream sits at row q / 4, words 4 (q % 4) ..
    const float* rd = stg + row32_off((lane >> 2) + 8 * vbase) + 4 * (lane & 3);   // + 8 rows = 144 words per k
    const long long o0 = orow + nw + 4 * (lane + 32 * vbase);
    if (full) {
#pragma unroll
        for (int k = 0; k < NV; ++k)
            __stcs(reinterpret_cast<float4*>(io.snr + o0 + 128 * k), *reinterpret_cast<const float4*>(rd + 144 * k));
    } else {
#pragma unroll
        for (int k = 0; k < NV; ++k) {
            const float4 v = *reinterpret_cast<const float4*>(rd + 144 * k);
            const int n = nw + 4 * (lane + 32 * (vbase + k));
            if (n + 3 < n_fund) {
                __stcs(reinterpret_cast<float4*>(io.snr + orow + n), v);
            } else {
                if (n < n_fund) st_cs(io.snr + orow + n, v.x);
                if (n + 1 < n_fund) st_cs(io.snr + orow + n + 1, v.y);
                if (n + 2 < n_fund) st_cs(io.snr + orow + n + 2, v.z);
            }
        }
    }
    sync_tile();
#pragma unroll
    for (int v = 0; v < NV; ++v) {
        const int col = PAIR ? 8 * half + 4 * v : 4 * v;
        *reinterpret_cast<int4*>(stgi + row32_off(lane) + col) =
            make_int4(res_bh[4 * v], res_bh[4 * v + 1], res_bh[4 * v + 2], res_bh[4 * v + 3]);
    }
    sync_tile();
    const int* rdi = reinterpret_cast<const int*>(rd);
    if (full) {
#pragma unroll
        for (int k = 0; k < NV; ++k)
            __stcs(reinterpret_cast<int4*>(io.best_h + o0 + 128 * k), *reinterpret_cast<const int4*>(rdi + 144 * k));
    } else {
#pragma unroll
        for (int k = 0; k < NV; ++k) {
            const int4 v = *reinterpret_cast<const int4*>(rdi + 144 * k);
            const int n = nw + 4 * (lane + 32 * (vbase + k));
            if (n + 3 < n_fund) {
                __stcs(reinterpret_cast<int4*>(io.best_h + orow + n), v);
            } else {
                if (n < n_fund) st_cs(io.best_h + orow + n, v.x);
                if (n + 1 < n_fund) st_cs(io.best_h + orow + n + 1, v.y);
                if (n + 2 < n_fund) st_cs(io.best_h + orow + n + 2, v.z);
            }
        }
    }
}
