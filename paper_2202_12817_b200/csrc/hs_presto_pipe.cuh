// PRESTO-like harmonic sum (Alg. 1; eq. 4), persistent pipelined
// form of the "rows" kernel (hs_presto_rows.cuh: same index algebra, same shared-memory rows, same
// arithmetic and order of additions).
//
// Why: staging moves 8.5 words per output from L2 into shared memory (34 B/bin, 36.5 GB per launch on
// cfg3), which is 2 ms at the ~18 TB/s the L2->SM path delivers (profiles/r01b_machine_model.md),
// about as long as the arithmetic and as the HBM traffic.  In the one-shot kernel a tile's buffer
// waits for its copies, then computes, then stores: the three do not overlap inside a tile and
// shared memory is too small to hold enough tiles in both states at once (the copies in flight must
// cover bandwidth x latency ~ 100 KB per SM).
//
// Here every WARP is its own pipeline over a strided sequence of 512-output tiles, with the spans of
// a tile split in two buffers of similar size:
//     buffer A = levels 0..4 (kk = 32, 16, 8, 4, 24, 2, 12, 20, 28),   buffer B = level 5 (kk = 1, 6, .., 30).
//     wait A(t) | levels 0..4 of tile t | issue A(t+1) | wait B(t) | level 5 of tile t |
//     transpose + store tile t through B | issue B(t+1) | ...
// so the copies of one buffer are always in flight while the warp computes out of the other: half
// of shared memory is being filled at any time and no warp waits with nothing to do.  Warps share
// nothing: there is no block-wide barrier in the loop, only the two mbarriers of the warp
// (1-D bulk async copies, TMA engine) and its cp.async group (padded rows of kk = 32, 16).
#pragma once
#include "hs_presto_rows.cuh"

namespace hs_pipe {
using namespace hs_rows;

__host__ __device__ constexpr int nf_a(int L) { return n_frac(L < 4 ? L : 4); }          // fractions in buffer A
__host__ __device__ constexpr int words_a(int L) { return span_off(nf_a(L), 1); }
__host__ __device__ constexpr int words_b(int L) { return L >= 5 ? span_off(17, 1) - span_off(9, 1) : 0; }
// a warp's region: A then B; B also serves as the transposition buffer (32 rows x pitch 20 = 640 words)
__host__ __device__ constexpr int words_warp(int L) { return words_a(L) + (words_b(L) > 640 ? words_b(L) : 640); }

__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    unsigned done = 0;
    while (!done) {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
                     : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    }
}

// copies of fractions [F0, F1) of the tile whose spans start at element kk b0 (interior tile).
// lane f - F0 issues the bulk copy of fraction f; padded fractions go by cp.async from all lanes.
template <int F0, int F1>
__device__ __forceinline__ void issue_bulk(float* __restrict__ smw, int sm_shift, const float* __restrict__ x, int b0,
                                           unsigned long long* bar, int lane) {
    // sm_shift: words to subtract from span_off (buffer B starts at span_off(9, 1))
    if (lane == 0) {
        unsigned total = 0;
#pragma unroll
        for (int f = F0; f < F1; ++f) if (!frac_padded(frac_kk(f))) total += 4u * span_words(frac_kk(f), 1);
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" :: "r"(smem_u32(bar)), "r"(total) : "memory");
    }
    __syncwarp();
#pragma unroll
    for (int f = F0; f < F1; ++f) {
        const int kk = frac_kk(f);
        if (!frac_padded(kk) && lane == f - F0) {
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
                         :: "r"(smem_u32(smw + span_off(f, 1) - sm_shift)), "l"(x + kk * b0), "r"(4u * span_words(kk, 1)),
                            "r"(smem_u32(bar)) : "memory");
        }
    }
}

// guarded fill of fractions [F0, F1) by the warp (edge tile)
template <int F0, int F1>
__device__ __forceinline__ void fill_guarded(float* __restrict__ smw, int sm_shift, const float* __restrict__ x, int b0,
                                             int N, int lane) {
#pragma unroll
    for (int f = F0; f < F1; ++f) {
        const int kk = frac_kk(f);
        if (frac_padded(kk)) continue;
        float* dst = smw + span_off(f, 1) - sm_shift;
        const int g = kk * b0, len = span_words(kk, 1);
#pragma unroll 1
        for (int i = lane; i < len; i += 32) dst[i] = (g + i < N) ? __ldg(x + g + i) : 0.f;
    }
}

// padded rows of KK = 32 / 16 for a one-warp tile: 32 rows, see hs_rows::stage_padded
template <int KK, bool INTERIOR>
__device__ __forceinline__ void fill_padded(float* __restrict__ dst, const float* __restrict__ x, int g, int N, int lane) {
    constexpr int RL = KK / 2, P = RL + 4, Q = 32 * RL / 4;
#pragma unroll
    for (int j = 0; j <= Q / 32; ++j) {
        const int q = lane + 32 * j;
        if (j == Q / 32 && lane != 0) break;
        const int e = g + 4 * q;
        const int r = (4 * q) / RL, col = (4 * q) % RL;
        if (INTERIOR) {
            if (r < 32)
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" :: "r"(smem_u32(dst + r * P + col)), "l"(x + e) : "memory");
            if (col == 0 && r >= 1)
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" :: "r"(smem_u32(dst + (r - 1) * P + RL)), "l"(x + e) : "memory");
        } else {
            float4 v;
            v.x = (e < N) ? __ldg(x + e) : 0.f;
            v.y = (e + 1 < N) ? __ldg(x + e + 1) : 0.f;
            v.z = (e + 2 < N) ? __ldg(x + e + 2) : 0.f;
            v.w = (e + 3 < N) ? __ldg(x + e + 3) : 0.f;
            if (r < 32) *reinterpret_cast<float4*>(dst + r * P + col) = v;
            if (col == 0 && r >= 1) *reinterpret_cast<float4*>(dst + (r - 1) * P + RL) = v;
        }
    }
}

// row of lane `lane` in fraction F of a one-warp tile whose region starts at smw (+ shift for buffer B)
template <int F>
__device__ __forceinline__ const float* rowp(const float* __restrict__ smw, int sm_shift, int lane) {
    constexpr int kk = frac_kk(F);
    if (frac_padded(kk)) return smw + span_off(F, 1) - sm_shift + lane * pad_pitch(kk);
    if (kk == 1) return smw + span_off(F, 1) - sm_shift + ((lane + 1) >> 1);
    return smw + span_off(F, 1) - sm_shift + (kk / 2) * lane;
}

}  // namespace hs_pipe

namespace hs_pipe {

// levels 0 .. min(L, 4) for the 16 outputs of the lane (buffer A)
template <int L>
__device__ __forceinline__ void levels_a(const float* __restrict__ smw, const HsStats& st, int lane, float (&S)[G],
                                         float (&best)[G], int (&bh)[G]) {
    float add[G];
    add_terms<32, 0, G, true>(rowp<0>(smw, 0, lane), S);                  // H' = 1: x[n]
#pragma unroll
    for (int u = 0; u < G; ++u) { best[u] = hs_snr(S[u], st.nmis[0], st.inv_sigma[0]); bh[u] = 1; }
    if (L >= 1) {
        add_terms<16, 0, G, true>(rowp<1>(smw, 0, lane), add);
        close_level<2, G>(st, S, add, best, bh);
    }
    if (L >= 2) {
        add_terms<8, 0, G, true>(rowp<2>(smw, 0, lane), add);
        close_level<4, G>(st, S, add, best, bh);
    }
    if (L >= 3) {
        add_terms<4, 0, G, true>(rowp<3>(smw, 0, lane), add);
        add_terms<24, 0, G, false>(rowp<4>(smw, 0, lane), add);
        close_level<8, G>(st, S, add, best, bh);
    }
    if (L >= 4) {
        add_terms<2, 0, G, true>(rowp<5>(smw, 0, lane), add);
        add_terms<12, 0, G, false>(rowp<6>(smw, 0, lane), add);
        add_terms<20, 0, G, false>(rowp<7>(smw, 0, lane), add);
        add_terms<28, 0, G, false>(rowp<8>(smw, 0, lane), add);
        close_level<16, G>(st, S, add, best, bh);
    }
}

// level 5 (buffer B)
__device__ __forceinline__ void level_b(const float* __restrict__ smw, const HsStats& st, int lane, float (&S)[G],
                                        float (&best)[G], int (&bh)[G]) {
    float add[G];
    add_terms<1, 0, G, true>(rowp<9>(smw, 0, lane), add);
    add_terms<6, 0, G, false>(rowp<10>(smw, 0, lane), add);
    add_terms<10, 0, G, false>(rowp<11>(smw, 0, lane), add);
    add_terms<14, 0, G, false>(rowp<12>(smw, 0, lane), add);
    add_terms<18, 0, G, false>(rowp<13>(smw, 0, lane), add);
    add_terms<22, 0, G, false>(rowp<14>(smw, 0, lane), add);
    add_terms<26, 0, G, false>(rowp<15>(smw, 0, lane), add);
    add_terms<30, 0, G, false>(rowp<16>(smw, 0, lane), add);
    close_level<32, G>(st, S, add, best, bh);
}

// the lane's 16 consecutive outputs -> coalesced 16-byte streaming stores, through 32 rows x pitch 20 of stg
template <typename T4, typename T>
__device__ __forceinline__ void store_rows(T* __restrict__ stg, const T (&res)[G], T* __restrict__ out, int nw, int n_fund,
                                           int lane) {
    constexpr int P = pad_pitch(32);
#pragma unroll
    for (int v = 0; v < G / 4; ++v) {
        T4 q; q.x = res[4 * v]; q.y = res[4 * v + 1]; q.z = res[4 * v + 2]; q.w = res[4 * v + 3];
        *reinterpret_cast<T4*>(stg + lane * P + 4 * v) = q;
    }
    __syncwarp();
#pragma unroll
    for (int k = 0; k < G / 4; ++k) {
        const int q = lane + 32 * k;                                  // float4 index in the warp's output stream
        const T4 v = *reinterpret_cast<const T4*>(stg + (q >> 2) * P + 4 * (q & 3));
        const int n = nw + 4 * q;
        if (n + 3 < n_fund) {
            __stcs(reinterpret_cast<T4*>(out + n), v);
        } else {
            if (n < n_fund) st_cs(out + n, v.x);
            if (n + 1 < n_fund) st_cs(out + n + 1, v.y);
            if (n + 2 < n_fund) st_cs(out + n + 2, v.z);
        }
    }
    __syncwarp();
}

}  // namespace hs_pipe

// grid = persistent CTAs of NWARP independent warps; total_tiles = spectra * tiles_per_row, tile = 512 outputs
template <int L, int NWARP>
__global__ void __launch_bounds__(32 * NWARP, 12 / NWARP)
hs_presto_pipe_kernel(const __grid_constant__ HsShape sh, const __grid_constant__ HsStats st, HsIO io, int tiles_per_row,
                      int total_tiles) {
    using namespace hs_pipe;
    constexpr int NFA = nf_a(L);
    constexpr bool HAS_B = L >= 5;
    extern __shared__ float4 hs_pipe_smem4[];
    __shared__ unsigned long long bars[2 * NWARP];
    const int lane = threadIdx.x & 31;
    const int w = threadIdx.x >> 5;
    float* smw = reinterpret_cast<float*>(hs_pipe_smem4) + w * smem_words(L, 1);
    unsigned long long* barA = &bars[2 * w];
    unsigned long long* barB = &bars[2 * w + 1];
    const int N = (int)sh.n_bins;
    const int n_fund = (int)sh.n_fund;
    const int stride = gridDim.x * NWARP;
    int t = blockIdx.x * NWARP + w;
    if (t >= total_tiles) return;
    if (lane == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" :: "r"(smem_u32(barA)) : "memory");
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" :: "r"(smem_u32(barB)) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncwarp();

    // issue the copies of buffer A / B of tile tt; returns whether they are asynchronous (interior tile)
    auto issue_a = [&](int tt) -> bool {
        const int s = tt / tiles_per_row, j = tt - s * tiles_per_row;
        const float* __restrict__ x = io.x + (long long)s * sh.in_stride;
        const int b0 = 16 * j;
        const bool interior = 512 * j + 512 + 4 <= N;
        if (interior) {
            issue_bulk<0, NFA>(smw, 0, x, b0, barA, lane);
            fill_padded<32, true>(smw + span_off(0, 1), x, 32 * b0, N, lane);
            if (L >= 1) fill_padded<16, true>(smw + span_off(1, 1), x, 16 * b0, N, lane);
            asm volatile("cp.async.commit_group;\n" ::: "memory");
        } else {
            fill_guarded<0, NFA>(smw, 0, x, b0, N, lane);
            fill_padded<32, false>(smw + span_off(0, 1), x, 32 * b0, N, lane);
            if (L >= 1) fill_padded<16, false>(smw + span_off(1, 1), x, 16 * b0, N, lane);
            __syncwarp();
        }
        return interior;
    };
    auto issue_b = [&](int tt) {
        const int s = tt / tiles_per_row, j = tt - s * tiles_per_row;
        const float* __restrict__ x = io.x + (long long)s * sh.in_stride;
        if (512 * j + 512 + 4 <= N) issue_bulk<9, 17>(smw, 0, x, 16 * j, barB, lane);
        else { fill_guarded<9, 17>(smw, 0, x, 16 * j, N, lane); __syncwarp(); }
    };

    unsigned pa = 0, pb = 0;
    bool async = issue_a(t);
    if (HAS_B) issue_b(t);
    while (true) {
        const int s = t / tiles_per_row, j = t - s * tiles_per_row;
        const long long orow = (long long)s * sh.out_stride;
        const int nw = 512 * j;
        float S[G], best[G];
        int bh[G];
        // ---- buffer A ----
        if (async) {
            asm volatile("cp.async.wait_group 0;\n" ::: "memory");
            mbar_wait(barA, pa); pa ^= 1u;
        }
        __syncwarp();
        levels_a<L>(smw, st, lane, S, best, bh);
        const int tn = t + stride;
        const bool has_next = tn < total_tiles;
        const bool async_cur = async;
        if (HAS_B) {
            __syncwarp();                                           // every lane is done with buffer A
            asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
            if (has_next) async = issue_a(tn);
            // ---- buffer B ----
            if (async_cur) { mbar_wait(barB, pb); pb ^= 1u; }
            level_b(smw, st, lane, S, best, bh);
            __syncwarp();                                           // every lane is done with buffer B
            float* stg = smw + span_off(9, 1);
            store_rows<float4, float>(stg, best, io.snr + orow, nw, n_fund, lane);
            store_rows<int4, int>(reinterpret_cast<int*>(stg), bh, io.best_h + orow, nw, n_fund, lane);
            asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
            if (has_next) issue_b(tn);
        } else {
            __syncwarp();
            float* stg = smw + span_off(0, 1);                      // the kk = 32 rows, no longer read
            store_rows<float4, float>(stg, best, io.snr + orow, nw, n_fund, lane);
            store_rows<int4, int>(reinterpret_cast<int*>(stg), bh, io.best_h + orow, nw, n_fund, lane);
            asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
            if (has_next) async = issue_a(tn);
        }
        if (!has_next) break;
        t = tn;
    }
}
