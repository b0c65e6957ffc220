// Tuned PRESTO-like harmonic sum (Alg. 1; eq. 4) for the common
// configuration: fundamental + even harmonics, H' in powers of two, no per-bin baseline,
// h n < 2^31.
//
// Every fraction h/H' that Alg. 1 visits for H' <= Hq = 2^LOG2H is k/Hq with
// k in {1, 2, 4, 6, 8, ..., Hq}: the harmonic sets are nested,
//     HARM(2H') scaled = 2*HARM(H')  U  {1} U {6, 10, 14, ..., 2H'-2},
// so one output needs Hq/2 + 1 gathers instead of the sum over H' of (1 + H'/2), and the
// partial sums are built incrementally, S_{2H'} = S_{H'} + (new terms).  Round(h n/H') is the
// exact integer (h n + H'/2) >> log2 H' (round half up, R3).
// Consecutive outputs read the same or the adjacent element (a compressing gather), so a warp of
// 32 consecutive n touches k/Hq*32 + 1 consecutive floats per fraction: coalesced by construction.
#pragma once
#include "hs_common.cuh"

template <int LOG2H>
__device__ __forceinline__ void hs_presto_one(const float* __restrict__ x, const HsStats& st, int n,
                                              float& best, int& bh) {
    // level 0: H' = 1
    float S = __ldg(x + n);
    best = hs_snr(S, st.nmis[0], st.inv_sigma[0]);
    bh = 1;
#pragma unroll
    for (int L = 1; L <= LOG2H; ++L) {
        const int Hp = 1 << L;
        const int half = Hp >> 1;
        // new fundamental term h = 1
        float add = __ldg(x + ((n + half) >> L));
        // new even harmonics h = 6, 10, ..., Hp - 2 (h = 2 mod 4; none for Hp < 8)
#pragma unroll
        for (int h = 6; h < Hp; h += 4) add = __fadd_rn(add, __ldg(x + ((h * n + half) >> L)));
        S = __fadd_rn(S, add);
        const float snr = hs_snr(S, st.nmis[Hp - 1], st.inv_sigma[Hp - 1]);
        if (snr > best) { best = snr; bh = Hp; }
    }
}

template <int BLOCK, int R, int LOG2H>
__global__ void __launch_bounds__(BLOCK)
hs_presto_tile_kernel(const __grid_constant__ HsShape sh, const __grid_constant__ HsStats st, HsIO io) {
    const int s = blockIdx.y;
    const int n_fund = (int)sh.n_fund;
    const int f0 = blockIdx.x * (BLOCK * R);
    const float* __restrict__ x = io.x + (long long)s * sh.in_stride;
    const long long orow = (long long)s * sh.out_stride;
#pragma unroll
    for (int j = 0; j < R; ++j) {
        const int n = f0 + j * BLOCK + threadIdx.x;
        if (n < n_fund) {
            float best; int bh;
            hs_presto_one<LOG2H>(x, st, n, best, bh);
            st_cs(io.snr + orow + n, best);
            st_cs(io.best_h + orow + n, bh);
        }
    }
}
