// Generic kernels: every flag combination, optional per-bin baseline, any H <= 32, 64-bit index
// arithmetic.  One thread per output bin, consecutive threads consecutive bins (the paper's own
// mapping).  These are the coverage path; the tuned kernels for the common
// configurations live in hs_greedy.cuh / hs_presto.cuh.
#pragma once
#include "hs_common.cuh"

template <bool HAS_BASE>
__device__ __forceinline__ float hs_load(const float* __restrict__ x, const float* __restrict__ ib, long long m) {
    float v = __ldg(x + m);
    if (HAS_BASE) v = __fmul_rn(v, __ldg(ib + m));   // whitening multiplier (NEXT-2), one fp32 multiply
    return v;
}

// Alg. 2, eq. 5.
template <bool HAS_BASE, bool DSTATS = false>
__global__ void __launch_bounds__(256)
hs_greedy_generic_kernel(const __grid_constant__ HsShape sh, const __grid_constant__ HsStats st_param, HsIO io) {
    const int s = blockIdx.y;
    __shared__ HsStats s_st;
    if (DSTATS) hs_load_dstats(s_st, io, s, sh.H);
    const HsStats& st = DSTATS ? s_st : st_param;
    const long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= sh.n_fund) return;
    const float* __restrict__ x = io.x + (long long)s * sh.in_stride;
    const float* __restrict__ ib = HAS_BASE ? io.inv_base + (long long)s * sh.in_stride : nullptr;
    const long long last = sh.n_bins - 1;
    const bool no_fs = sh.flags & HSF_NO_FUND_SELECT;
    const bool no_drift = sh.flags & HSF_NO_DRIFT;

    long long d = 0;
    float sum = 0.f, best = HS_NEG_INF;
    int bh = 0;
    unsigned path = 0;
    for (int h = 1; h <= sh.H; ++h) {
        const long long m = (long long)h * n + d;                 // eq. 5
        if (m > last) break;                                      // band edge (R4)
        const float a = hs_load<HAS_BASE>(x, ib, m);
        float b = HS_NEG_INF;
        if (m + 1 <= last && !no_drift && !(h == 1 && no_fs)) b = hs_load<HAS_BASE>(x, ib, m + 1);
        const bool shift = b > a;                                 // strict >: ties stay
        d += shift;
        sum = __fadd_rn(sum, shift ? b : a);
        path |= (unsigned)shift << (h - 1);
        const float snr = hs_snr(sum, st.nmis[h - 1], st.inv_sigma[h - 1]);
        if (snr > best) { best = snr; bh = h; }                   // first maximum wins (R6)
    }
    const long long o = (long long)s * sh.out_stride + n;
    st_cs(io.snr + o, best);
    st_cs(io.best_h + o, bh);
    if (io.path) st_cs(io.path + o, path);
}

// Alg. 1, eq. 4, and the _all / + variants.
template <bool HAS_BASE, bool DSTATS = false>
__global__ void __launch_bounds__(256)
hs_presto_generic_kernel(const __grid_constant__ HsShape sh, const __grid_constant__ HsStats st_param, HsIO io) {
    const int s = blockIdx.y;
    __shared__ HsStats s_st;
    if (DSTATS) hs_load_dstats(s_st, io, s, sh.H);
    const HsStats& st = DSTATS ? s_st : st_param;
    const long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= sh.n_fund) return;
    const float* __restrict__ x = io.x + (long long)s * sh.in_stride;
    const float* __restrict__ ib = HAS_BASE ? io.inv_base + (long long)s * sh.in_stride : nullptr;
    const bool all_h = sh.flags & HSF_ALL_HARMONICS;
    const bool all_o = sh.flags & HSF_ALL_ORDERS;

    float best = HS_NEG_INF;
    int bh = 0;
    for (int Hp = 1; Hp <= sh.H; Hp = all_o ? Hp + 1 : Hp * 2) {
        // Round(h n / H') = (2 h n + H') / (2 H') in exact integers (R3), advanced from h to h + step without a
        // division per term: the numerator grows by 2 n step = (q_n 2 H' + r_n) step, q_n = n / H', r_n = 2 (n % H').
        // (n < 2^31: 32-bit arithmetic; ONE division per H'.)
        const unsigned den = 2u * Hp;
        const unsigned qn = (unsigned)n / (unsigned)Hp, rn = 2u * ((unsigned)n - qn * Hp);
        unsigned q = qn, r = rn + Hp;                                         // h = 1: (2 n + H') / (2 H')
        if (r >= den) { r -= den; ++q; }
        float sum = hs_load<HAS_BASE>(x, ib, q);                              // fundamental
        const int step = all_h ? 1 : 2;
        // h = 2 is reached from h = 1 by one increment whatever the step
        q += qn; r += rn;
        if (r >= den) { r -= den; ++q; }
        for (int h = 2; h <= Hp; h += step) {
            sum = __fadd_rn(sum, hs_load<HAS_BASE>(x, ib, q));
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                if (k < step) {
                    q += qn; r += rn;
                    if (r >= den) { r -= den; ++q; }
                }
            }
        }
        const float snr = hs_snr(sum, st.nmis[Hp - 1], st.inv_sigma[Hp - 1]);  // once per H' (R2)
        if (snr > best) { best = snr; bh = Hp; }
    }
    const long long o = (long long)s * sh.out_stride + n;
    st_cs(io.snr + o, best);
    st_cs(io.best_h + o, bh);
}
