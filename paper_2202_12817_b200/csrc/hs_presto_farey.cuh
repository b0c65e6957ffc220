// PRESTO_all and PRESTO+ (flags HS_PRESTO_ALL_HARMONICS [| HS_PRESTO_ALL_ORDERS]):
//     S_{H'}[n] = sum_{h = 1..H'} x[Round(h n / H')],   H' = 1, 2, 4, .. (PRESTO_all)  or  H' = 1..H (PRESTO+).
//
// Round(h n / H') = (2 h n + H') / (2 H') depends on the fraction h/H' only, so every term of every H' is one of the
// terms of the REDUCED fractions p/d, d <= H, gcd(p, d) = 1 (a Farey sequence: 323 of them at H = 32 against the
// 528 terms PRESTO+ visits, 32 against 63 for PRESTO_all), and
//     S_{H'} = sum over the divisors d of H' of  N_d,    N_d = sum_{p <= d, gcd(p, d) = 1} x[Round(p n / d)].
// Every (p, d) is a compile-time constant here: with n = a d + b the index is p a + (2 p b + d) / (2 d), one
// division of n by a constant per d and a multiply-shift per term.  One thread per top bin n, consecutive lanes
// consecutive bins: the 32 lanes of a warp read p/d * 32 + 1 consecutive words per term (coalesced, L1-resident).
// The sums are formed in fp32 as written above (N_d by increasing p, S_{H'} by increasing d).
#pragma once
#include "hs_common.cuh"

namespace hs_farey {
__host__ __device__ constexpr int gcd(int a, int b) { return b == 0 ? a : gcd(b, a % b); }
__host__ __device__ constexpr bool pow2(int v) { return (v & (v - 1)) == 0; }
}  // namespace hs_farey

namespace hs_farey {

// acc += x[Round(P n / D)] for P = P0..D with gcd(P, D) = 1 (n = a D + b), by increasing P
template <int D, int P>
__device__ __forceinline__ void terms(const float* __restrict__ x, unsigned a, unsigned b, float& acc) {
    if constexpr (gcd(P, D) == 1) {
        const unsigned idx = (unsigned)P * a + (2u * P * b + D) / (2u * D);
        const float v = __ldg(x + idx);
        acc = (P == 1) ? v : __fadd_rn(acc, v);
    }
    if constexpr (P < D) terms<D, P + 1>(x, a, b, acc);
}

// N_D for D = D0..HS_MAX_H
template <bool ALL_ORDERS, int D>
__device__ __forceinline__ void levels(const float* __restrict__ x, unsigned n, int H, float (&Nd)[HS_MAX_H + 1]) {
    Nd[D] = 0.f;
    if constexpr (ALL_ORDERS || pow2(D)) {
        if (D <= H) {
            const unsigned a = n / (unsigned)D, b = n - a * (unsigned)D;
            float acc = 0.f;
            terms<D, 1>(x, a, b, acc);
            Nd[D] = acc;
        }
    }
    if constexpr (D < HS_MAX_H) levels<ALL_ORDERS, D + 1>(x, n, H, Nd);
}

// S_{HP} = sum of N_d over the divisors d of HP, by increasing d
template <int HP, int Dv>
__device__ __forceinline__ void divisor_sum(const float (&Nd)[HS_MAX_H + 1], float& S) {
    if constexpr (HP % Dv == 0) S = (Dv == 1) ? Nd[1] : __fadd_rn(S, Nd[Dv]);
    if constexpr (Dv < HP) divisor_sum<HP, Dv + 1>(Nd, S);
}

template <bool ALL_ORDERS, int HP>
__device__ __forceinline__ void orders(const float (&Nd)[HS_MAX_H + 1], const HsStats& st, int H, float& best, int& bh) {
    if constexpr (ALL_ORDERS || pow2(HP)) {
        if (HP <= H) {
            float S = 0.f;
            divisor_sum<HP, 1>(Nd, S);
            const float snr = hs_snr(S, st.nmis[HP - 1], st.inv_sigma[HP - 1]);   // once per H' (R2)
            if (snr > best) { best = snr; bh = HP; }                           // first maximum wins (R6)
        }
    }
    if constexpr (HP < HS_MAX_H) orders<ALL_ORDERS, HP + 1>(Nd, st, H, best, bh);
}

}  // namespace hs_farey

template <bool ALL_ORDERS>
__global__ void __launch_bounds__(256)
hs_presto_farey_kernel(const __grid_constant__ HsShape sh, const __grid_constant__ HsStats st, HsIO io) {
    using namespace hs_farey;
    const int s = blockIdx.y;
    const unsigned n = blockIdx.x * 256u + threadIdx.x;
    if (n >= (unsigned)sh.n_fund) return;
    const float* x = io.x + (long long)s * sh.in_stride;
    asm volatile("" : "+l"(x));                               // one materialised row pointer
    const int H = sh.H;
    float Nd[HS_MAX_H + 1];
    levels<ALL_ORDERS, 1>(x, n, H, Nd);
    float best = HS_NEG_INF;
    int bh = 0;
    orders<ALL_ORDERS, 1>(Nd, st, H, best, bh);
    const long long o = (long long)s * sh.out_stride + n;
    st_cs(io.snr + o, best);
    st_cs(io.best_h + o, bh);
}
