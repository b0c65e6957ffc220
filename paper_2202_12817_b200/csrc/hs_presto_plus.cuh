// PRESTO+ / PRESTO_all (flags HS_PRESTO_ALL_HARMONICS [| HS_PRESTO_ALL_ORDERS]) rebuilt for B200:
//     S_{H'}[n] = sum_{h = 1..H'} x[Round(h n / H')],   H' = 1..H (PRESTO+)  or  H' = 1, 2, 4, .. (PRESTO_all).
// As in hs_presto_farey.cuh every term is a term of a REDUCED fraction P/D (gcd(P, D) = 1, D <= H: 323 of them at
// H = 32), S_{H'} = sum over the divisors d of H' of N_d, N_d[n] = sum_{P coprime to d} x[Round(P n / d)].
// What is new is where the terms come from and who adds them:
//   * a CTA owns a tile of T = 512 consecutive top bins; for a group of denominators the spans
//     x[Round(P n0 / D) .. Round(P (n0 + T - 1) / D)] of all their fractions are staged in shared memory by 16-byte
//     cp.async copies (each word of a span is used exactly once, so staging only turns 324 narrow loads per bin into
//     40 wide ones: the one-thread-per-bin kernel was bound by its L1-miss requests, 0.1 warp-loads per clock and SM);
//   * for denominator D thread t adds the terms of the outputs t, t + B_D, t + 2 B_D, .. with B_D = D (256 / D), a
//     multiple of D: moving an output by B_D moves the index of fraction P/D by exactly P (256 / D), so after the
//     first output every term is ONE shared-memory load at an immediate offset and one add;
//   * N_D goes to shared memory ([D][output]); at the end thread t forms S_{H'} of outputs t, t + 256 from the N_d of
//     the divisors, the SNR once per H' (reading R2) and the first maximum (R6).
// The sums are formed in fp32 exactly as in hs_presto_farey.cuh (N_d by increasing P, S_{H'} by increasing d).
// Measured on cfg3 (256 x 2^22): PRESTO+ 376 ms at H = 32 (Farey kernel 415), 82 ms at H = 16 (Farey 202, coverage kernel
// 147).  ncu at H = 32: 3 470 thread instructions per output at 0.9 IPC, `no_instruction` 4.9 warps per issue: the 323
// unrolled fraction blocks are 312 KB of straight-line code that the instruction caches cannot hold.  A version with
// run-time loops over P (170 KB, twice the dynamic instructions) ran in 744 ms; 128 threads per CTA (four outputs per
// thread and denominator) in 446 ms.  Not an HBM kernel: the bound is 442 fp32 adds and 323 shared-memory loads per
// output (14 / 40 ms); it is used for PRESTO+ only, PRESTO_all stays on the Farey kernel (16.0 against 19.6 ms).
#pragma once
#include "hs_common.cuh"
#include "hs_presto_farey.cuh"

namespace hs_plus {
using hs_farey::gcd;
using hs_farey::pow2;

constexpr int T = 512;           // outputs per CTA tile
constexpr int NT = 256;          // threads per CTA
constexpr int CAP = 8192;        // words of the span buffer (32 KB): the largest single denominator (31) needs 7 920

__host__ __device__ constexpr bool used(int P, int D) { return gcd(P, D) == 1 && (P < D || D == 1); }
// words reserved for the span of P/D: its length <= P (T - 1) / D + 2, plus the alignment shift (<= 3), rounded up to 4
__host__ __device__ constexpr int span_cap(int P, int D) { return ((P * (T - 1)) / D + 2 + 3 + 3) & ~3; }
__host__ __device__ constexpr int span_off(int P, int D) {      // offset of the span of P/D inside the spans of D
    int o = 0;
    for (int q = 1; q < P; ++q) if (used(q, D)) o += span_cap(q, D);
    return o;
}
__host__ __device__ constexpr int d_words(int D) { return span_off(D + 1, D); }
template <bool ALL_ORDERS> __host__ __device__ constexpr bool d_active(int D) { return ALL_ORDERS || pow2(D); }
// denominators D0 .. group_end(D0) share one filling of the span buffer
template <bool ALL_ORDERS> __host__ __device__ constexpr int group_end(int D0) {
    int w = 0, D = D0;
    for (; D <= HS_MAX_H; ++D) {
        const int add = d_active<ALL_ORDERS>(D) ? d_words(D) : 0;
        if (D > D0 && w + add > CAP) break;
        w += add;
    }
    return D - 1;
}
template <bool ALL_ORDERS> __host__ __device__ constexpr int d_base(int D0, int D) {   // offset of D's spans inside its group
    int w = 0;
    for (int q = D0; q < D; ++q) if (d_active<ALL_ORDERS>(q)) w += d_words(q);
    return w;
}

__device__ __forceinline__ unsigned smem_u32p(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

// Round(P n / D) with n = a D + b (b < D): P a + (2 P b + D) / (2 D)
template <int P, int D>
__device__ __forceinline__ unsigned idx_of(unsigned a, unsigned b) { return (unsigned)P * a + (2u * P * b + D) / (2u * D); }

// ---- staging: warp `warp` copies the spans whose running number is warp, warp + NT / 32, .. ----
template <int D, int P>
__device__ __forceinline__ void stage_spans(float* __restrict__ buf, const float* __restrict__ x, unsigned a0, unsigned b0,
                                            long long lim, int warp, int lane, int& counter) {
    if constexpr (used(P, D)) {
        if ((counter++ & (NT / 32 - 1)) == warp) {
            const unsigned g0 = idx_of<P, D>(a0, b0);
            const unsigned ga = g0 & ~3u;
            constexpr int chunks = span_cap(P, D) / 4;
#pragma unroll
            for (int c0 = 0; c0 < chunks; c0 += 32) {
                const int c = c0 + lane;
                if (c < chunks && (long long)ga + 4 * c + 3 < lim)
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" :: "r"(smem_u32p(buf + span_off(P, D) + 4 * c)), "l"(x + ga + 4 * c) : "memory");
            }
        }
    }
    if constexpr (P < D) stage_spans<D, P + 1>(buf, x, a0, b0, lim, warp, lane, counter);
}

// ---- N_D of the thread's outputs t + B_D k ----
template <int D, int P, int K>
__device__ __forceinline__ void add_fraction(const float* __restrict__ buf, unsigned a0, unsigned b0, unsigned da, unsigned b,
                                             float (&acc)[K], int t) {
    if constexpr (used(P, D)) {
        constexpr int M = NT / D, B = D * M;
        const unsigned g0 = idx_of<P, D>(a0, b0);
        // index of the thread's first output relative to the span start, plus the alignment shift of the staged copy
        const unsigned rel = (unsigned)P * da + (2u * P * b + D) / (2u * D) - (2u * P * b0 + D) / (2u * D) + (g0 & 3u);
        const float* p = buf + span_off(P, D) + rel;
#pragma unroll
        for (int k = 0; k < K; ++k) {
            if (k == 0 || t + B * k < T) {
                const float v = p[P * M * k];
                acc[k] = (P == 1) ? v : __fadd_rn(acc[k], v);
            }
        }
    }
    if constexpr (P < D) add_fraction<D, P + 1, K>(buf, a0, b0, da, b, acc, t);
}

template <bool ALL_ORDERS, int D0, int D>
__device__ __forceinline__ void stage_group(float* __restrict__ buf, const float* __restrict__ x, unsigned n0, long long lim, int H,
                                            int warp, int lane, int& counter) {
    if constexpr (d_active<ALL_ORDERS>(D)) {
        if (D <= H) stage_spans<D, 1>(buf + d_base<ALL_ORDERS>(D0, D), x, n0 / (unsigned)D, n0 % (unsigned)D, lim, warp, lane, counter);
    }
    if constexpr (D < group_end<ALL_ORDERS>(D0)) stage_group<ALL_ORDERS, D0, D + 1>(buf, x, n0, lim, H, warp, lane, counter);
}

template <bool ALL_ORDERS, int D0, int D>
__device__ __forceinline__ void compute_group(const float* __restrict__ buf, float* __restrict__ nd, unsigned n0, int H, int t) {
    if constexpr (d_active<ALL_ORDERS>(D)) {
        constexpr int M = NT / D, B = D * M, K = (T + B - 1) / B;
        if (D <= H && t < B) {
            const unsigned a0 = n0 / (unsigned)D, b0 = n0 % (unsigned)D;
            const unsigned q = b0 + (unsigned)t;                     // n0 + t = (a0 + q / D) D + q % D
            const unsigned da = q / (unsigned)D, b = q - da * (unsigned)D;
            float acc[K];
#pragma unroll
            for (int k = 0; k < K; ++k) acc[k] = 0.f;
            add_fraction<D, 1, K>(buf + d_base<ALL_ORDERS>(D0, D), a0, b0, da, b, acc, t);
#pragma unroll
            for (int k = 0; k < K; ++k)
                if (k == 0 || t + B * k < T) nd[(D - 1) * T + t + B * k] = acc[k];
        }
    }
    if constexpr (D < group_end<ALL_ORDERS>(D0)) compute_group<ALL_ORDERS, D0, D + 1>(buf, nd, n0, H, t);
}

template <bool ALL_ORDERS, int D0>
__device__ __forceinline__ void groups(float* __restrict__ buf, float* __restrict__ nd, const float* __restrict__ x, unsigned n0,
                                       long long lim, int H, int t) {
    if (D0 <= H) {
        int counter = 0;
        stage_group<ALL_ORDERS, D0, D0>(buf, x, n0, lim, H, t >> 5, t & 31, counter);
        asm volatile("cp.async.commit_group;\n cp.async.wait_group 0;\n" ::: "memory");
        __syncthreads();
        compute_group<ALL_ORDERS, D0, D0>(buf, nd, n0, H, t);
        __syncthreads();                                             // the buffer is free again; N_D is visible
    }
    constexpr int next = group_end<ALL_ORDERS>(D0) + 1;
    if constexpr (next <= HS_MAX_H) groups<ALL_ORDERS, next>(buf, nd, x, n0, lim, H, t);
}

constexpr int smem_bytes() { return 4 * (HS_MAX_H * T + CAP); }

}  // namespace hs_plus

// grid: (tiles of 512 outputs, spectra); block: 256 threads; dynamic shared memory: hs_plus::smem_bytes()
template <bool ALL_ORDERS>
__global__ void __launch_bounds__(hs_plus::NT, 2)
hs_presto_plus_kernel(const __grid_constant__ HsShape sh, const __grid_constant__ HsStats st, HsIO io) {
    using namespace hs_plus;
    extern __shared__ float4 hs_plus_smem4[];
    float* nd = reinterpret_cast<float*>(hs_plus_smem4);            // [HS_MAX_H][T]
    float* buf = nd + HS_MAX_H * T;                                  // [CAP]
    const int s = blockIdx.y;
    const int t = threadIdx.x;
    const unsigned n0 = blockIdx.x * (unsigned)T;
    const float* x = io.x + (long long)s * sh.in_stride;
    const int H = sh.H;
    groups<ALL_ORDERS, 1>(buf, nd, x, n0, sh.in_stride, H, t);
#pragma unroll
    for (int k = 0; k < T / NT; ++k) {
        const unsigned n = n0 + t + NT * k;
        if (n < (unsigned)sh.n_fund) {
            float Nd[HS_MAX_H + 1];
            Nd[0] = 0.f;
#pragma unroll
            for (int d = 1; d <= HS_MAX_H; ++d) Nd[d] = (d <= H && d_active<ALL_ORDERS>(d)) ? nd[(d - 1) * T + t + NT * k] : 0.f;
            float best = HS_NEG_INF;
            int bh = 0;
            hs_farey::orders<ALL_ORDERS, 1>(Nd, st, H, best, bh);
            const long long o = (long long)s * sh.out_stride + n;
            st_cs(io.snr + o, best);
            st_cs(io.best_h + o, bh);
        }
    }
}
