// The step before the path (NEXT-2): the statistics mu[s][h], sigma[s][h] that eq. 2 needs.
// The paper only names the step ("{mu, sigma} = GetMeanStdev()"; "mean and standard deviation
// for partial sum of length H"; shared by all algorithms).  Reading R14:
// per spectrum s and order h, the mean and the population standard deviation, over the bins n in [n_lo, n_hi), of the
// partial sum S_h(n) that the selected variant forms at order h -- bins whose order h is not evaluated (greedy band
// edge, reading R4) do not count -- followed by n_clip rounds of outlier rejection: round p keeps the sums with
// lo <= S_h(n) <= hi, lo / hi = mean -/+ clip * std of round p - 1, rounded to fp32.
//
// One launch per round: a thread owns one bin n and walks its orders exactly as the coverage kernels do (fp32 sums in
// the written order), the kept sums of a warp are reduced by shuffles in fp64 (count, sum, sum of squares), added to
// the CTA's accumulators in shared memory and from there to the round's accumulators in global memory (fp64 atomics:
// the order of the additions is not fixed, the values agree to rounding).  A last tiny launch turns the accumulators
// of the final round into mu / sigma.
#pragma once
#include "hs_common.cuh"
#include "hs_generic.cuh"

struct HsStatsArgs {
    long long n_lo, n_hi;          // bins n_lo <= n < n_hi
    double clip;                   // rejection at mean -/+ clip * std
    const double* prev;            // accumulators of the round before ([S][32][3]: count, sum, sum of squares) or null
    double* acc;                   // accumulators of this round ([S][32][3]), zeroed by the caller
};

__device__ __forceinline__ double hs_warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

// mean and population standard deviation from (count, sum, sum of squares); no fused multiply-add, so that the
// fp32 limits derived from them are those of a plain double-precision evaluation
__device__ __forceinline__ void hs_moments(const double* a, double& mean, double& sd) {
    mean = 0.0; sd = 0.0;
    if (a[0] > 0.0) {
        mean = __ddiv_rn(a[1], a[0]);
        const double var = __dsub_rn(__ddiv_rn(a[2], a[0]), __dmul_rn(mean, mean));
        sd = var > 0.0 ? __dsqrt_rn(var) : 0.0;
    }
}

template <bool GREEDY, bool HAS_BASE>
__global__ void __launch_bounds__(256)
hs_stats_pass_kernel(const __grid_constant__ HsShape sh, HsIO io, HsStatsArgs a) {
    __shared__ double s_acc[HS_MAX_H][3];
    __shared__ float s_lo[HS_MAX_H], s_hi[HS_MAX_H];
    const int s = blockIdx.y;
    if (threadIdx.x < HS_MAX_H) {
        float lo = HS_NEG_INF, hi = -HS_NEG_INF;
        if (a.prev) {
            double mean, sd;
            hs_moments(a.prev + ((long long)s * HS_MAX_H + threadIdx.x) * 3, mean, sd);
            lo = __double2float_rn(__dsub_rn(mean, __dmul_rn(a.clip, sd)));
            hi = __double2float_rn(__dadd_rn(mean, __dmul_rn(a.clip, sd)));
        }
        s_lo[threadIdx.x] = lo; s_hi[threadIdx.x] = hi;
        s_acc[threadIdx.x][0] = 0.0; s_acc[threadIdx.x][1] = 0.0; s_acc[threadIdx.x][2] = 0.0;
    }
    __syncthreads();
    const long long n = a.n_lo + (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool have = n < a.n_hi;
    const float* __restrict__ x = io.x + (long long)s * sh.in_stride;
    const float* __restrict__ ib = HAS_BASE ? io.inv_base + (long long)s * sh.in_stride : nullptr;
    const int lane = threadIdx.x & 31;

    auto add = [&](int h, bool valid, float v) {            // every lane of the warp calls this for every order
        const bool keep = valid && v >= s_lo[h - 1] && v <= s_hi[h - 1];
        const unsigned m = __ballot_sync(0xffffffffu, keep);
        if (m == 0) return;
        const double dv = keep ? (double)v : 0.0;
        const double s1 = hs_warp_sum(dv), s2 = hs_warp_sum(__dmul_rn(dv, dv));
        if (lane == 0) {
            atomicAdd(&s_acc[h - 1][0], (double)__popc(m));
            atomicAdd(&s_acc[h - 1][1], s1);
            atomicAdd(&s_acc[h - 1][2], s2);
        }
    };

    if (GREEDY) {                                           // Alg. 2 as hs_greedy_generic_kernel walks it
        const long long last = sh.n_bins - 1;
        const bool no_fs = sh.flags & HSF_NO_FUND_SELECT, no_drift = sh.flags & HSF_NO_DRIFT;
        long long d = 0;
        float sum = 0.f;
        bool alive = have;
        for (int h = 1; h <= sh.H; ++h) {
            const long long m = (long long)h * n + d;
            alive = alive && m <= last;
            if (alive) {
                const float av = hs_load<HAS_BASE>(x, ib, m);
                float bv = HS_NEG_INF;
                if (m + 1 <= last && !no_drift && !(h == 1 && no_fs)) bv = hs_load<HAS_BASE>(x, ib, m + 1);
                const bool shift = bv > av;
                d += shift;
                sum = __fadd_rn(sum, shift ? bv : av);
            }
            add(h, alive, sum);
        }
    } else {                                                // Alg. 1 family as hs_presto_generic_kernel walks it
        const bool all_h = sh.flags & HSF_ALL_HARMONICS, all_o = sh.flags & HSF_ALL_ORDERS;
        for (int Hp = 1; Hp <= sh.H; Hp = all_o ? Hp + 1 : Hp * 2) {
            float sum = 0.f;
            if (have) {
                const unsigned den = 2u * Hp;
                const unsigned qn = (unsigned)n / (unsigned)Hp, rn = 2u * ((unsigned)n - qn * Hp);
                unsigned q = qn, r = rn + Hp;
                if (r >= den) { r -= den; ++q; }
                sum = hs_load<HAS_BASE>(x, ib, q);
                const int step = all_h ? 1 : 2;
                q += qn; r += rn;
                if (r >= den) { r -= den; ++q; }
                for (int h = 2; h <= Hp; h += step) {
                    sum = __fadd_rn(sum, hs_load<HAS_BASE>(x, ib, q));
                    for (int k = 0; k < step; ++k) {
                        q += qn; r += rn;
                        if (r >= den) { r -= den; ++q; }
                    }
                }
            }
            add(Hp, have, sum);
        }
    }
    __syncthreads();
    if (threadIdx.x < 3 * HS_MAX_H) {
        const int h = threadIdx.x / 3, k = threadIdx.x % 3;
        const double v = s_acc[h][k];
        if (v != 0.0) atomicAdd(a.acc + ((long long)s * HS_MAX_H + h) * 3 + k, v);
    }
}

// mu[s][h], sigma[s][h] from the accumulators of the last round: no samples -> (0, 1); zero deviation -> sigma 1
__global__ void hs_stats_finish_kernel(const double* __restrict__ acc, int S, int H, float* __restrict__ mu, float* __restrict__ sigma) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= S * H) return;
    const int s = i / H, h = i % H;
    const double* a = acc + ((long long)s * HS_MAX_H + h) * 3;
    double mean, sd;
    hs_moments(a, mean, sd);
    mu[i] = a[0] > 0.0 ? __double2float_rn(mean) : 0.f;
    sigma[i] = (a[0] > 0.0 && sd > 0.0) ? __double2float_rn(sd) : 1.f;
}
