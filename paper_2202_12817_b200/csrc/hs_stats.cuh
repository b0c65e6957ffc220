// The step before the path (NEXT-2): the statistics mu[s][h], sigma[s][h] that eq. 2 needs.
// The paper only names the step ("{mu, sigma} = GetMeanStdev()"; "mean and standard deviation
// for partial sum of length H"; shared by all algorithms).  Reading R14:
// per spectrum s and order h, the mean and the population standard deviation, over the bins n in [n_lo, n_hi), of the
// partial sum S_h(n) that the selected variant forms at order h -- bins whose order h is not evaluated (greedy band
// edge, reading R4) do not count -- followed by n_clip rounds of outlier rejection: round p keeps the sums with
// lo <= S_h(n) <= hi, lo / hi = mean -/+ clip * std of round p - 1, rounded to fp32.
//
// One launch per round: a lane owns one bin n at a time and walks its orders exactly as the coverage kernels do (fp32
// sums in the written order); the sums of a warp are transposed through shared memory so that lane h - 1 adds up order
// h in fp64 (count, sum, sum of squares) in registers, and adds its totals to the round's accumulators in global
// memory with fp64 atomics at the end (the order of the additions is not fixed, the values agree to rounding).  A last
// tiny launch turns the accumulators of the final round into mu / sigma.
#pragma once
#include "hs_common.cuh"
#include "hs_generic.cuh"

struct HsStatsArgs {
    long long n_lo, n_hi;          // bins n_lo <= n < n_hi
    double clip;                   // rejection at mean -/+ clip * std
    const double* prev;            // accumulators of the round before ([S][32][3]: count, sum, sum of squares) or null
    double* acc;                   // accumulators of this round ([S][32][3]), zeroed by the caller
    float* cache;                  // hs_stats_store_kernel: the sums are written here, [S][H][cpad] (NaN = no sample)
    long long cpad;                // elements between the rows of `cache` (>= n_hi - n_lo, multiple of 4)
};

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

// grid: (chunks, spectra); a warp takes groups of 32 consecutive bins of [n_lo, n_hi) in a grid-stride loop.  Lane l walks
// the orders of its bin and leaves S_h (NaN: order not evaluated, or rejected) in the warp's [order][lane] tile of
// shared memory; then lane h - 1 adds up the 32 entries of order h in fp64 (count, sum, sum of squares) into its own
// registers -- a transposition instead of 20 shuffles per order -- and adds them to global memory once, at the end.
template <bool GREEDY, bool HAS_BASE>
__global__ void __launch_bounds__(256)
hs_stats_pass_kernel(const __grid_constant__ HsShape sh, HsIO io, HsStatsArgs a) {
    constexpr int WARPS = 8, PITCH = 33;                    // 33: both the lane-major stores and the order-major loads are conflict-free
    __shared__ float s_v[WARPS][HS_MAX_H * PITCH];
    const int s = blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // rejection limits of this lane's order (lane = h - 1) from the accumulators of the round before
    float lo = HS_NEG_INF, hi = -HS_NEG_INF;
    if (a.prev) {
        double mean, sd;
        hs_moments(a.prev + ((long long)s * HS_MAX_H + lane) * 3, mean, sd);
        lo = __double2float_rn(__dsub_rn(mean, __dmul_rn(a.clip, sd)));
        hi = __double2float_rn(__dadd_rn(mean, __dmul_rn(a.clip, sd)));
    }
    const float* __restrict__ x = io.x + (long long)s * sh.in_stride;
    const float* __restrict__ ib = HAS_BASE ? io.inv_base + (long long)s * sh.in_stride : nullptr;
    float* tile = s_v[warp];
    const float NOT = __int_as_float(0x7fc00000);           // NaN marks "no sample"
    double cnt = 0.0, s1 = 0.0, s2 = 0.0;                   // of order lane + 1

    const long long groups = (a.n_hi - a.n_lo + 31) / 32;
    for (long long g = (long long)blockIdx.x * WARPS + warp; g < groups; g += (long long)gridDim.x * WARPS) {
        const long long n = a.n_lo + g * 32 + lane;
        const bool have = n < a.n_hi;
#pragma unroll 1
        for (int h = sh.H; h < HS_MAX_H; ++h) tile[h * PITCH + lane] = NOT;
        if (GREEDY) {                                       // Alg. 2 as hs_greedy_generic_kernel walks it
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
                tile[(h - 1) * PITCH + lane] = alive ? sum : NOT;
            }
        } else {                                            // Alg. 1 family as hs_presto_generic_kernel walks it
            const bool all_h = sh.flags & HSF_ALL_HARMONICS, all_o = sh.flags & HSF_ALL_ORDERS;
            for (int Hp = 1; Hp <= sh.H; ++Hp) {
                const bool in_set = all_o || (Hp & (Hp - 1)) == 0;
                float sum = 0.f;
                if (have && in_set) {
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
                tile[(Hp - 1) * PITCH + lane] = (have && in_set) ? sum : NOT;
            }
        }
        __syncwarp();
        const float* row = tile + lane * PITCH;             // the 32 sums of order lane + 1
#pragma unroll 8
        for (int l = 0; l < 32; ++l) {
            const float v = row[l];
            if (v >= lo && v <= hi) {                       // false for NaN
                const double dv = (double)v;
                cnt += 1.0; s1 += dv; s2 += __dmul_rn(dv, dv);
            }
        }
        __syncwarp();
    }
    // the CTA's totals (shared-memory atomics), then one set of global atomics per CTA
    __shared__ double s_acc[HS_MAX_H][3];
    if (warp == 0) { s_acc[lane][0] = 0.0; s_acc[lane][1] = 0.0; s_acc[lane][2] = 0.0; }
    __syncthreads();
    if (cnt != 0.0) { atomicAdd(&s_acc[lane][0], cnt); atomicAdd(&s_acc[lane][1], s1); atomicAdd(&s_acc[lane][2], s2); }
    __syncthreads();
    if (threadIdx.x < 3 * HS_MAX_H) {
        const double v = s_acc[threadIdx.x / 3][threadIdx.x % 3];
        if (v != 0.0) atomicAdd(a.acc + (long long)s * HS_MAX_H * 3 + threadIdx.x, v);
    }
}

// The gather of the cached path: the sums S_h(n), n in [n_lo, n_hi), h = 1..H, are written to a.cache as fp32 -- order by
// order, 128 bytes per warp and order -- and nothing else happens here: no shared-memory tile and no moments, so the
// kernel runs at full occupancy with two independent chains per lane (the greedy form).  Every round, the first
// included, then streams the rows back (hs_stats_cached_kernel).  The chains are those of hs_stats_pass_kernel, term
// for term, so the stored values are the values that kernel compares.
template <bool GREEDY, bool HAS_BASE>
__global__ void __launch_bounds__(256)
hs_stats_store_kernel(const __grid_constant__ HsShape sh, HsIO io, HsStatsArgs a) {
    constexpr int WARPS = 8, R = 2;
    const int s = blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const float* __restrict__ x = io.x + (long long)s * sh.in_stride;
    const float* __restrict__ ib = HAS_BASE ? io.inv_base + (long long)s * sh.in_stride : nullptr;
    float* __restrict__ crow = a.cache + (long long)s * sh.H * a.cpad;
    const float NOT = __int_as_float(0x7fc00000);           // NaN marks "no sample"
    const long long groups = (a.n_hi - a.n_lo + 31) / 32;
    for (long long g0 = ((long long)blockIdx.x * WARPS + warp) * R; g0 < groups; g0 += (long long)gridDim.x * WARPS * R) {
        if (GREEDY) {
            const long long last = sh.n_bins - 1;
            const bool no_fs = sh.flags & HSF_NO_FUND_SELECT, no_drift = sh.flags & HSF_NO_DRIFT;
            long long n[R], d[R];
            float sum[R];
            bool have[R], alive[R];
#pragma unroll
            for (int j = 0; j < R; ++j) {
                n[j] = a.n_lo + (g0 + j) * 32 + lane;
                have[j] = n[j] < a.n_hi;
                alive[j] = have[j]; d[j] = 0; sum[j] = 0.f;
            }
            for (int h = 1; h <= sh.H; ++h) {
                float av[R], bv[R];
#pragma unroll
                for (int j = 0; j < R; ++j) {
                    const long long m = (long long)h * n[j] + d[j];
                    alive[j] = alive[j] && m <= last;
                    av[j] = 0.f; bv[j] = HS_NEG_INF;
                    if (alive[j]) {
                        av[j] = hs_load<HAS_BASE>(x, ib, m);
                        if (m + 1 <= last && !no_drift && !(h == 1 && no_fs)) bv[j] = hs_load<HAS_BASE>(x, ib, m + 1);
                    }
                }
#pragma unroll
                for (int j = 0; j < R; ++j) {
                    if (alive[j]) {
                        const bool shift = bv[j] > av[j];
                        d[j] += shift;
                        sum[j] = __fadd_rn(sum[j], shift ? bv[j] : av[j]);
                    }
                    if (have[j]) crow[(long long)(h - 1) * a.cpad + (n[j] - a.n_lo)] = alive[j] ? sum[j] : NOT;
                }
            }
        } else {                                            // Alg. 1 family as hs_presto_generic_kernel walks it
            const bool all_h = sh.flags & HSF_ALL_HARMONICS, all_o = sh.flags & HSF_ALL_ORDERS;
            for (int j = 0; j < R; ++j) {
                const long long n = a.n_lo + (g0 + j) * 32 + lane;
                if (n >= a.n_hi) continue;
                for (int Hp = 1; Hp <= sh.H; ++Hp) {
                    const bool in_set = all_o || (Hp & (Hp - 1)) == 0;
                    float sum = 0.f;
                    if (in_set) {
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
                    crow[(long long)(Hp - 1) * a.cpad + (n - a.n_lo)] = in_set ? sum : NOT;
                }
            }
        }
    }
}

// A round of the cached path (the first one has no limits: prev == nullptr): order h of spectrum s streams its row of stored sums (fp32, NaN = no sample),
// keeps lo <= S <= hi with the limits of the round before -- the comparison and the fp64 moments of
// hs_stats_pass_kernel, on the same fp32 values -- and adds its totals to the round's accumulators.
// grid: (chunks, H, spectra); the additions are fp64 in an unspecified order, as in the pass kernel.
__global__ void __launch_bounds__(256)
hs_stats_cached_kernel(const float* __restrict__ cache, long long cpad, long long count, int H, double clip,
                       const double* __restrict__ prev, double* __restrict__ acc) {
    const int h = blockIdx.y, s = blockIdx.z;
    float lo = HS_NEG_INF, hi = -HS_NEG_INF;
    if (prev) {
        double mean, sd;
        hs_moments(prev + ((long long)s * HS_MAX_H + h) * 3, mean, sd);
        lo = __double2float_rn(__dsub_rn(mean, __dmul_rn(clip, sd)));
        hi = __double2float_rn(__dadd_rn(mean, __dmul_rn(clip, sd)));
    }
    const float* __restrict__ row = cache + ((long long)s * H + h) * cpad;
    double cnt = 0.0, s1 = 0.0, s2 = 0.0;
    auto take = [&](float v) {
        if (v >= lo && v <= hi) {                           // false for NaN
            const double dv = (double)v;
            cnt += 1.0; s1 += dv; s2 += __dmul_rn(dv, dv);
        }
    };
    const long long n4 = count >> 2;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += (long long)gridDim.x * blockDim.x) {
        const float4 q = __ldcs(reinterpret_cast<const float4*>(row) + i);
        take(q.x); take(q.y); take(q.z); take(q.w);
    }
    if (blockIdx.x == 0 && threadIdx.x < (count & 3)) take(row[(n4 << 2) + threadIdx.x]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        cnt += __shfl_down_sync(0xffffffffu, cnt, o);
        s1 += __shfl_down_sync(0xffffffffu, s1, o);
        s2 += __shfl_down_sync(0xffffffffu, s2, o);
    }
    __shared__ double s_acc[3];
    if (threadIdx.x < 3) s_acc[threadIdx.x] = 0.0;
    __syncthreads();
    if ((threadIdx.x & 31) == 0 && cnt != 0.0) { atomicAdd(&s_acc[0], cnt); atomicAdd(&s_acc[1], s1); atomicAdd(&s_acc[2], s2); }
    __syncthreads();
    if (threadIdx.x < 3 && s_acc[threadIdx.x] != 0.0) atomicAdd(acc + ((long long)s * HS_MAX_H + h) * 3 + threadIdx.x, s_acc[threadIdx.x]);
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

// Spectrum whitening as its own pass ("further preprocessing, which includes spectrum whitening"):
// y[s][b] = x[s][b] * inv_baseline[s][b], ONE fp32 multiply -- exactly the product the fused path forms (reading R13),
// so hs_run_*(y, NULL) returns the bits of hs_run_*(x, inv_baseline).  16-byte streaming loads, 16-byte stores;
// the gather of the harmonic sum then reads one array instead of two.
__global__ void __launch_bounds__(256)
hs_whiten_kernel(const float* __restrict__ x, const float* __restrict__ ib, float* __restrict__ y, long long in_stride,
                 long long y_stride, int n_bins) {
    const int s = blockIdx.y;
    const float* xr = x + (long long)s * in_stride;
    const float* br = ib + (long long)s * in_stride;
    float* yr = y + (long long)s * y_stride;
    // rows on 32-byte units: 32-byte loads and stores (whole sectors per lane), the remainder below as before
    if ((((reinterpret_cast<uintptr_t>(xr)) | reinterpret_cast<uintptr_t>(br) | reinterpret_cast<uintptr_t>(yr)) & 31u) == 0) {
        const int n8 = n_bins >> 3;
        for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n8; i += gridDim.x * blockDim.x) {
            float a[8], b[8];
            asm volatile("ld.global.cs.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n"
                         : "=f"(a[0]), "=f"(a[1]), "=f"(a[2]), "=f"(a[3]), "=f"(a[4]), "=f"(a[5]), "=f"(a[6]), "=f"(a[7]) : "l"(xr + 8ll * i));
            asm volatile("ld.global.cs.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n"
                         : "=f"(b[0]), "=f"(b[1]), "=f"(b[2]), "=f"(b[3]), "=f"(b[4]), "=f"(b[5]), "=f"(b[6]), "=f"(b[7]) : "l"(br + 8ll * i));
#pragma unroll
            for (int k = 0; k < 8; ++k) a[k] = __fmul_rn(a[k], b[k]);
            asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};\n" :: "l"(yr + 8ll * i), "f"(a[0]), "f"(a[1]), "f"(a[2]), "f"(a[3]),
                         "f"(a[4]), "f"(a[5]), "f"(a[6]), "f"(a[7]) : "memory");
        }
        if (blockIdx.x == 0 && threadIdx.x < (n_bins & 7)) {
            const int i = (n8 << 3) + threadIdx.x;
            yr[i] = __fmul_rn(__ldg(xr + i), __ldg(br + i));
        }
        return;
    }
    const int n4 = n_bins >> 2;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += gridDim.x * blockDim.x) {
        const float4 a = __ldcs(reinterpret_cast<const float4*>(xr) + i);
        const float4 b = __ldcs(reinterpret_cast<const float4*>(br) + i);
        reinterpret_cast<float4*>(yr)[i] = make_float4(__fmul_rn(a.x, b.x), __fmul_rn(a.y, b.y), __fmul_rn(a.z, b.z), __fmul_rn(a.w, b.w));
    }
    if (blockIdx.x == 0 && threadIdx.x < (n_bins & 3)) {
        const int i = (n4 << 2) + threadIdx.x;
        yr[i] = __fmul_rn(__ldg(xr + i), __ldg(br + i));
    }
}
