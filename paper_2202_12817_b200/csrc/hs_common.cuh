// Shared device-side definitions of the harmonic-sum kernels (CUDA path only; the CPU oracle
// under oracle/ shares nothing with this directory).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define HS_MAX_H 32

// Normalisation statistics travel by value as a __grid_constant__ kernel parameter
// (mu_H, sigma_H of the partial sum of length H).  Eq. 2, (sum - mu)/sigma, is formed
// as ONE fused multiply-add, sum * (1/sigma) + (-mu/sigma), with both constants rounded once on
// the host: index h-1 holds order h.
struct HsStats {
    float nmis[HS_MAX_H];        // -mu * (1/sigma)
    float inv_sigma[HS_MAX_H];   // 1/sigma
};

struct HsShape {
    long long n_bins;      // N
    long long n_fund;      // outputs for n < n_fund
    long long in_stride;   // elements between input rows
    long long out_stride;  // elements between output rows
    int n_spectra;         // S
    int H;                 // maximum harmonic order
    unsigned flags;        // HS_* algorithm flags (hs.h)
    int Z;                 // 2-D plans (hs_plan_2d): rows are z = -Z .. Z, n_spectra = 2 Z + 1; 0 otherwise
};

struct HsIO {
    const float* __restrict__ x;         // [S][in_stride]
    const float* __restrict__ inv_base;  // nullable
    float* __restrict__ snr;             // [S][out_stride]
    int* __restrict__ best_h;            // [S][out_stride]
    unsigned* __restrict__ path;         // nullable (greedy only)
    const float* __restrict__ d_mu;      // nullable: per-spectrum statistics [S][H] on the device (hs_run_*_dstats);
    const float* __restrict__ d_sigma;   //           then the by-value HsStats is not used
};

// flag values (mirrors include/hs.h; csrc includes hs.h in hs_api.cu and static_asserts equality)
#define HSF_NO_FUND_SELECT 1u
#define HSF_NO_DRIFT 2u
#define HSF_ALL_HARMONICS 4u
#define HSF_ALL_ORDERS 8u

#define HS_NEG_INF (__int_as_float(0xff800000))

// eq. 2 term in the library's fp32 form
__device__ __forceinline__ float hs_snr(float sum, float nmis, float inv_sigma) {
    return __fmaf_rn(sum, inv_sigma, nmis);
}

// streaming (evict-first) stores for the outputs: they are written once and never re-read, and
// must not push the L2-resident spectrum out
__device__ __forceinline__ void st_cs(float* p, float v) { __stcs(p, v); }
__device__ __forceinline__ void st_cs(int* p, int v) { __stcs(p, v); }
__device__ __forceinline__ void st_cs(unsigned* p, unsigned v) { __stcs(p, v); }

// Per-spectrum statistics (hs_run_*_dstats): the CTA forms the two constants of spectrum s from d_mu / d_sigma exactly
// as the host does for the by-value statistics (IEEE reciprocal, one fp32 multiply) and keeps them in shared memory.
// Unusable entries (sigma <= 0, NaN or infinite; mu NaN or infinite) are replaced by (mu, sigma) = (0, 1).
// Must be called by every thread of the CTA.
__device__ __forceinline__ void hs_load_dstats(HsStats& s_st, const HsIO& io, int s, int H) {
    if (threadIdx.x < HS_MAX_H) {
        float is = 1.f, nm = 0.f;
        if ((int)threadIdx.x < H) {
            float sg = __ldg(io.d_sigma + (long long)s * H + threadIdx.x);
            float mu = __ldg(io.d_mu + (long long)s * H + threadIdx.x);
            // the host path rejects such statistics (fill_stats); device arrays are never read on the host, so an
            // order whose sigma is not a positive finite number or whose mu is not finite is normalised with (0, 1)
            // -- what hs_stats_finish_kernel writes for an order without samples -- in every kernel alike
            if (!(sg > 0.f) || !(sg < __int_as_float(0x7f800000)) || !(fabsf(mu) < __int_as_float(0x7f800000))) { sg = 1.f; mu = 0.f; }
            is = __fdiv_rn(1.0f, sg);
            nm = -__fmul_rn(mu, is);
        }
        s_st.inv_sigma[threadIdx.x] = is;
        s_st.nmis[threadIdx.x] = nm;
    }
    __syncthreads();
}
