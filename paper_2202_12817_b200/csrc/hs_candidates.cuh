// Candidate list (reading R11: every (spectrum, bin) whose maximum SNR reaches the threshold,
// with its harmonic count; the step after the harmonic sum, "only the highest SNR value is
// returned for each element n" -> candidate selection).
//
// One streaming pass over the snr array (16-byte loads); best_h is read for the hits only.  The hits of a
// warp are appended with ONE atomic per warp (shuffle prefix sum of the per-thread hit counts), so the pass
// stays HBM-bound at any hit density.  The order of the list is unspecified.
#pragma once
#include "hs_common.cuh"

struct HsCandidate {       // == hs_candidate (hs.h)
    int spectrum;
    int bin;
    float snr;
    int best_h;
};

template <int BLOCK>
__global__ void __launch_bounds__(BLOCK)
hs_candidates_kernel(const float* __restrict__ snr, const int* __restrict__ best_h, long long out_stride, int n_fund, int s0,
                     float threshold, HsCandidate* __restrict__ out, unsigned long long capacity,
                     unsigned long long* __restrict__ count) {
    const int s = blockIdx.y;
    const float* __restrict__ row = snr + (long long)s * out_stride;
    const int* __restrict__ brow = best_h + (long long)s * out_stride;
    const int lane = threadIdx.x & 31;
    const int n4 = (n_fund + 3) >> 2;
    for (int q0 = blockIdx.x * BLOCK; q0 < n4; q0 += gridDim.x * BLOCK) {      // warp-uniform trip count
        const int q = q0 + threadIdx.x;
        const int n = 4 * q;
        float v[4] = {0.f, 0.f, 0.f, 0.f};
        unsigned hit = 0;
        if (q < n4) {
            if (n + 3 < n_fund) {
                const float4 t = __ldcs(reinterpret_cast<const float4*>(row + n));
                v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
            } else {
#pragma unroll
                for (int e = 0; e < 4; ++e) if (n + e < n_fund) v[e] = __ldcs(row + n + e);
            }
#pragma unroll
            for (int e = 0; e < 4; ++e) hit |= (n + e < n_fund && v[e] >= threshold) ? (1u << e) : 0u;
        }
        if (__any_sync(0xffffffffu, hit != 0)) {
            const int c = __popc(hit);
            int incl = c;                                                      // inclusive prefix sum over the warp
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += t;
            }
            const int total = __shfl_sync(0xffffffffu, incl, 31);
            unsigned long long base = 0;
            if (lane == 0) base = atomicAdd(count, (unsigned long long)total);
            base = __shfl_sync(0xffffffffu, base, 0);
            unsigned long long pos = base + (unsigned long long)(incl - c);
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                if (hit & (1u << e)) {
                    if (pos < capacity) {
                        HsCandidate cand;
                        cand.spectrum = s0 + s; cand.bin = n + e; cand.snr = v[e]; cand.best_h = __ldg(brow + n + e);
                        *reinterpret_cast<int4*>(out + pos) = *reinterpret_cast<const int4*>(&cand);
                    }
                    ++pos;
                }
            }
        }
    }
}
