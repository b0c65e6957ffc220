// 2-D harmonic sums over an f-fdot plane (NEXT-4; BASELINE.json configs[4]; the paper only mentions higher-dimensional
// harmonic sums).  Reading R15: plane P[z + Z][r], z in [-Z, Z] (n_z = 2 Z + 1 rows of
// n_bins), outputs for every (z, r).
//   simple 2-D sum (HS_GREEDY_NO_DRIFT)   S_h(r, z) = sum_{k <= h} P[k z][k r]; order k exists iff k r <= N - 1 and |k z| <= Z
//   greedy 2-D (OURS: the paper has no 2-D rule)   drifts d_r, d_z >= 0; at order h the candidates are the 2 x 2 block
//       P[w .. w+1][m .. m+1], m = h r + d_r, w = h z + d_z; the largest is added (ties: the first of (m,w), (m+1,w),
//       (m,w+1), (m+1,w+1)) and the drifts follow it; path bit h-1 = r-shift, bit 16+h-1 = z-shift (H <= 16)
//   PRESTO-like 2-D   output at the TOP harmonic (r, z); terms P[Round(k z / H')][Round(k r / H')], Round half up
//       (floor((2a + b) / (2b)), also for negative z)
// The Alg. 1 form of the PRESTO-like sum runs through hs_presto_tile_kernel<.., TWOD> (hs_presto_tile.cuh): a term's
// row Round(k z / H') is the same for the whole tile, so the 1-D staging applies row by row.  This file holds the
// greedy / simple kernel and the coverage kernel of the PRESTO-like family (_all, +).
#pragma once
#include "hs_common.cuh"

// One thread runs R chains (fundamentals r = f0 + j BLOCK + t of row z): 32 consecutive r per warp, so that the
// 2 x 2 blocks of order h sit in two contiguous spans (rows w, w + 1) and the gather is served at sector granularity.
// The element offset of P[w][m] is carried incrementally: + (z stride + r) per order, + 1 per r-shift, + stride per z-shift.
template <int BLOCK, int R, bool FUND_SELECT, bool WANT_PATH, bool DRIFT>
__global__ void __launch_bounds__(BLOCK)
hs_greedy2d_kernel(const __grid_constant__ HsShape sh, const __grid_constant__ HsStats st, HsIO io) {
    // Grid: blockIdx.y = row.  Order k of row z reads rows k z, k z + 1, which no other row of CTAs in flight shares:
    // the gather comes from HBM (ncu: 15.3 GB read for a 1.7 GB plane), whatever the CTA order -- a column-major
    // order (all z of an r tile together) was measured too: 3.27 ms against 3.15 ms.
    const int zi = blockIdx.y;
    const int Z = sh.Z;
    const int z = zi - Z;
    const int N = (int)sh.n_bins, last = N - 1;
    const int f0 = blockIdx.x * (BLOCK * R);
    const long long stride = sh.in_stride;
    const float* __restrict__ P = io.x;

    // ---- tiles whose fundamentals all have order 1 only (2 r > N - 1, or 2 z (+ 1) outside the plane: 3/4 of a
    // 201 x 2^21 plane): pure streaming.  A thread takes 4 consecutive bins of rows z and z + 1: 16-byte loads, the
    // neighbour's first word by shuffle, 16-byte stores.
    const bool order1_only = (2 * f0 > last) || (z > 0 ? 2 * z > Z : 2 * z + 1 < -Z);
    if (order1_only && f0 + BLOCK * R + 1 <= N && (BLOCK * R) % 128 == 0) {
        if (threadIdx.x < BLOCK * R / 4) {                       // whole warps
            const int n0 = f0 + 4 * threadIdx.x;
            const bool two = DRIFT && FUND_SELECT;
            const bool zrow = two && z + 1 <= Z;
            const float* pa = P + (long long)zi * stride + n0;
            const float4 a4 = __ldcs(reinterpret_cast<const float4*>(pa));
            float4 b4 = make_float4(HS_NEG_INF, HS_NEG_INF, HS_NEG_INF, HS_NEG_INF);
            if (zrow) b4 = __ldg(reinterpret_cast<const float4*>(pa + stride));    // read again as row z of the next row of CTAs
            float an = __shfl_down_sync(0xffffffffu, a4.x, 1), bn = __shfl_down_sync(0xffffffffu, b4.x, 1);
            if ((threadIdx.x & 31) == 31) { an = __ldg(pa + 4); bn = zrow ? __ldg(pa + stride + 4) : HS_NEG_INF; }
            const float A[5] = {a4.x, a4.y, a4.z, a4.w, an}, B[5] = {b4.x, b4.y, b4.z, b4.w, bn};
            float snr[4];
            unsigned pb[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                float v = A[k];
                unsigned bits = 0;
                if (two) {
                    if (A[k + 1] > v) { v = A[k + 1]; bits = 1u; }                  // strict >: the first maximum stays
                    if (B[k] > v) { v = B[k]; bits = 1u << 16; }
                    if (B[k + 1] > v) { v = B[k + 1]; bits = 1u | (1u << 16); }
                }
                snr[k] = hs_snr(v, st.nmis[0], st.inv_sigma[0]);
                pb[k] = bits;
            }
            const long long o = (long long)zi * sh.out_stride + n0;
            __stcs(reinterpret_cast<float4*>(io.snr + o), make_float4(snr[0], snr[1], snr[2], snr[3]));
            __stcs(reinterpret_cast<int4*>(io.best_h + o), make_int4(1, 1, 1, 1));
            if (WANT_PATH) __stcs(reinterpret_cast<uint4*>(io.path + o), make_uint4(pb[0], pb[1], pb[2], pb[3]));
        }
        return;
    }

    int r[R], m[R], w[R], bh[R];
    long long off[R], step[R];
    float sum[R], best[R];
    unsigned path[R];
    bool live[R], alive[R];
#pragma unroll
    for (int j = 0; j < R; ++j) {
        r[j] = f0 + j * BLOCK + threadIdx.x;
        live[j] = r[j] < N;
        if (!live[j]) r[j] = last;                               // clamp: harmless duplicate work
        m[j] = 0; w[j] = 0; bh[j] = 0; sum[j] = 0.f; best[j] = HS_NEG_INF; path[j] = 0; alive[j] = true;
        off[j] = (long long)Z * stride;                          // P[0 + Z][0]
        step[j] = (long long)z * stride + r[j];
    }
    for (int h = 1; h <= sh.H; ++h) {
        const float nmis = st.nmis[h - 1], is = st.inv_sigma[h - 1];
        float c[R][4];
        bool any = false;
#pragma unroll
        for (int j = 0; j < R; ++j) {
            m[j] += r[j]; w[j] += z; off[j] += step[j];
            alive[j] = alive[j] && m[j] <= last && w[j] >= -Z && w[j] <= Z;      // once an order is skipped all later ones are
            any = any || alive[j];
            c[j][0] = c[j][1] = c[j][2] = c[j][3] = HS_NEG_INF;
            if (alive[j]) {
                const bool dr = DRIFT && (FUND_SELECT || h != 1);
                const bool r1 = dr && m[j] + 1 <= last, z1 = dr && w[j] + 1 <= Z;
                const float* p = P + off[j];
                c[j][0] = __ldg(p);
                if (r1) c[j][1] = __ldg(p + 1);
                if (z1) c[j][2] = __ldg(p + stride);
                if (r1 && z1) c[j][3] = __ldg(p + stride + 1);
            }
        }
        if (!__any_sync(0xffffffffu, any)) break;                // no chain of the warp is alive any more
#pragma unroll
        for (int j = 0; j < R; ++j) {
            if (alive[j]) {
                int pick = 0;
                float v = c[j][0];
                if (c[j][1] > v) { v = c[j][1]; pick = 1; }     // strict >: the first maximum stays
                if (c[j][2] > v) { v = c[j][2]; pick = 2; }
                if (c[j][3] > v) { v = c[j][3]; pick = 3; }
                if (pick & 1) { m[j] += 1; off[j] += 1; if (WANT_PATH) path[j] |= 1u << (h - 1); }
                if (pick & 2) { w[j] += 1; off[j] += stride; if (WANT_PATH) path[j] |= 1u << (16 + h - 1); }
                sum[j] = __fadd_rn(sum[j], v);
                const float snr = hs_snr(sum[j], nmis, is);
                if (snr > best[j]) { best[j] = snr; bh[j] = h; }
            }
        }
    }
    const long long orow = (long long)zi * sh.out_stride;
#pragma unroll
    for (int j = 0; j < R; ++j) {
        if (live[j]) {
            const long long o = orow + (f0 + j * BLOCK + threadIdx.x);
            st_cs(io.snr + o, best[j]);
            st_cs(io.best_h + o, bh[j]);
            if (WANT_PATH) st_cs(io.path + o, path[j]);
        }
    }
}

__device__ __forceinline__ int hs_round_half_up(int a, int b) {          // floor((2a + b) / (2b)), b > 0
    const int num = 2 * a + b, den = 2 * b;
    int q = num / den;
    if (num % den != 0 && num < 0) --q;
    return q;
}

// PRESTO-like 2-D family, one thread per top bin (r, z): coverage (every flag combination)
__global__ void __launch_bounds__(256)
hs_presto2d_generic_kernel(const __grid_constant__ HsShape sh, const __grid_constant__ HsStats st, HsIO io) {
    const int zi = blockIdx.y;
    const int Z = sh.Z, z = zi - Z;
    const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= sh.n_bins) return;
    const bool all_h = sh.flags & HSF_ALL_HARMONICS, all_o = sh.flags & HSF_ALL_ORDERS;
    const float* __restrict__ P = io.x;
    float best = HS_NEG_INF;
    int bh = 0;
    for (int Hp = 1; Hp <= sh.H; Hp = all_o ? Hp + 1 : Hp * 2) {
        float sum = 0.f;
        const int stepk = all_h ? 1 : 2;
        for (int k = 1; k <= Hp; k = (k == 1) ? 2 : k + stepk) {
            const int wr = hs_round_half_up(k * z, Hp);
            const int mr = hs_round_half_up(k * (int)r, Hp);
            const float v = __ldg(P + (long long)(wr + Z) * sh.in_stride + mr);
            sum = (k == 1) ? v : __fadd_rn(sum, v);
        }
        const float snr = hs_snr(sum, st.nmis[Hp - 1], st.inv_sigma[Hp - 1]);
        if (snr > best) { best = snr; bh = Hp; }
    }
    const long long o = (long long)zi * sh.out_stride + r;
    st_cs(io.snr + o, best);
    st_cs(io.best_h + o, bh);
}
