// Greedy harmonic sum (Alg. 2), band-specialised, over a 1-bit comparison mask.
//
// The greedy decision at order h, "is x[m+1] > x[m]" with m = h n + d (eq. 5, PAPER.md:182;
// PAPER.md:240-244), depends on the spectrum alone, not on the sums.  So
//
//   hs_cmp_mask_kernel    streams a spectrum once (float4, coalesced) and writes
//                         c[m] = (x[m+1] > x[m]), one bit per bin (c[N-1] = 0: a missing second bin
//                         never wins, reading R4).  The fundamentals of the TOP BAND, 2 n > N-1,
//                         have a single order, whose two bins this kernel already holds: it writes
//                         their outputs (half of all bins) as 16-byte stores.
//   hs_greedy_band_kernel the other fundamentals.  Orders 1..HD: the direct form (read x[m], x[m+1],
//                         keep the larger) -- the spans are dense there.  Orders above HD:
//                         (1) the rest of the drift path from the mask alone,
//                             bit h-1 of `path` = c[h n + d_{h-1}],  d_h = popc(path & (2^h - 1));
//                         (2) ONE load per order of the selected bin x[h n + d_h],
//                             all loads of a batch of orders independent of one another;
//                         then accumulate / normalise / max in order.
//
// Why (profiles/r01b_machine_model.md): a B200 SM takes one 128-byte line request per clock from
// the LSU whether it hits L1 or not, and at order h >= 32 every lane of a warp is in its own line.
// The direct form issues two requests per order and must wait for them before it knows the next
// address; the mask form issues one, and turns the chain of H dependent L2 round trips into a
// chain of cheap bit look-ups followed by independent loads.  The mask of the spectra in flight is
// a few MiB and lives in L2.
#pragma once
#include "hs_common.cuh"

// min(cap, a / b) for 0 <= a < 2^31, 1 <= b < 2^31, 0 <= cap <= 64, without the integer-division sequence
__device__ __forceinline__ int hs_div_cap(int a, int b, int cap) {
    const float q = __fdividef((float)a, (float)b);               // within 1 of the quotient when it is <= 64
    int h = min(cap, (int)fminf(q, 65.f));
    if ((unsigned long long)(unsigned)h * (unsigned)b > (unsigned)a) --h;
    else if (h < cap && (unsigned long long)(unsigned)(h + 1) * (unsigned)b <= (unsigned)a) ++h;
    return h;
}

// c[m] for one chunk of spectra, plus the outputs of the top band [n_top, n_fund).
// Thread t of a warp owns bins 4t..4t+3 of a 128-bin group; the 8 nibbles of a 32-bin word are
// OR-reduced inside their 8-lane group.  grid = (ceil(mask_stride / (BLOCK/8)), spectra).
template <int BLOCK, bool FUND_SELECT, bool WANT_PATH>
__global__ void __launch_bounds__(BLOCK)
hs_cmp_mask_kernel(const __grid_constant__ HsShape sh, const __grid_constant__ HsStats st, HsIO io,
                   unsigned* __restrict__ mask, int mask_stride, int n_top) {
    const int s = blockIdx.y;
    const int N = (int)sh.n_bins;
    const float* __restrict__ x = io.x + (long long)s * sh.in_stride;
    const int lane = threadIdx.x & 31;
    const int b0 = (blockIdx.x * BLOCK + threadIdx.x) * 4;          // first bin of this thread
    float v[5] = {0.f, 0.f, 0.f, 0.f, 0.f};
    if (b0 + 3 < N) {
        const float4 t = __ldg(reinterpret_cast<const float4*>(x + b0));
        v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
    } else {
        if (b0 < N) v[0] = __ldg(x + b0);
        if (b0 + 1 < N) v[1] = __ldg(x + b0 + 1);
        if (b0 + 2 < N) v[2] = __ldg(x + b0 + 2);
    }
    v[4] = __shfl_down_sync(0xffffffffu, v[0], 1);
    if (lane == 31) v[4] = (b0 + 4 < N) ? __ldg(x + b0 + 4) : 0.f;
    unsigned nib = 0;
#pragma unroll
    for (int e = 0; e < 4; ++e) nib |= (b0 + e + 1 < N && v[e + 1] > v[e]) ? (1u << e) : 0u;
    unsigned w = nib << (4 * (lane & 7));
    w |= __shfl_xor_sync(0xffffffffu, w, 1);
    w |= __shfl_xor_sync(0xffffffffu, w, 2);
    w |= __shfl_xor_sync(0xffffffffu, w, 4);
    const int word = (blockIdx.x * BLOCK + threadIdx.x) >> 3;
    if ((lane & 7) == 0 && word < mask_stride) mask[(long long)s * mask_stride + word] = w;

    // ---- top band: order 1 is the only order (PAPER.md:228-234 with mu[0], sigma[0]) ----
    const int n_fund = (int)sh.n_fund;
    if (b0 + 3 >= n_top && b0 < n_fund) {
        float snr[4];
        unsigned pb[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const bool shift = FUND_SELECT && ((nib >> e) & 1u);
            snr[e] = hs_snr(shift ? v[e + 1] : v[e], st.nmis[0], st.inv_sigma[0]);
            pb[e] = shift ? 1u : 0u;
        }
        const long long o = (long long)s * sh.out_stride + b0;
        if (b0 >= n_top && b0 + 3 < n_fund) {
            __stcs(reinterpret_cast<float4*>(io.snr + o), make_float4(snr[0], snr[1], snr[2], snr[3]));
            __stcs(reinterpret_cast<int4*>(io.best_h + o), make_int4(1, 1, 1, 1));
            if (WANT_PATH) __stcs(reinterpret_cast<uint4*>(io.path + o), make_uint4(pb[0], pb[1], pb[2], pb[3]));
        } else {
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                if (b0 + e >= n_top && b0 + e < n_fund) {
                    st_cs(io.snr + o + e, snr[e]);
                    st_cs(io.best_h + o + e, 1);
                    if (WANT_PATH) st_cs(io.path + o + e, pb[e]);
                }
            }
        }
    }
}

// One order of the direct form for the R fundamentals of a thread (h compile-time, inside the band
// for the whole tile: m + 1 <= N - 1).
template <int h, int R, bool FUND_SELECT>
__device__ __forceinline__ void hs_gb_direct(const float* __restrict__ x, const HsStats& st, const unsigned (&n)[R],
                                             unsigned (&m)[R], unsigned (&path)[R], float (&sum)[R], float (&best)[R],
                                             int (&bh)[R]) {
    float a[R], b[R];
#pragma unroll
    for (int j = 0; j < R; ++j) {
        m[j] += n[j];
        a[j] = __ldg(x + m[j]);
        b[j] = __ldg(x + m[j] + 1);
    }
#pragma unroll
    for (int j = 0; j < R; ++j) {
        bool shift = b[j] > a[j];                                   // strict >: ties stay
        if (!FUND_SELECT && h == 1) shift = false;
        m[j] += shift;
        path[j] |= (unsigned)shift << (h - 1);
        sum[j] = __fadd_rn(sum[j], shift ? b[j] : a[j]);
        const float snr = hs_snr(sum[j], st.nmis[h - 1], st.inv_sigma[h - 1]);
        if (snr > best[j]) { best[j] = snr; bh[j] = h; }
    }
}

// Orders H0+1 .. H0+CNT from the resolved path: R*CNT independent loads, then the in-order
// accumulate / normalise / max.  h is compile-time, so the statistics are
// constant-bank operands and bit h-1 of the path is an immediate shift.  CHECK: some fundamentals of
// the tile stop before H0+CNT (cnt[j] = their last evaluated order, reading R4).
template <int H0, int CNT, int R, bool CHECK>
__device__ __forceinline__ void hs_gb_batch(const float* __restrict__ x, const HsStats& st, const unsigned (&n)[R],
                                            const unsigned (&path)[R], const int (&cnt)[R], unsigned (&m)[R],
                                            float (&sum)[R], float (&best)[R], int (&bh)[R]) {
    float v[R][CNT];
#pragma unroll
    for (int j = 0; j < R; ++j) {
#pragma unroll
        for (int u = 0; u < CNT; ++u) {
            const int h = H0 + u + 1;
            m[j] += n[j] + ((path[j] >> (h - 1)) & 1u);            // m = h n + d_h: the selected bin
            v[j][u] = (!CHECK || h <= cnt[j]) ? __ldg(x + m[j]) : 0.f;
        }
    }
#pragma unroll
    for (int j = 0; j < R; ++j) {
#pragma unroll
        for (int u = 0; u < CNT; ++u) {
            const int h = H0 + u + 1;
            sum[j] = __fadd_rn(sum[j], v[j][u]);
            const float snr = hs_snr(sum[j], st.nmis[h - 1], st.inv_sigma[h - 1]);
            if ((!CHECK || h <= cnt[j]) && snr > best[j]) { best[j] = snr; bh[j] = h; }
        }
    }
}

template <int H0, int CNT, int R>
__device__ __forceinline__ void hs_gb_batch_any(int h_safe, const float* __restrict__ x, const HsStats& st,
                                                const unsigned (&n)[R], const unsigned (&path)[R], const int (&cnt)[R],
                                                unsigned (&m)[R], float (&sum)[R], float (&best)[R], int (&bh)[R]) {
    if (H0 + CNT <= h_safe) hs_gb_batch<H0, CNT, R, false>(x, st, n, path, cnt, m, sum, best, bh);
    else hs_gb_batch<H0, CNT, R, true>(x, st, n, path, cnt, m, sum, best, bh);
}

// Shared-memory copy of the mask bits a tile of T fundamentals can look at.  Order h reads bins
// [h f0, h (f0 + T - 1) + h - 1]: the words from w0(h) = ((h f0) >> 5) & ~3 on, at most h T/32 + 6 of
// them.  Order h owns the fixed slot [off(h), off(h) + h T/32 + 8) words.
template <int T>
__host__ __device__ constexpr int hs_gb_off(int h) { return (T / 32) * (h * (h - 1) / 2) + 8 * (h - 1); }
template <int T>
__host__ __device__ constexpr int hs_gb_slot(int h) { return (T / 32) * h + 8; }

__device__ __forceinline__ unsigned hs_gb_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

// the body for a tile whose first HD orders are direct (HD = 0: every order goes through the mask)
template <int BLOCK, int R, int HD, bool FUND_SELECT, bool WANT_PATH>
__device__ __forceinline__ void hs_gb_tile(const HsShape& sh, const HsStats& st, const HsIO& io,
                                           const float* __restrict__ x, const unsigned* __restrict__ c, int s, int f0,
                                           int n_end, int n_hi, int h_safe, int h_top, unsigned* __restrict__ sbits,
                                           unsigned long long* bar) {
    constexpr int T = BLOCK * R;
    const unsigned last = (unsigned)sh.n_bins - 1u;
    // ---- stage the mask spans of orders HD+1..h_top: one 1-D bulk async copy per order (lane = order) ----
    if (h_top > HD && threadIdx.x < 32) {
        if (threadIdx.x == 0) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" :: "r"(hs_gb_smem_u32(bar)) : "memory");
            asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
            const unsigned total = 4u * (unsigned)(hs_gb_off<T>(h_top + 1) - hs_gb_off<T>(HD + 1));
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" :: "r"(hs_gb_smem_u32(bar)), "r"(total) : "memory");
        }
        __syncwarp();
        const int h = HD + 1 + (int)threadIdx.x;
        if (h <= h_top) {
            const unsigned w0 = (((unsigned)h * (unsigned)f0) >> 5) & ~3u;
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
                         :: "r"(hs_gb_smem_u32(sbits + hs_gb_off<T>(h))), "l"(c + w0), "r"(4u * (unsigned)hs_gb_slot<T>(h)),
                            "r"(hs_gb_smem_u32(bar)) : "memory");
        }
    }
    unsigned n[R], path[R], m[R];
    int cnt[R], bh[R];
    float sum[R], best[R];
#pragma unroll
    for (int j = 0; j < R; ++j) {
        n[j] = (unsigned)min(f0 + j * BLOCK + (int)threadIdx.x, n_hi);   // clamp: duplicate work, no OOB
        path[j] = 0; m[j] = 0; sum[j] = 0.f; best[j] = HS_NEG_INF; bh[j] = 0; cnt[j] = HD;
    }
    // ---- orders 1..HD: direct ----
    if (HD >= 1) hs_gb_direct<1, R, FUND_SELECT>(x, st, n, m, path, sum, best, bh);
    if (HD >= 2) hs_gb_direct<2, R, FUND_SELECT>(x, st, n, m, path, sum, best, bh);
    if (HD >= 3) hs_gb_direct<3, R, FUND_SELECT>(x, st, n, m, path, sum, best, bh);
    if (HD >= 4) hs_gb_direct<4, R, FUND_SELECT>(x, st, n, m, path, sum, best, bh);
    static_assert(HD <= 4, "direct orders");
    if (h_top > HD) {
        // the bulk copies (phase 0); the barrier init by thread 0 is ordered before the wait by __syncthreads
        __syncthreads();
        {
            unsigned done = 0;
            while (!done) {
                asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n selp.u32 %0, 1, 0, p;\n}\n"
                             : "=r"(done) : "r"(hs_gb_smem_u32(bar)) : "memory");
            }
        }
        // ---- pass 1: the rest of the drift path from the comparison bits ----
        unsigned q[R], mm[R];                                      // q collects the bits from the top down
#pragma unroll
        for (int j = 0; j < R; ++j) { q[j] = 0; mm[j] = m[j]; }
        int h = HD + 1;
        for (; h <= h_safe; ++h) {
            unsigned w[R];
            const int base = hs_gb_off<T>(h) - (int)((((unsigned)h * (unsigned)f0) >> 5) & ~3u);
#pragma unroll
            for (int j = 0; j < R; ++j) {
                mm[j] += n[j];
                w[j] = sbits[base + (int)(mm[j] >> 5)];
            }
#pragma unroll
            for (int j = 0; j < R; ++j) {
                unsigned t = w[j] >> (mm[j] & 31);
                if (!FUND_SELECT && HD == 0 && h == 1) t = 0;
                mm[j] += t & 1u;
                q[j] = __funnelshift_r(q[j], t, 1);
            }
        }
#pragma unroll
        for (int j = 0; j < R; ++j) cnt[j] = h - 1;
        for (; h <= h_top; ++h) {
            const int base = hs_gb_off<T>(h) - (int)((((unsigned)h * (unsigned)f0) >> 5) & ~3u);
#pragma unroll
            for (int j = 0; j < R; ++j) {
                mm[j] += n[j];
                unsigned t = 0;
                if (mm[j] <= last) {                               // once false it stays false: m only grows
                    t = sbits[base + (int)(mm[j] >> 5)] >> (mm[j] & 31);   // c[last] = 0
                    if (!FUND_SELECT && HD == 0 && h == 1) t = 0;
                    mm[j] += t & 1u;
                    cnt[j] = h;
                } else {
                    mm[j] = last + 1u;                             // stays out of range, cannot wrap
                }
                q[j] = __funnelshift_r(q[j], t, 1);
            }
        }
        const int steps = h - 1 - HD;                              // >= 1: bits sit in the top `steps` positions
#pragma unroll
        for (int j = 0; j < R; ++j) path[j] |= (q[j] >> (32 - steps)) << HD;

        // ---- pass 2: one independent load per order, accumulated in order ----
        if (HD < 1) hs_gb_batch_any<0, 1, R>(h_safe, x, st, n, path, cnt, m, sum, best, bh);
        if (HD < 2 && h_top >= 2) hs_gb_batch_any<1, 1, R>(h_safe, x, st, n, path, cnt, m, sum, best, bh);
        if (HD < 3 && h_top >= 3) hs_gb_batch_any<2, 1, R>(h_safe, x, st, n, path, cnt, m, sum, best, bh);
        if (HD < 4 && h_top >= 4) hs_gb_batch_any<3, 1, R>(h_safe, x, st, n, path, cnt, m, sum, best, bh);
        if (h_top >= 5) {
            hs_gb_batch_any<4, 4, R>(h_safe, x, st, n, path, cnt, m, sum, best, bh);
            if (h_top >= 9) {
                hs_gb_batch_any<8, 8, R>(h_safe, x, st, n, path, cnt, m, sum, best, bh);
                if (h_top >= 17) {
                    hs_gb_batch_any<16, 8, R>(h_safe, x, st, n, path, cnt, m, sum, best, bh);
                    if (h_top >= 25) hs_gb_batch_any<24, 8, R>(h_safe, x, st, n, path, cnt, m, sum, best, bh);
                }
            }
        }
    }
    const long long orow = (long long)s * sh.out_stride;
#pragma unroll
    for (int j = 0; j < R; ++j) {
        const int nj = f0 + j * BLOCK + (int)threadIdx.x;
        if (nj < n_end) {
            st_cs(io.snr + orow + nj, best[j]);
            st_cs(io.best_h + orow + nj, bh[j]);
            if (WANT_PATH) st_cs(io.path + orow + nj, path[j]);
        }
    }
}

// fundamentals [0, n_end) of each spectrum of the chunk; grid = (ceil(n_end / (BLOCK R)), spectra)
template <int BLOCK, int R, int HD, bool FUND_SELECT, bool WANT_PATH>
__global__ void __launch_bounds__(BLOCK)
hs_greedy_band_kernel(const __grid_constant__ HsShape sh, const __grid_constant__ HsStats st, HsIO io,
                      const unsigned* __restrict__ mask, int mask_stride, int n_end) {
    extern __shared__ float4 hs_gb_smem4[];
    unsigned* sbits = reinterpret_cast<unsigned*>(hs_gb_smem4);
    __shared__ unsigned long long bar;
    const int s = blockIdx.y;
    const int N = (int)sh.n_bins;
    const int f0 = blockIdx.x * (BLOCK * R);
    const float* x = io.x + (long long)s * sh.in_stride;
    const unsigned* c = mask + (long long)s * mask_stride;
    // keep the row pointers as opaque 64-bit values: every access is then one IMAD.WIDE off them
    asm volatile("" : "+l"(x));
    asm volatile("" : "+l"(c));
    const int n_hi = min(f0 + BLOCK * R, n_end) - 1;              // largest fundamental of the tile
    // orders 1..h_safe: m + 1 = h n + d + 1 <= h (n + 1) <= N - 1 for every fundamental of the tile;
    // orders above h_top are outside the band for all of them
    const int h_safe = hs_div_cap(N - 1, n_hi + 1, sh.H);
    const int h_top = (f0 == 0) ? sh.H : hs_div_cap(N - 1, f0, sh.H);
    if (h_safe >= HD) hs_gb_tile<BLOCK, R, HD, FUND_SELECT, WANT_PATH>(sh, st, io, x, c, s, f0, n_end, n_hi, h_safe, h_top, sbits, &bar);
    else hs_gb_tile<BLOCK, R, 0, FUND_SELECT, WANT_PATH>(sh, st, io, x, c, s, f0, n_end, n_hi, h_safe, h_top, sbits, &bar);
}
