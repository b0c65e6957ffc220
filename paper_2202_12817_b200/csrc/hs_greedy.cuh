// Tuned greedy harmonic sum (Alg. 2) for the common configuration:
// drift tracking on (or off: the simple sum), in-row indices < 2^31.
//
// Mapping: a CTA owns a tile of R*BLOCK consecutive fundamentals of
// one spectrum; thread t runs R independent chains, chain j on fundamental f0 + j*BLOCK + t, so
// that the 32 lanes of a warp always hold 32 consecutive fundamentals: at order h their pairs
// x[m], x[m+1] (m = h n + d, eq. 5) sit in the contiguous span [h n0, h (n0+32) + h]
// and the gather is served at 32-byte sector granularity out of L1/L2.  The grid is
// spectrum-major (blockIdx.y = spectrum) so a spectrum is swept while it is L2-resident:
// every bin b is re-read at order h by the fundamentals near b/h.
// The R chains give the memory system R independent dependent-load chains per thread.
//
// Tile order inside a spectrum (MIX): consecutive CTAs take tiles from 16 equally wide bands of
// fundamentals in turn (8 of every 16 from the one-order top band, which only streams HBM; one from
// the lowest sixteenth, which gathers all H orders out of L2), so that every SM holds a mix of
// HBM-bound and L2-bound tiles at any moment instead of running the two kinds one after the other.
//
// Addressing: the chain keeps the BYTE offset of x[m] inside the row in one 32-bit register
// (4 m < 2^33 does not fit: the offset is kept in ELEMENTS and the load address is formed by one
// IMAD.WIDE from the row pointer, which is materialised once).
#pragma once
#include "hs_common.cuh"

namespace hs_greedy {
constexpr int NBAND = 16;
// tile visited by CTA i of a spectrum with nt tiles: band i % 16, position i / 16 inside the band
__device__ __forceinline__ int mixed_tile(int i, int nt) {
    const int per = (nt + NBAND - 1) / NBAND;
    return (i % NBAND) * per + i / NBAND;               // may be >= nt: the CTA has nothing to do
}
__host__ __device__ constexpr int mixed_grid(int nt) { return NBAND * ((nt + NBAND - 1) / NBAND); }
}  // namespace hs_greedy

// HAS_BASE: every x[b] is the fp32 product x[b] * inv_baseline[b] (reading R13; cfg4's whitening multiplier).
// DRIFT = false: the simple harmonic sum (eq. 3; HS_GREEDY_NO_DRIFT): the second bin is never read.
// DSTATS: per-spectrum statistics from device memory (hs_run_greedy_dstats) instead of the by-value ones.
template <int BLOCK, int R, bool FUND_SELECT, bool WANT_PATH, bool HAS_BASE = false, bool DRIFT = true, bool MIX = true, bool DSTATS = false>
__global__ void __launch_bounds__(BLOCK, (R == 4) ? 1536 / BLOCK : 1)
hs_greedy_tile_kernel(const __grid_constant__ HsShape sh, const __grid_constant__ HsStats st_param, HsIO io) {
    const int s = blockIdx.y;
    __shared__ HsStats s_st;
    if (DSTATS) hs_load_dstats(s_st, io, s, sh.H);
    const HsStats& st = DSTATS ? s_st : st_param;
    const int N = (int)sh.n_bins;
    const int last = N - 1;
    const int n_fund = (int)sh.n_fund;
    int tile = blockIdx.x;
    if (MIX) {
        const int nt = (n_fund + BLOCK * R - 1) / (BLOCK * R);
        tile = hs_greedy::mixed_tile(blockIdx.x, nt);
        if (tile >= nt) return;
    }
    const int f0 = tile * (BLOCK * R);
    const float* x = io.x + (long long)s * sh.in_stride;
    const float* ib = HAS_BASE ? io.inv_base + (long long)s * sh.in_stride : nullptr;
    asm volatile("" : "+l"(x));                                  // one materialised row pointer for all the loads
    if (HAS_BASE) asm volatile("" : "+l"(ib));

    // Orders 1..h_safe need no band-edge test for any fundamental of the tile:
    // m + 1 = h n + d + 1 <= h (n + 1) + 1 <= last.   Orders above h_top are dead for all of them.
    const int n_hi = min(f0 + BLOCK * R, n_fund) - 1;           // largest fundamental of the tile
    const int H = sh.H;
    int h_safe = (last - 1) / (n_hi + 1);
    h_safe = min(h_safe, H);
    const int h_top = (f0 == 0) ? H : min(H, last / f0);

    // ---- top band: order 1 is the only order of every fundamental of the tile (2 f0 > N - 1): pure streaming.
    // A thread takes 4 consecutive bins: one 16-byte load, the neighbour's first word by shuffle, 16-byte stores.
    if (!HAS_BASE && h_top == 1 && f0 + BLOCK * R <= n_fund && f0 + BLOCK * R + 1 <= N && (BLOCK * R) % 256 == 0) {
        const long long orow = (long long)s * sh.out_stride;
        const bool al32 = (((reinterpret_cast<uintptr_t>(x + f0)) | reinterpret_cast<uintptr_t>(io.snr + orow + f0) |
                            reinterpret_cast<uintptr_t>(io.best_h + orow + f0) | (WANT_PATH ? reinterpret_cast<uintptr_t>(io.path + orow + f0) : 0)) & 31u) == 0;
        if (al32) {
            // 8 consecutive bins per thread: one 32-byte load, the neighbour's first word by shuffle, 32-byte stores
            // (whole sectors per lane: 6.9 TB/s against 6.2 for 16-byte stores, profiles/r02_machine_model.md)
            if (threadIdx.x < BLOCK * R / 8) {                      // whole warps: BLOCK R / 8 is a multiple of 32
                const int n0 = f0 + 8 * threadIdx.x;
                float e[9];
                asm volatile("ld.global.cs.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n"
                             : "=f"(e[0]), "=f"(e[1]), "=f"(e[2]), "=f"(e[3]), "=f"(e[4]), "=f"(e[5]), "=f"(e[6]), "=f"(e[7]) : "l"(x + n0));
                e[8] = __shfl_down_sync(0xffffffffu, e[0], 1);
                if ((threadIdx.x & 31) == 31) e[8] = __ldg(x + n0 + 8);
                float snr[8];
                unsigned pb[8];
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    const bool shift = FUND_SELECT && DRIFT && e[k + 1] > e[k];  // strict >: ties stay
                    snr[k] = hs_snr(shift ? e[k + 1] : e[k], st.nmis[0], st.inv_sigma[0]);
                    pb[k] = shift ? 1u : 0u;
                }
                const long long o = orow + n0;
                asm volatile("st.global.cs.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};\n" :: "l"(io.snr + o), "f"(snr[0]), "f"(snr[1]), "f"(snr[2]),
                             "f"(snr[3]), "f"(snr[4]), "f"(snr[5]), "f"(snr[6]), "f"(snr[7]) : "memory");
                asm volatile("st.global.cs.v8.s32 [%0], {%1,%1,%1,%1,%1,%1,%1,%1};\n" :: "l"(io.best_h + o), "r"(1) : "memory");
                if (WANT_PATH)
                    asm volatile("st.global.cs.v8.u32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};\n" :: "l"(io.path + o), "r"(pb[0]), "r"(pb[1]), "r"(pb[2]),
                                 "r"(pb[3]), "r"(pb[4]), "r"(pb[5]), "r"(pb[6]), "r"(pb[7]) : "memory");
            }
            return;
        }
        if (threadIdx.x < BLOCK * R / 4) {                          // rows on odd 16-byte units: 16-byte loads and stores
            const int n0 = f0 + 4 * threadIdx.x;
            const float4 v = __ldcs(reinterpret_cast<const float4*>(x + n0));      // last use of these bins: evict first
            float nxt = __shfl_down_sync(0xffffffffu, v.x, 1);
            if ((threadIdx.x & 31) == 31) nxt = __ldg(x + n0 + 4);
            const float e[5] = {v.x, v.y, v.z, v.w, nxt};
            float snr[4];
            unsigned pb[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const bool shift = FUND_SELECT && DRIFT && e[k + 1] > e[k];  // strict >: ties stay
                snr[k] = hs_snr(shift ? e[k + 1] : e[k], st.nmis[0], st.inv_sigma[0]);
                pb[k] = shift ? 1u : 0u;
            }
            const long long o = orow + n0;
            __stcs(reinterpret_cast<float4*>(io.snr + o), make_float4(snr[0], snr[1], snr[2], snr[3]));
            __stcs(reinterpret_cast<int4*>(io.best_h + o), make_int4(1, 1, 1, 1));
            if (WANT_PATH) __stcs(reinterpret_cast<uint4*>(io.path + o), make_uint4(pb[0], pb[1], pb[2], pb[3]));
        }
        return;
    }

    // chain state: m = element offset of x[h n + d] (advanced by n per order, by 1 per shift)
    unsigned n[R], m[R];
    int bh[R];
    float sum[R], best[R];
    unsigned path[R];
    bool live[R];
#pragma unroll
    for (int j = 0; j < R; ++j) {
        const int nj = f0 + j * BLOCK + threadIdx.x;
        live[j] = nj < n_fund;
        n[j] = live[j] ? nj : n_hi;                              // clamp: harmless duplicate work, no OOB
        m[j] = 0; bh[j] = 0; sum[j] = 0.f; best[j] = HS_NEG_INF; path[j] = 0;
    }

    int h = 1;
    // ---- unchecked orders ----
#pragma unroll 2
    for (; h <= h_safe; ++h) {
        const float nmis = st.nmis[h - 1], is = st.inv_sigma[h - 1];
        float a[R], b[R];
#pragma unroll
        for (int j = 0; j < R; ++j) {
            m[j] += n[j];
            const float* p = x + m[j];
            a[j] = __ldg(p);
            if (HAS_BASE) a[j] = __fmul_rn(a[j], __ldg(ib + m[j]));
            b[j] = HS_NEG_INF;
            if (DRIFT) {
                b[j] = __ldg(p + 1);
                if (HAS_BASE) b[j] = __fmul_rn(b[j], __ldg(ib + m[j] + 1));
            }
        }
#pragma unroll
        for (int j = 0; j < R; ++j) {
            bool shift = b[j] > a[j];
            if (!FUND_SELECT) shift = shift && (h != 1);
            m[j] += shift;
            sum[j] = __fadd_rn(sum[j], shift ? b[j] : a[j]);
            if (WANT_PATH) path[j] |= (unsigned)shift << (h - 1);
            const float snr = hs_snr(sum[j], nmis, is);
            if (snr > best[j]) { best[j] = snr; bh[j] = h; }
        }
    }
    // ---- orders that may cross the band edge for some fundamentals (R4) ----
    bool alive[R];
#pragma unroll
    for (int j = 0; j < R; ++j) alive[j] = true;
    for (; h <= h_top; ++h) {
        const float nmis = st.nmis[h - 1], is = st.inv_sigma[h - 1];
#pragma unroll
        for (int j = 0; j < R; ++j) {
            m[j] += n[j];                                        // < N + 32 n: no wrap (hs_api.cu limits N)
            alive[j] = alive[j] && (m[j] <= (unsigned)last);
            if (alive[j]) {
                float a = __ldg(x + m[j]);
                if (HAS_BASE) a = __fmul_rn(a, __ldg(ib + m[j]));
                float b = HS_NEG_INF;
                if (DRIFT && m[j] + 1 <= (unsigned)last && (FUND_SELECT || h != 1)) {
                    b = __ldg(x + m[j] + 1);
                    if (HAS_BASE) b = __fmul_rn(b, __ldg(ib + m[j] + 1));
                }
                const bool shift = b > a;
                m[j] += shift;
                sum[j] = __fadd_rn(sum[j], shift ? b : a);
                if (WANT_PATH) path[j] |= (unsigned)shift << (h - 1);
                const float snr = hs_snr(sum[j], nmis, is);
                if (snr > best[j]) { best[j] = snr; bh[j] = h; }
            }
        }
    }
    const long long orow = (long long)s * sh.out_stride;
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
