// C-ABI boundary (include/hs.h): plan object, argument validation, kernel selection, launches,
// and the host-buffer entry points.  No torch types, no CPU fallback.
#include "../../include/hs.h"

#include <cuda_runtime.h>
#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <new>

#include "hs_common.cuh"
#include "hs_generic.cuh"
#include "hs_greedy.cuh"
#include "hs_greedy_mask.cuh"
#include "hs_presto.cuh"
#include "hs_presto_smem.cuh"
#include "hs_presto_rows.cuh"
#include "hs_presto_farey.cuh"
#include "hs_candidates.cuh"

static_assert(HS_GREEDY_NO_FUND_SELECT == HSF_NO_FUND_SELECT, "flag mismatch");
static_assert(HS_GREEDY_NO_DRIFT == HSF_NO_DRIFT, "flag mismatch");
static_assert(HS_PRESTO_ALL_HARMONICS == HSF_ALL_HARMONICS, "flag mismatch");
static_assert(HS_PRESTO_ALL_ORDERS == HSF_ALL_ORDERS, "flag mismatch");

namespace {

// the band kernel copies fixed-size mask slots that may run past the end of the last row (never looked at)
constexpr size_t HS_MASK_SLACK_BYTES = 16384;

thread_local int32_t g_last_cuda_error = 0;

struct HostStage {          // staging for the *_host entry points (created on first use)
    bool ready = false;
    int rows = 0;           // spectra per slot
    cudaStream_t stream[2] = {nullptr, nullptr};
    float* d_in[2] = {nullptr, nullptr};
    float* d_base[2] = {nullptr, nullptr};
    float* d_snr[2] = {nullptr, nullptr};
    int32_t* d_bh[2] = {nullptr, nullptr};
    uint32_t* d_path[2] = {nullptr, nullptr};
};

}  // namespace

struct hs_plan_s {
    HsShape shape;
    uint32_t tune;
    int device;
    int sm_count;
    int64_t launches;
    HostStage stage;
    // comparison-mask scratch of the two-pass greedy kernels (hs_greedy_mask.cuh): one bit per bin for
    // the `chunk` spectra in flight, allocated by hs_plan
    unsigned* d_mask;
    int mask_stride;        // 32-bit words per spectrum (multiple of 4)
    int chunk;              // spectra per (mask, gather) launch pair: their spectra stay L2-resident
};

namespace {

hs_status cuda_fail(cudaError_t e) {
    g_last_cuda_error = (int32_t)e;
    return HS_ERR_CUDA;
}

#define HS_CUDA(call)                                   \
    do {                                                \
        cudaError_t e__ = (call);                       \
        if (e__ != cudaSuccess) return cuda_fail(e__);  \
    } while (0)

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

hs_status fill_stats(const hs_plan_s* p, const float* mu, const float* sigma, HsStats* st) {
    if (!mu || !sigma) return HS_ERR_INVALID_ARG;
    for (int h = 0; h < HS_MAX_H; ++h) { st->nmis[h] = 0.f; st->inv_sigma[h] = 1.f; }
    for (int h = 0; h < p->shape.H; ++h) {
        if (!(sigma[h] > 0.f) || !(sigma[h] < INFINITY) || !(mu[h] == mu[h])) return HS_ERR_INVALID_ARG;
        st->inv_sigma[h] = 1.0f / sigma[h];     // correctly rounded fp32 reciprocal
        st->nmis[h] = -(mu[h] * st->inv_sigma[h]);
    }
    return HS_OK;
}

int floor_log2(int v) { int l = 0; while ((2 << l) <= v) ++l; return l; }

// ------------------------------------------------------------------------------------------
// kernel selection + launch (device buffers).  `sh` may describe a sub-batch (host staging).
// ------------------------------------------------------------------------------------------
template <int BLOCK, int R>
hs_status launch_greedy_tile(hs_plan_s* p, const HsShape& sh, const HsStats& st, const HsIO& io, cudaStream_t stream) {
    const long long tile = (long long)BLOCK * R;
    dim3 grid((unsigned)((sh.n_fund + tile - 1) / tile), (unsigned)sh.n_spectra);
    const bool fs = !(sh.flags & HS_GREEDY_NO_FUND_SELECT);
    const bool wp = io.path != nullptr;
    if (io.inv_base) {
        if (fs && wp) hs_greedy_tile_kernel<BLOCK, R, true, true, true><<<grid, BLOCK, 0, stream>>>(sh, st, io);
        else if (fs && !wp) hs_greedy_tile_kernel<BLOCK, R, true, false, true><<<grid, BLOCK, 0, stream>>>(sh, st, io);
        else if (!fs && wp) hs_greedy_tile_kernel<BLOCK, R, false, true, true><<<grid, BLOCK, 0, stream>>>(sh, st, io);
        else hs_greedy_tile_kernel<BLOCK, R, false, false, true><<<grid, BLOCK, 0, stream>>>(sh, st, io);
    } else if (fs && wp) hs_greedy_tile_kernel<BLOCK, R, true, true><<<grid, BLOCK, 0, stream>>>(sh, st, io);
    else if (fs && !wp) hs_greedy_tile_kernel<BLOCK, R, true, false><<<grid, BLOCK, 0, stream>>>(sh, st, io);
    else if (!fs && wp) hs_greedy_tile_kernel<BLOCK, R, false, true><<<grid, BLOCK, 0, stream>>>(sh, st, io);
    else hs_greedy_tile_kernel<BLOCK, R, false, false><<<grid, BLOCK, 0, stream>>>(sh, st, io);
    p->launches += 1;
    HS_CUDA(cudaGetLastError());
    return HS_OK;
}

// band-specialised mask form (hs_greedy_mask.cuh): per chunk of spectra, one launch writes the comparison
// mask and the top band's outputs, one launch does the other fundamentals
template <int BLOCK, int R, int HD, bool FS, bool WP>
void launch_greedy_band_chunk(hs_plan_s* p, const HsShape& sh, const HsStats& st, const HsIO& io, int n_top, cudaStream_t stream) {
    dim3 mgrid((unsigned)((p->mask_stride + 31) / 32), (unsigned)sh.n_spectra);
    hs_cmp_mask_kernel<256, FS, WP><<<mgrid, 256, 0, stream>>>(sh, st, io, p->d_mask, p->mask_stride, n_top);
    p->launches += 1;
    const int n_end = (int)std::min<long long>(sh.n_fund, n_top);
    if (n_end > 0) {
        const int tile = BLOCK * R;
        dim3 grid((unsigned)((n_end + tile - 1) / tile), (unsigned)sh.n_spectra);
        const int smem = 4 * hs_gb_off<BLOCK * R>(sh.H + 1);      // mask spans of every order a tile can reach
        static bool attr_set = false;                             // per instantiation
        if (!attr_set) {
            cudaFuncSetAttribute(hs_greedy_band_kernel<BLOCK, R, HD, FS, WP>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 4 * hs_gb_off<BLOCK * R>(HS_MAX_H + 1));
            attr_set = true;
        }
        hs_greedy_band_kernel<BLOCK, R, HD, FS, WP><<<grid, BLOCK, smem, stream>>>(sh, st, io, p->d_mask, p->mask_stride, n_end);
        p->launches += 1;
    }
}

template <int BLOCK, int R, int HD>
hs_status launch_greedy_band(hs_plan_s* p, const HsShape& full, const HsStats& st, const HsIO& io0, cudaStream_t stream) {
    const bool fs = !(full.flags & HS_GREEDY_NO_FUND_SELECT);
    const bool wp = io0.path != nullptr;
    // fundamentals n >= n_top have exactly one order: 2 n > N - 1
    const int n_top = (full.H == 1) ? 0 : (int)((full.n_bins - 1) / 2 + 1);
    for (int s0 = 0; s0 < full.n_spectra; s0 += p->chunk) {
        HsShape sh = full;
        sh.n_spectra = std::min(p->chunk, full.n_spectra - s0);
        HsIO io = io0;
        io.x += (long long)s0 * full.in_stride;
        io.snr += (long long)s0 * full.out_stride;
        io.best_h += (long long)s0 * full.out_stride;
        if (wp) io.path += (long long)s0 * full.out_stride;
        if (fs && wp) launch_greedy_band_chunk<BLOCK, R, HD, true, true>(p, sh, st, io, n_top, stream);
        else if (fs && !wp) launch_greedy_band_chunk<BLOCK, R, HD, true, false>(p, sh, st, io, n_top, stream);
        else if (!fs && wp) launch_greedy_band_chunk<BLOCK, R, HD, false, true>(p, sh, st, io, n_top, stream);
        else launch_greedy_band_chunk<BLOCK, R, HD, false, false>(p, sh, st, io, n_top, stream);
    }
    HS_CUDA(cudaGetLastError());
    return HS_OK;
}

hs_status launch_greedy(hs_plan_s* p, const HsShape& sh, const HsStats& st, const HsIO& io, cudaStream_t stream) {
    if (sh.n_fund == 0) return HS_OK;
    if (sh.n_spectra > 65535) return HS_ERR_UNSUPPORTED;
    const bool no_drift = sh.flags & HS_GREEDY_NO_DRIFT;
    // the tile kernel keeps h n in 32 bits: h n < N + 32 * (tile of 1024 fundamentals)
    const bool fast_ok = sh.n_bins <= (1ll << 31) - (1ll << 17) && p->tune != 255 && (!no_drift || (!io.inv_base && p->tune <= 1));
    if (fast_ok && no_drift) {                              // simple harmonic sum: the tile kernel without the second bin
        const long long tile = 128 * 4;
        dim3 grid((unsigned)((sh.n_fund + tile - 1) / tile), (unsigned)sh.n_spectra);
        const bool fs = !(sh.flags & HS_GREEDY_NO_FUND_SELECT), wp = io.path != nullptr;
        if (fs && wp) hs_greedy_tile_kernel<128, 4, true, true, false, false><<<grid, 128, 0, stream>>>(sh, st, io);
        else if (fs) hs_greedy_tile_kernel<128, 4, true, false, false, false><<<grid, 128, 0, stream>>>(sh, st, io);
        else if (wp) hs_greedy_tile_kernel<128, 4, false, true, false, false><<<grid, 128, 0, stream>>>(sh, st, io);
        else hs_greedy_tile_kernel<128, 4, false, false, false, false><<<grid, 128, 0, stream>>>(sh, st, io);
        p->launches += 1;
        HS_CUDA(cudaGetLastError());
        return HS_OK;
    }
    if (fast_ok && !io.inv_base && p->d_mask && sh.n_bins <= (1ll << 30)) {
        switch (p->tune) {
            case 20: return launch_greedy_band<256, 1, 2>(p, sh, st, io, stream);
            case 21: return launch_greedy_band<256, 2, 2>(p, sh, st, io, stream);
            case 22: return launch_greedy_band<256, 4, 2>(p, sh, st, io, stream);
            case 23: return launch_greedy_band<128, 2, 2>(p, sh, st, io, stream);
            case 24: return launch_greedy_band<128, 4, 2>(p, sh, st, io, stream);
            case 25: return launch_greedy_band<256, 2, 0>(p, sh, st, io, stream);
            case 26: return launch_greedy_band<256, 2, 4>(p, sh, st, io, stream);
            case 27: return launch_greedy_band<128, 4, 4>(p, sh, st, io, stream);
            case 28: return launch_greedy_band<256, 4, 4>(p, sh, st, io, stream);
            case 29: return launch_greedy_band<512, 2, 2>(p, sh, st, io, stream);
            default: break;
        }
    }
    if (fast_ok) {
        switch (p->tune) {
            case 1: return launch_greedy_tile<256, 1>(p, sh, st, io, stream);
            case 2: return launch_greedy_tile<256, 2>(p, sh, st, io, stream);
            case 3: return launch_greedy_tile<256, 4>(p, sh, st, io, stream);
            case 4: return launch_greedy_tile<128, 1>(p, sh, st, io, stream);
            case 5: return launch_greedy_tile<128, 2>(p, sh, st, io, stream);
            case 6: return launch_greedy_tile<128, 4>(p, sh, st, io, stream);
            case 7: return launch_greedy_tile<512, 1>(p, sh, st, io, stream);
            case 8: return launch_greedy_tile<512, 2>(p, sh, st, io, stream);
            default: return launch_greedy_tile<128, 4>(p, sh, st, io, stream);
        }
    }
    dim3 grid((unsigned)((sh.n_fund + 255) / 256), (unsigned)sh.n_spectra);
    if (io.inv_base) hs_greedy_generic_kernel<true><<<grid, 256, 0, stream>>>(sh, st, io);
    else hs_greedy_generic_kernel<false><<<grid, 256, 0, stream>>>(sh, st, io);
    p->launches += 1;
    HS_CUDA(cudaGetLastError());
    return HS_OK;
}

template <int BLOCK, int R>
hs_status launch_presto_tile(hs_plan_s* p, const HsShape& sh, const HsStats& st, const HsIO& io, cudaStream_t stream) {
    const long long tile = (long long)BLOCK * R;
    dim3 grid((unsigned)((sh.n_fund + tile - 1) / tile), (unsigned)sh.n_spectra);
    switch (floor_log2(sh.H)) {
        case 0: hs_presto_tile_kernel<BLOCK, R, 0><<<grid, BLOCK, 0, stream>>>(sh, st, io); break;
        case 1: hs_presto_tile_kernel<BLOCK, R, 1><<<grid, BLOCK, 0, stream>>>(sh, st, io); break;
        case 2: hs_presto_tile_kernel<BLOCK, R, 2><<<grid, BLOCK, 0, stream>>>(sh, st, io); break;
        case 3: hs_presto_tile_kernel<BLOCK, R, 3><<<grid, BLOCK, 0, stream>>>(sh, st, io); break;
        case 4: hs_presto_tile_kernel<BLOCK, R, 4><<<grid, BLOCK, 0, stream>>>(sh, st, io); break;
        default: hs_presto_tile_kernel<BLOCK, R, 5><<<grid, BLOCK, 0, stream>>>(sh, st, io); break;
    }
    p->launches += 1;
    HS_CUDA(cudaGetLastError());
    return HS_OK;
}

template <int T, int L, int BLOCK, bool BULK>
hs_status launch_presto_smem_L(hs_plan_s* p, const HsShape& sh, const HsStats& st, const HsIO& io, cudaStream_t stream) {
    constexpr int smem = 4 * hs_presto_span_floats<L>(T);
    static bool attr_set = false;                       // per instantiation; the attribute is per device function
    if (!attr_set) {
        HS_CUDA(cudaFuncSetAttribute(hs_presto_smem_kernel<T, L, BLOCK, BULK>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        attr_set = true;
    }
    dim3 grid((unsigned)((sh.n_fund + T - 1) / T), (unsigned)sh.n_spectra);
    hs_presto_smem_kernel<T, L, BLOCK, BULK><<<grid, BLOCK, smem, stream>>>(sh, st, io);
    p->launches += 1;
    HS_CUDA(cudaGetLastError());
    return HS_OK;
}

template <int T, int BLOCK, bool BULK>
hs_status launch_presto_smem(hs_plan_s* p, const HsShape& sh, const HsStats& st, const HsIO& io, cudaStream_t stream) {
    switch (floor_log2(sh.H)) {
        case 0: return launch_presto_smem_L<T, 0, BLOCK, BULK>(p, sh, st, io, stream);
        case 1: return launch_presto_smem_L<T, 1, BLOCK, BULK>(p, sh, st, io, stream);
        case 2: return launch_presto_smem_L<T, 2, BLOCK, BULK>(p, sh, st, io, stream);
        case 3: return launch_presto_smem_L<T, 3, BLOCK, BULK>(p, sh, st, io, stream);
        case 4: return launch_presto_smem_L<T, 4, BLOCK, BULK>(p, sh, st, io, stream);
        default: return launch_presto_smem_L<T, 5, BLOCK, BULK>(p, sh, st, io, stream);
    }
}

template <int L, int W, bool BULK, int NE>
hs_status launch_presto_rows_L(hs_plan_s* p, const HsShape& sh, const HsStats& st, const HsIO& io, cudaStream_t stream) {
    constexpr int smem = 4 * hs_rows::smem_words(L, W);
    static bool attr_set = false;                       // per instantiation
    if (!attr_set) {
        HS_CUDA(cudaFuncSetAttribute(hs_presto_rows_kernel<L, W, BULK, NE>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        attr_set = true;
    }
    constexpr int T = hs_rows::WT * W;
    dim3 grid((unsigned)((sh.n_fund + T - 1) / T), (unsigned)sh.n_spectra);
    hs_presto_rows_kernel<L, W, BULK, NE><<<grid, (NE < 0 ? 64 : 32) * W, smem, stream>>>(sh, st, io);
    p->launches += 1;
    HS_CUDA(cudaGetLastError());
    return HS_OK;
}

template <int W, bool BULK, int NE>
hs_status launch_presto_rows(hs_plan_s* p, const HsShape& sh, const HsStats& st, const HsIO& io, cudaStream_t stream) {
    switch (floor_log2(sh.H)) {
        case 0: return launch_presto_rows_L<0, W, BULK, NE>(p, sh, st, io, stream);
        case 1: return launch_presto_rows_L<1, W, BULK, NE>(p, sh, st, io, stream);
        case 2: return launch_presto_rows_L<2, W, BULK, NE>(p, sh, st, io, stream);
        case 3: return launch_presto_rows_L<3, W, BULK, NE>(p, sh, st, io, stream);
        case 4: return launch_presto_rows_L<4, W, BULK, NE>(p, sh, st, io, stream);
        default: return launch_presto_rows_L<5, W, BULK, NE>(p, sh, st, io, stream);
    }
}

hs_status launch_presto(hs_plan_s* p, const HsShape& sh, const HsStats& st, const HsIO& io, cudaStream_t stream) {
    if (sh.n_fund == 0) return HS_OK;
    if (sh.n_spectra > 65535) return HS_ERR_UNSUPPORTED;
    // PRESTO_all, and PRESTO+ at H > 16 (measured: below that the coverage kernel is faster): hs_presto_farey.cuh
    if ((sh.flags & HS_PRESTO_ALL_HARMONICS) && !io.inv_base && p->tune != 255 &&
        (!(sh.flags & HS_PRESTO_ALL_ORDERS) || sh.H > 16 || p->tune == 1)) {
        dim3 fgrid((unsigned)((sh.n_fund + 255) / 256), (unsigned)sh.n_spectra);
        if (sh.flags & HS_PRESTO_ALL_ORDERS) hs_presto_farey_kernel<true><<<fgrid, 256, 0, stream>>>(sh, st, io);
        else hs_presto_farey_kernel<false><<<fgrid, 256, 0, stream>>>(sh, st, io);
        p->launches += 1;
        HS_CUDA(cudaGetLastError());
        return HS_OK;
    }
    const bool fast_ok = !io.inv_base && !(sh.flags & (HS_PRESTO_ALL_HARMONICS | HS_PRESTO_ALL_ORDERS)) &&
                         sh.n_bins * 32 < (1ll << 31) - 64 && p->tune != 255;
    if (fast_ok) {
        switch (p->tune) {
            case 1: return launch_presto_tile<256, 1>(p, sh, st, io, stream);
            case 2: return launch_presto_tile<256, 2>(p, sh, st, io, stream);
            case 3: return launch_presto_tile<256, 4>(p, sh, st, io, stream);
            case 4: return launch_presto_tile<128, 1>(p, sh, st, io, stream);
            case 5: return launch_presto_tile<128, 2>(p, sh, st, io, stream);
            case 6: return launch_presto_tile<512, 1>(p, sh, st, io, stream);
            case 7: return launch_presto_tile<256, 1>(p, sh, st, io, stream);
            case 10: return launch_presto_smem<1024, 256, true>(p, sh, st, io, stream);
            case 11: return launch_presto_smem<2048, 256, true>(p, sh, st, io, stream);
            case 12: return launch_presto_smem<1024, 256, false>(p, sh, st, io, stream);
            case 13: return launch_presto_smem<2048, 256, false>(p, sh, st, io, stream);
            case 14: return launch_presto_smem<512, 128, true>(p, sh, st, io, stream);
            case 15: return launch_presto_smem<1024, 128, true>(p, sh, st, io, stream);
            case 16: return launch_presto_smem<2048, 512, true>(p, sh, st, io, stream);
            case 30: return launch_presto_rows<4, true, 8>(p, sh, st, io, stream);
            case 31: return launch_presto_rows<2, true, 8>(p, sh, st, io, stream);
            case 33: return launch_presto_rows<2, false, 8>(p, sh, st, io, stream);
            case 50: return launch_presto_rows<2, true, -8>(p, sh, st, io, stream);
            case 35: return launch_presto_rows<2, true, 16>(p, sh, st, io, stream);

            default:                                        // measured: two warps per tile win at H >= 32 only
                if (sh.H >= 32) return launch_presto_rows<2, true, -8>(p, sh, st, io, stream);
                return launch_presto_rows<2, true, 8>(p, sh, st, io, stream);
        }
    }
    dim3 grid((unsigned)((sh.n_fund + 255) / 256), (unsigned)sh.n_spectra);
    if (io.inv_base) hs_presto_generic_kernel<true><<<grid, 256, 0, stream>>>(sh, st, io);
    else hs_presto_generic_kernel<false><<<grid, 256, 0, stream>>>(sh, st, io);
    p->launches += 1;
    HS_CUDA(cudaGetLastError());
    return HS_OK;
}

hs_status check_device_args(const hs_plan_s* p, const float* x, const float* ib, const float* snr, const int32_t* bh,
                            const uint32_t* path) {
    if (!p || !x || !snr || !bh) return HS_ERR_INVALID_ARG;
    if (!aligned16(x) || !aligned16(snr) || !aligned16(bh) || (ib && !aligned16(ib)) || (path && !aligned16(path)))
        return HS_ERR_INVALID_ARG;
    if ((const void*)x == (const void*)snr || (const void*)x == (const void*)bh || (const void*)snr == (const void*)bh)
        return HS_ERR_INVALID_ARG;
    return HS_OK;
}

// ------------------------------------------------------------------------------------------
// host staging
// ------------------------------------------------------------------------------------------
void free_stage(HostStage& g) {
    for (int i = 0; i < 2; ++i) {
        if (g.d_in[i]) cudaFree(g.d_in[i]);
        if (g.d_base[i]) cudaFree(g.d_base[i]);
        if (g.d_snr[i]) cudaFree(g.d_snr[i]);
        if (g.d_bh[i]) cudaFree(g.d_bh[i]);
        if (g.d_path[i]) cudaFree(g.d_path[i]);
        if (g.stream[i]) cudaStreamDestroy(g.stream[i]);
        g.d_in[i] = g.d_base[i] = g.d_snr[i] = nullptr; g.d_bh[i] = nullptr; g.d_path[i] = nullptr; g.stream[i] = nullptr;
    }
    g.ready = false;
}

hs_status ensure_stage(hs_plan_s* p, bool need_base, bool need_path) {
    HostStage& g = p->stage;
    const HsShape& sh = p->shape;
    if (!g.ready) {
        // slot size: about 256 MiB of input per slot, at least one spectrum
        const long long row_bytes = sh.in_stride * 4;
        long long rows = std::max(1ll, (256ll << 20) / std::max(1ll, row_bytes));
        rows = std::min<long long>(rows, sh.n_spectra);
        g.rows = (int)rows;
        for (int i = 0; i < 2; ++i) {
            if (cudaStreamCreateWithFlags(&g.stream[i], cudaStreamNonBlocking) != cudaSuccess) { free_stage(g); return HS_ERR_ALLOC; }
            if (cudaMalloc(&g.d_in[i], rows * sh.in_stride * 4) != cudaSuccess ||
                cudaMalloc(&g.d_snr[i], rows * sh.out_stride * 4) != cudaSuccess ||
                cudaMalloc(&g.d_bh[i], rows * sh.out_stride * 4) != cudaSuccess) { (void)cudaGetLastError(); free_stage(g); return HS_ERR_ALLOC; }
        }
        g.ready = true;
    }
    for (int i = 0; i < 2; ++i) {
        if (need_base && !g.d_base[i] && cudaMalloc(&g.d_base[i], (long long)g.rows * sh.in_stride * 4) != cudaSuccess) { (void)cudaGetLastError(); return HS_ERR_ALLOC; }
        if (need_path && !g.d_path[i] && cudaMalloc(&g.d_path[i], (long long)g.rows * sh.out_stride * 4) != cudaSuccess) { (void)cudaGetLastError(); return HS_ERR_ALLOC; }
    }
    return HS_OK;
}

hs_status run_host(hs_plan_s* p, bool greedy, const float* hx, const float* hb, const float* mu, const float* sigma,
                   float* hsnr, int32_t* hbh, uint32_t* hpath) {
    if (!p || !hx || !hsnr || !hbh) return HS_ERR_INVALID_ARG;
    HsStats st;
    hs_status rc = fill_stats(p, mu, sigma, &st);
    if (rc != HS_OK) return rc;
    if (!greedy && (p->shape.flags & HS_PRESTO_ALL_ORDERS) && !(p->shape.flags & HS_PRESTO_ALL_HARMONICS)) return HS_ERR_INVALID_ARG;
    HS_CUDA(cudaSetDevice(p->device));
    rc = ensure_stage(p, hb != nullptr, greedy && hpath != nullptr);
    if (rc != HS_OK) return rc;
    HostStage& g = p->stage;
    const HsShape& full = p->shape;
    hs_status result = HS_OK;
    int chunk = 0;
    for (int s0 = 0; s0 < full.n_spectra && result == HS_OK; s0 += g.rows, ++chunk) {
        const int i = chunk & 1;
        const int rows = std::min(g.rows, full.n_spectra - s0);
        cudaStream_t stm = g.stream[i];
        HsShape sh = full;
        sh.n_spectra = rows;
        // strided rows: copy only the used part of each row when strides are padded
        cudaError_t e = cudaMemcpy2DAsync(g.d_in[i], full.in_stride * 4, hx + (long long)s0 * full.in_stride, full.in_stride * 4,
                                          full.n_bins * 4, rows, cudaMemcpyHostToDevice, stm);
        if (e == cudaSuccess && hb)
            e = cudaMemcpy2DAsync(g.d_base[i], full.in_stride * 4, hb + (long long)s0 * full.in_stride, full.in_stride * 4,
                                  full.n_bins * 4, rows, cudaMemcpyHostToDevice, stm);
        if (e != cudaSuccess) { result = cuda_fail(e); break; }
        HsIO io{g.d_in[i], hb ? g.d_base[i] : nullptr, g.d_snr[i], g.d_bh[i], (greedy && hpath) ? g.d_path[i] : nullptr};
        result = greedy ? launch_greedy(p, sh, st, io, stm) : launch_presto(p, sh, st, io, stm);
        if (result != HS_OK) break;
        const size_t w = (size_t)full.n_fund * 4, pitch = (size_t)full.out_stride * 4;
        e = cudaMemcpy2DAsync(hsnr + (long long)s0 * full.out_stride, pitch, g.d_snr[i], pitch, w, rows, cudaMemcpyDeviceToHost, stm);
        if (e == cudaSuccess)
            e = cudaMemcpy2DAsync(hbh + (long long)s0 * full.out_stride, pitch, g.d_bh[i], pitch, w, rows, cudaMemcpyDeviceToHost, stm);
        if (e == cudaSuccess && greedy && hpath)
            e = cudaMemcpy2DAsync(hpath + (long long)s0 * full.out_stride, pitch, g.d_path[i], pitch, w, rows, cudaMemcpyDeviceToHost, stm);
        if (e != cudaSuccess) { result = cuda_fail(e); break; }
    }
    for (int i = 0; i < 2; ++i) {
        cudaError_t e = cudaStreamSynchronize(g.stream[i]);
        if (e != cudaSuccess && result == HS_OK) result = cuda_fail(e);
    }
    return result;
}

}  // namespace

extern "C" {

hs_status hs_plan(hs_plan_t* plan, int64_t n_bins, int32_t n_spectra, int32_t H, int64_t in_stride, int64_t out_stride,
                  int64_t n_fund, uint32_t flags, int32_t device) {
    if (!plan) return HS_ERR_INVALID_ARG;
    *plan = nullptr;
    if (n_bins < 2 || n_bins > (1ll << 31) - 64 || n_spectra < 1 || H < 1 || H > HS_MAX_H) return HS_ERR_INVALID_ARG;
    if (n_fund < 0 || n_fund > n_bins) return HS_ERR_INVALID_ARG;
    if (n_fund == 0) n_fund = n_bins;
    if (in_stride == 0) in_stride = (n_bins + 3) & ~3ll;
    if (out_stride == 0) out_stride = (n_fund + 3) & ~3ll;
    if (in_stride < n_bins || out_stride < n_fund || (in_stride & 3) || (out_stride & 3)) return HS_ERR_INVALID_ARG;
    const uint32_t known = HS_GREEDY_NO_FUND_SELECT | HS_GREEDY_NO_DRIFT | HS_PRESTO_ALL_HARMONICS | HS_PRESTO_ALL_ORDERS | HS_TUNE_MASK | HS_CHUNK_MASK;
    if (flags & ~known) return HS_ERR_INVALID_ARG;
    if ((flags & HS_PRESTO_ALL_ORDERS) && !(flags & HS_PRESTO_ALL_HARMONICS)) return HS_ERR_INVALID_ARG;
    if (device < 0) return HS_ERR_INVALID_ARG;
    int count = 0;
    HS_CUDA(cudaGetDeviceCount(&count));
    if (device >= count) return HS_ERR_INVALID_ARG;
    int sms = 0;
    HS_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device));
    hs_plan_s* p = new (std::nothrow) hs_plan_s();
    if (!p) return HS_ERR_ALLOC;
    p->shape.n_bins = n_bins;
    p->shape.n_fund = n_fund;
    p->shape.in_stride = in_stride;
    p->shape.out_stride = out_stride;
    p->shape.n_spectra = n_spectra;
    p->shape.H = H;
    p->shape.flags = flags & ~(HS_TUNE_MASK | HS_CHUNK_MASK);
    p->tune = (flags & HS_TUNE_MASK) >> HS_TUNE_SHIFT;
    p->device = device;
    p->sm_count = sms;
    p->launches = 0;
    p->d_mask = nullptr;
    p->mask_stride = 0;
    p->chunk = 0;
    if (n_bins <= (1ll << 30) && !(flags & HS_GREEDY_NO_DRIFT)) {
        // spectra per launch pair: keep the chunk's spectra (and the outputs streaming past them) inside L2
        int l2 = 0;
        cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, device);
        const long long row_bytes = in_stride * 4;
        long long chunk = (flags & HS_CHUNK_MASK) >> HS_CHUNK_SHIFT;
        if (chunk == 0) chunk = std::max(1ll, std::min(8ll, ((long long)l2 / 2) / std::max(1ll, row_bytes)));
        chunk = std::min<long long>(chunk, n_spectra);
        p->chunk = (int)chunk;
        p->mask_stride = (int)((((n_bins + 31) / 32) + 3) & ~3ll);
        cudaError_t e = cudaSetDevice(device);
        if (e == cudaSuccess) e = cudaMalloc(&p->d_mask, (size_t)p->chunk * p->mask_stride * 4 + HS_MASK_SLACK_BYTES);
        if (e == cudaSuccess) e = cudaMemset(p->d_mask, 0, (size_t)p->chunk * p->mask_stride * 4 + HS_MASK_SLACK_BYTES);
        if (e != cudaSuccess) { (void)cudaGetLastError(); delete p; return HS_ERR_ALLOC; }
    }
    *plan = p;
    return HS_OK;
}

hs_status hs_run_greedy(hs_plan_t plan, const float* d_spectra, const float* d_inv_baseline, const float* mu,
                        const float* sigma, float* d_snr, int32_t* d_best_h, uint32_t* d_path, void* cuda_stream) {
    hs_status rc = check_device_args(plan, d_spectra, d_inv_baseline, d_snr, d_best_h, d_path);
    if (rc != HS_OK) return rc;
    HsStats st;
    rc = fill_stats(plan, mu, sigma, &st);
    if (rc != HS_OK) return rc;
    HsIO io{d_spectra, d_inv_baseline, d_snr, d_best_h, d_path};
    return launch_greedy(plan, plan->shape, st, io, (cudaStream_t)cuda_stream);
}

hs_status hs_run_presto(hs_plan_t plan, const float* d_spectra, const float* d_inv_baseline, const float* mu,
                        const float* sigma, float* d_snr, int32_t* d_best_h, void* cuda_stream) {
    hs_status rc = check_device_args(plan, d_spectra, d_inv_baseline, d_snr, d_best_h, nullptr);
    if (rc != HS_OK) return rc;
    HsStats st;
    rc = fill_stats(plan, mu, sigma, &st);
    if (rc != HS_OK) return rc;
    HsIO io{d_spectra, d_inv_baseline, d_snr, d_best_h, nullptr};
    return launch_presto(plan, plan->shape, st, io, (cudaStream_t)cuda_stream);
}

hs_status hs_run_greedy_host(hs_plan_t plan, const float* h_spectra, const float* h_inv_baseline, const float* mu,
                             const float* sigma, float* h_snr, int32_t* h_best_h, uint32_t* h_path) {
    return run_host(plan, true, h_spectra, h_inv_baseline, mu, sigma, h_snr, h_best_h, h_path);
}

hs_status hs_run_presto_host(hs_plan_t plan, const float* h_spectra, const float* h_inv_baseline, const float* mu,
                             const float* sigma, float* h_snr, int32_t* h_best_h) {
    return run_host(plan, false, h_spectra, h_inv_baseline, mu, sigma, h_snr, h_best_h, nullptr);
}

hs_status hs_find_candidates(hs_plan_t plan, const float* d_snr, const int32_t* d_best_h, float threshold,
                             hs_candidate* d_out, int64_t capacity, uint64_t* d_count, void* cuda_stream) {
    static_assert(sizeof(hs_candidate) == sizeof(HsCandidate) && sizeof(hs_candidate) == 16, "candidate layout");
    if (!plan || !d_snr || !d_best_h || !d_count || capacity < 0 || (capacity > 0 && !d_out)) return HS_ERR_INVALID_ARG;
    if (!aligned16(d_snr) || !aligned16(d_best_h) || (d_out && !aligned16(d_out)) || (reinterpret_cast<uintptr_t>(d_count) & 7u))
        return HS_ERR_INVALID_ARG;
    if (!(threshold == threshold)) return HS_ERR_INVALID_ARG;
    const HsShape& sh = plan->shape;
    if (sh.n_spectra > 65535) return HS_ERR_UNSUPPORTED;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    HS_CUDA(cudaMemsetAsync(d_count, 0, sizeof(uint64_t), stream));
    if (sh.n_fund == 0) return HS_OK;
    const long long n4 = (sh.n_fund + 3) / 4;
    // a few waves of 256-thread CTAs per spectrum row, grid-stride inside the row
    const long long per_row = std::max(1ll, std::min((n4 + 255) / 256, (long long)std::max(1, plan->sm_count * 64 / sh.n_spectra + 1)));
    dim3 grid((unsigned)per_row, (unsigned)sh.n_spectra);
    hs_candidates_kernel<256><<<grid, 256, 0, stream>>>(d_snr, d_best_h, sh.out_stride, (int)sh.n_fund, threshold,
                                                        reinterpret_cast<HsCandidate*>(d_out), (unsigned long long)capacity,
                                                        reinterpret_cast<unsigned long long*>(d_count));
    plan->launches += 1;
    HS_CUDA(cudaGetLastError());
    return HS_OK;
}

int64_t hs_launch_count(hs_plan_t plan) { return plan ? plan->launches : -1; }

hs_status hs_destroy(hs_plan_t plan) {
    if (!plan) return HS_OK;
    if (plan->stage.ready || plan->d_mask) {
        cudaSetDevice(plan->device);
        if (plan->stage.ready) free_stage(plan->stage);
        if (plan->d_mask) cudaFree(plan->d_mask);
    }
    delete plan;
    return HS_OK;
}

const char* hs_status_string(hs_status s) {
    switch (s) {
        case HS_OK: return "HS_OK";
        case HS_ERR_INVALID_ARG: return "HS_ERR_INVALID_ARG: invalid argument";
        case HS_ERR_UNSUPPORTED: return "HS_ERR_UNSUPPORTED: valid but unimplemented combination";
        case HS_ERR_ALLOC: return "HS_ERR_ALLOC: allocation failed";
        case HS_ERR_CUDA: return "HS_ERR_CUDA: CUDA runtime error (see hs_last_cuda_error)";
    }
    return "unknown hs_status";
}

int32_t hs_last_cuda_error(void) { return g_last_cuda_error; }

}  // extern "C"
