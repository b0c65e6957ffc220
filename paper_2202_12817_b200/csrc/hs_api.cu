// C-ABI boundary (include/hs.h): plan object, argument validation, kernel selection, launches,
// and the host-buffer entry points.  No torch types, no CPU fallback.
#include "../../include/hs.h"

#include <cuda_runtime.h>
#include <algorithm>
#include <atomic>
#include <cstring>
#include <new>

#include "hs_common.cuh"
#include "hs_generic.cuh"
#include "hs_greedy.cuh"
#include "hs_presto_tile.cuh"
#include "hs_presto_farey.cuh"
#include "hs_presto_plus.cuh"
#include "hs_candidates.cuh"
#include "hs_stats.cuh"
#include "hs_2d.cuh"

static_assert(HS_GREEDY_NO_FUND_SELECT == HSF_NO_FUND_SELECT, "flag mismatch");
static_assert(HS_GREEDY_NO_DRIFT == HSF_NO_DRIFT, "flag mismatch");
static_assert(HS_PRESTO_ALL_HARMONICS == HSF_ALL_HARMONICS, "flag mismatch");
static_assert(HS_PRESTO_ALL_ORDERS == HSF_ALL_ORDERS, "flag mismatch");

namespace {

thread_local int32_t g_last_cuda_error = 0;

struct HostStage {          // staging for the *_host entry points (created on first use)
    bool ready = false;
    int rows = 0;           // spectra per slot
    cudaStream_t stream[2] = {nullptr, nullptr};
    float* d_in[2] = {nullptr, nullptr};
    float* d_base[2] = {nullptr, nullptr};
    float* d_snr[2][2] = {{nullptr, nullptr}, {nullptr, nullptr}};     // [slot][form]: form 0 = first output set, 1 = second (hs_run_both_host)
    int32_t* d_bh[2][2] = {{nullptr, nullptr}, {nullptr, nullptr}};
    uint32_t* d_path[2] = {nullptr, nullptr};
    HsCandidate* d_cand = nullptr;           // hs_search_host: greedy list followed by the PRESTO list
    int64_t cand_cap = 0;
    uint64_t* d_cand_count = nullptr;        // [2]
};

}  // namespace

struct hs_plan_s {
    HsShape shape;
    uint32_t tune;          // hs_plan_set_tuning (0 = the library's choice)
    bool two_d;             // hs_plan_2d: the batch is one f-fdot plane (rows z = -Z .. Z)
    int device;
    int sm_count;
    int64_t launches;
    const char* last_kernel;   // name of the kernel variant launched last (hs_last_kernel)
    long long host_slot_bytes; // input bytes per staging slot of the *_host entry points (hs_plan_set_host_slot_bytes)
    HostStage stage;
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

// Every entry point runs on the plan's device and leaves the caller's current device as it found it.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(int device) {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != device) {
            err = cudaSetDevice(device);
            switched = (err == cudaSuccess);
        }
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
};

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device (context) setting: one opt-in per kernel
// instantiation AND device.  `done` is a per-instantiation bit set over device ordinals.
template <class K>
cudaError_t opt_in_smem(K kernel, int bytes, int device, std::atomic<uint64_t>& done) {
    const uint64_t bit = device < 64 ? (1ull << device) : 0;
    if (bit && (done.load(std::memory_order_acquire) & bit)) return cudaSuccess;
    const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess && bit) done.fetch_or(bit, std::memory_order_release);
    return e;
}

// gridDim.y carries the spectrum index and is limited to 65 535: larger batches are launched in slices
constexpr int HS_MAX_GRID_Y = 65535;
constexpr uint32_t HS_TUNE_GENERIC = 255;      // hs_plan_set_tuning: force the coverage kernels (hs_generic.cuh)
HsIO io_at(const HsIO& io, const HsShape& sh, long long s0) {
    HsIO r = io;
    r.x += s0 * sh.in_stride;
    if (r.inv_base) r.inv_base += s0 * sh.in_stride;
    r.snr += s0 * sh.out_stride;
    r.best_h += s0 * sh.out_stride;
    if (r.path) r.path += s0 * sh.out_stride;
    if (r.d_mu) { r.d_mu += s0 * sh.H; r.d_sigma += s0 * sh.H; }
    return r;
}

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
template <int BLOCK, int R, bool MIX, bool IB, bool DS>
void launch_greedy_tile_k(bool fs, bool wp, dim3 grid, const HsShape& sh, const HsStats& st, const HsIO& io, cudaStream_t stream) {
    if (fs && wp) hs_greedy_tile_kernel<BLOCK, R, true, true, IB, true, MIX, DS><<<grid, BLOCK, 0, stream>>>(sh, st, io);
    else if (fs) hs_greedy_tile_kernel<BLOCK, R, true, false, IB, true, MIX, DS><<<grid, BLOCK, 0, stream>>>(sh, st, io);
    else if (wp) hs_greedy_tile_kernel<BLOCK, R, false, true, IB, true, MIX, DS><<<grid, BLOCK, 0, stream>>>(sh, st, io);
    else hs_greedy_tile_kernel<BLOCK, R, false, false, IB, true, MIX, DS><<<grid, BLOCK, 0, stream>>>(sh, st, io);
}

template <int BLOCK, int R, bool MIX>
hs_status launch_greedy_tile(hs_plan_s* p, const HsShape& sh, const HsStats& st, const HsIO& io, cudaStream_t stream) {
    const long long tile = (long long)BLOCK * R;
    const int nt = (int)((sh.n_fund + tile - 1) / tile);
    dim3 grid((unsigned)(MIX ? hs_greedy::mixed_grid(nt) : nt), (unsigned)sh.n_spectra);
    const bool fs = !(sh.flags & HS_GREEDY_NO_FUND_SELECT);
    const bool wp = io.path != nullptr;
    if (io.inv_base && io.d_mu) launch_greedy_tile_k<BLOCK, R, MIX, true, true>(fs, wp, grid, sh, st, io, stream);
    else if (io.inv_base) launch_greedy_tile_k<BLOCK, R, MIX, true, false>(fs, wp, grid, sh, st, io, stream);
    else if (io.d_mu) launch_greedy_tile_k<BLOCK, R, MIX, false, true>(fs, wp, grid, sh, st, io, stream);
    else launch_greedy_tile_k<BLOCK, R, MIX, false, false>(fs, wp, grid, sh, st, io, stream);
    p->last_kernel = BLOCK == 128 ? (MIX ? "hs_greedy_tile_kernel<128,4,mix>" : "hs_greedy_tile_kernel<128,4>") : "hs_greedy_tile_kernel<256,4,mix>";
    p->launches += 1;
    HS_CUDA(cudaGetLastError());
    return HS_OK;
}

hs_status launch_greedy_slice(hs_plan_s* p, const HsShape& sh, const HsStats& st, const HsIO& io, cudaStream_t stream) {
    const bool no_drift = sh.flags & HS_GREEDY_NO_DRIFT;
    // the tile kernel keeps h n in 32 bits: h n < N + 32 * (tile of 1024 fundamentals)
    const bool fast_ok = sh.n_bins <= (1ll << 31) - (1ll << 17) && p->tune != HS_TUNE_GENERIC && (!no_drift || (!io.inv_base && !io.d_mu));
    if (fast_ok && no_drift) {                              // simple harmonic sum: the tile kernel without the second bin
        const long long tile = 128 * 4;
        dim3 grid((unsigned)hs_greedy::mixed_grid((int)((sh.n_fund + tile - 1) / tile)), (unsigned)sh.n_spectra);
        const bool fs = !(sh.flags & HS_GREEDY_NO_FUND_SELECT), wp = io.path != nullptr;
        if (fs && wp) hs_greedy_tile_kernel<128, 4, true, true, false, false><<<grid, 128, 0, stream>>>(sh, st, io);
        else if (fs) hs_greedy_tile_kernel<128, 4, true, false, false, false><<<grid, 128, 0, stream>>>(sh, st, io);
        else if (wp) hs_greedy_tile_kernel<128, 4, false, true, false, false><<<grid, 128, 0, stream>>>(sh, st, io);
        else hs_greedy_tile_kernel<128, 4, false, false, false, false><<<grid, 128, 0, stream>>>(sh, st, io);
        p->last_kernel = "hs_greedy_tile_kernel<128,4,mix,nodrift>";
        p->launches += 1;
        HS_CUDA(cudaGetLastError());
        return HS_OK;
    }
    if (fast_ok) {
        switch (io.d_mu ? 0u : p->tune) {
            case 3: return launch_greedy_tile<256, 4, true>(p, sh, st, io, stream);
            case 4: return launch_greedy_tile<128, 4, false>(p, sh, st, io, stream);     // tiles in ascending order (no band mix)
            default: return launch_greedy_tile<128, 4, true>(p, sh, st, io, stream);
        }
    }
    dim3 grid((unsigned)((sh.n_fund + 255) / 256), (unsigned)sh.n_spectra);
    if (io.inv_base && io.d_mu) hs_greedy_generic_kernel<true, true><<<grid, 256, 0, stream>>>(sh, st, io);
    else if (io.inv_base) hs_greedy_generic_kernel<true><<<grid, 256, 0, stream>>>(sh, st, io);
    else if (io.d_mu) hs_greedy_generic_kernel<false, true><<<grid, 256, 0, stream>>>(sh, st, io);
    else hs_greedy_generic_kernel<false><<<grid, 256, 0, stream>>>(sh, st, io);
    p->last_kernel = "hs_greedy_generic_kernel";
    p->launches += 1;
    HS_CUDA(cudaGetLastError());
    return HS_OK;
}

template <int L, int W, bool SPLIT = false>
hs_status launch_presto_tile_L(hs_plan_s* p, const HsShape& sh, const HsStats& st, const HsIO& io, cudaStream_t stream) {
    constexpr int smem = 4 * hs_tile::smem_words(L, W);
    static std::atomic<uint64_t> opted{0};              // per instantiation, one bit per device
    static std::atomic<uint64_t> opted_ds{0};
    constexpr int T = hs_tile::TILE * W;
    constexpr int NTHR = 64 * W;
    dim3 grid((unsigned)((sh.n_fund + T - 1) / T), (unsigned)sh.n_spectra);
    if (io.d_mu) {
        HS_CUDA(opt_in_smem(hs_presto_tile_kernel<L, W, true, false, SPLIT>, smem, p->device, opted_ds));
        hs_presto_tile_kernel<L, W, true, false, SPLIT><<<grid, NTHR, smem, stream>>>(sh, st, io);
    } else {
        HS_CUDA(opt_in_smem(hs_presto_tile_kernel<L, W, false, false, SPLIT>, smem, p->device, opted));
        hs_presto_tile_kernel<L, W, false, false, SPLIT><<<grid, NTHR, smem, stream>>>(sh, st, io);
    }
    p->last_kernel = W == 2 ? "hs_presto_tile_kernel<W=2>" : W == 1 ? "hs_presto_tile_kernel<W=1>" : "hs_presto_tile_kernel<W=3>";
    p->launches += 1;
    HS_CUDA(cudaGetLastError());
    return HS_OK;
}

template <int W, bool SPLIT = false>
hs_status launch_presto_tile(hs_plan_s* p, const HsShape& sh, const HsStats& st, const HsIO& io, cudaStream_t stream) {
    switch (floor_log2(sh.H)) {
        case 0: return launch_presto_tile_L<0, W, SPLIT>(p, sh, st, io, stream);
        case 1: return launch_presto_tile_L<1, W, SPLIT>(p, sh, st, io, stream);
        case 2: return launch_presto_tile_L<2, W, SPLIT>(p, sh, st, io, stream);
        case 3: return launch_presto_tile_L<3, W, SPLIT>(p, sh, st, io, stream);
        case 4: return launch_presto_tile_L<4, W, SPLIT>(p, sh, st, io, stream);
        default: return launch_presto_tile_L<5, W, SPLIT>(p, sh, st, io, stream);
    }
}

hs_status launch_presto_slice(hs_plan_s* p, const HsShape& sh, const HsStats& st, const HsIO& io, cudaStream_t stream) {
    // PRESTO_all / PRESTO+: reduced (Farey) fractions; default = the staged kernel (hs_presto_plus.cuh), tune 1 = the
    // one-thread-per-bin Farey kernel (hs_presto_farey.cuh)
    // (PRESTO+ at H <= 4 is 10 terms per bin: the coverage kernel is faster there, 70 against 56 Gbin/s on 1024 x 2^17)
    if ((sh.flags & HS_PRESTO_ALL_HARMONICS) && !io.inv_base && !io.d_mu && p->tune != HS_TUNE_GENERIC &&
        !((sh.flags & HS_PRESTO_ALL_ORDERS) && sh.H <= 4 && p->tune == 0)) {
        const bool all_o = sh.flags & HS_PRESTO_ALL_ORDERS;
        if (p->tune == 1 || (!all_o && p->tune != 2)) {          // measured: PRESTO_all 16.0 ms (Farey) against 19.6 ms (staged)
            dim3 fgrid((unsigned)((sh.n_fund + 255) / 256), (unsigned)sh.n_spectra);
            if (all_o) hs_presto_farey_kernel<true><<<fgrid, 256, 0, stream>>>(sh, st, io);
            else hs_presto_farey_kernel<false><<<fgrid, 256, 0, stream>>>(sh, st, io);
            p->last_kernel = "hs_presto_farey_kernel";
        } else {
            static std::atomic<uint64_t> opted_a{0}, opted_b{0};
            dim3 pgrid((unsigned)((sh.n_fund + hs_plus::T - 1) / hs_plus::T), (unsigned)sh.n_spectra);
            if (all_o) {
                HS_CUDA(opt_in_smem(hs_presto_plus_kernel<true>, hs_plus::smem_bytes(), p->device, opted_a));
                hs_presto_plus_kernel<true><<<pgrid, hs_plus::NT, hs_plus::smem_bytes(), stream>>>(sh, st, io);
            } else {
                HS_CUDA(opt_in_smem(hs_presto_plus_kernel<false>, hs_plus::smem_bytes(), p->device, opted_b));
                hs_presto_plus_kernel<false><<<pgrid, hs_plus::NT, hs_plus::smem_bytes(), stream>>>(sh, st, io);
            }
            p->last_kernel = "hs_presto_plus_kernel";
        }
        p->launches += 1;
        HS_CUDA(cudaGetLastError());
        return HS_OK;
    }
    const bool fast_ok = !io.inv_base && !(sh.flags & (HS_PRESTO_ALL_HARMONICS | HS_PRESTO_ALL_ORDERS)) &&
                         sh.n_bins * 32 < (1ll << 31) - 64 && p->tune != HS_TUNE_GENERIC;
    if (fast_ok) {
        switch (io.d_mu ? 0u : p->tune) {                    // measured on cfg3: W = 2 3.06 ms, W = 3 3.03 ms, W = 1 3.69 ms
            case 50: return launch_presto_tile<1>(p, sh, st, io, stream);
            case 52: return launch_presto_tile<3>(p, sh, st, io, stream);
            case 53: return launch_presto_tile<2, false>(p, sh, st, io, stream);            // one mbarrier for all spans
            default: return sh.H >= 32 ? launch_presto_tile<2, true>(p, sh, st, io, stream) : launch_presto_tile<2, false>(p, sh, st, io, stream);
        }
    }
    dim3 grid((unsigned)((sh.n_fund + 255) / 256), (unsigned)sh.n_spectra);
    if (io.inv_base && io.d_mu) hs_presto_generic_kernel<true, true><<<grid, 256, 0, stream>>>(sh, st, io);
    else if (io.inv_base) hs_presto_generic_kernel<true><<<grid, 256, 0, stream>>>(sh, st, io);
    else if (io.d_mu) hs_presto_generic_kernel<false, true><<<grid, 256, 0, stream>>>(sh, st, io);
    else hs_presto_generic_kernel<false><<<grid, 256, 0, stream>>>(sh, st, io);
    p->last_kernel = "hs_presto_generic_kernel";
    p->launches += 1;
    HS_CUDA(cudaGetLastError());
    return HS_OK;
}

// gridDim.y = spectrum: batches of more than 65 535 spectra go out in slices
hs_status launch_form(hs_plan_s* p, bool greedy, const HsShape& full, const HsStats& st, const HsIO& io0, cudaStream_t stream) {
    if (full.n_fund == 0) return HS_OK;
    for (long long s0 = 0; s0 < full.n_spectra; s0 += HS_MAX_GRID_Y) {
        HsShape sh = full;
        sh.n_spectra = (int)std::min<long long>(HS_MAX_GRID_Y, full.n_spectra - s0);
        const HsIO io = io_at(io0, full, s0);
        const hs_status rc = greedy ? launch_greedy_slice(p, sh, st, io, stream) : launch_presto_slice(p, sh, st, io, stream);
        if (rc != HS_OK) return rc;
    }
    return HS_OK;
}
hs_status launch_greedy(hs_plan_s* p, const HsShape& sh, const HsStats& st, const HsIO& io, cudaStream_t stream) {
    return launch_form(p, true, sh, st, io, stream);
}
hs_status launch_presto(hs_plan_s* p, const HsShape& sh, const HsStats& st, const HsIO& io, cudaStream_t stream) {
    return launch_form(p, false, sh, st, io, stream);
}

hs_status check_device_args(const hs_plan_s* p, const float* x, const float* ib, const float* snr, const int32_t* bh,
                            const uint32_t* path) {
    if (!p || !x || !snr || !bh) return HS_ERR_INVALID_ARG;
    if (!aligned16(x) || !aligned16(snr) || !aligned16(bh) || (ib && !aligned16(ib)) || (path && !aligned16(path)))
        return HS_ERR_INVALID_ARG;
    // no two of the arrays may share a byte: [S][in_stride] inputs, [S][out_stride] outputs (4-byte elements)
    const HsShape& sh = p->shape;
    const uintptr_t in_bytes = (uintptr_t)sh.n_spectra * (uintptr_t)sh.in_stride * 4u, out_bytes = (uintptr_t)sh.n_spectra * (uintptr_t)sh.out_stride * 4u;
    const void* ptr[5] = {x, ib, snr, bh, path};
    const uintptr_t len[5] = {in_bytes, in_bytes, out_bytes, out_bytes, out_bytes};
    for (int i = 0; i < 5; ++i)
        for (int j = std::max(i + 1, 2); j < 5; ++j) {          // inputs may alias each other (they are only read), nothing may alias an output
            if (!ptr[i] || !ptr[j]) continue;
            const uintptr_t a = reinterpret_cast<uintptr_t>(ptr[i]), b = reinterpret_cast<uintptr_t>(ptr[j]);
            if (a < b + len[j] && b < a + len[i]) return HS_ERR_INVALID_ARG;
        }
    return HS_OK;
}

// ------------------------------------------------------------------------------------------
// host staging
// ------------------------------------------------------------------------------------------
void free_stage(HostStage& g) {
    for (int i = 0; i < 2; ++i) {
        if (g.d_in[i]) cudaFree(g.d_in[i]);
        if (g.d_base[i]) cudaFree(g.d_base[i]);
        for (int f = 0; f < 2; ++f) {
            if (g.d_snr[i][f]) cudaFree(g.d_snr[i][f]);
            if (g.d_bh[i][f]) cudaFree(g.d_bh[i][f]);
            g.d_snr[i][f] = nullptr; g.d_bh[i][f] = nullptr;
        }
        if (g.d_path[i]) cudaFree(g.d_path[i]);
        if (g.stream[i]) cudaStreamDestroy(g.stream[i]);
        g.d_in[i] = g.d_base[i] = nullptr; g.d_path[i] = nullptr; g.stream[i] = nullptr;
    }
    if (g.d_cand) cudaFree(g.d_cand);
    if (g.d_cand_count) cudaFree(g.d_cand_count);
    g.d_cand = nullptr; g.d_cand_count = nullptr; g.cand_cap = 0;
    g.ready = false;
}

hs_status ensure_stage(hs_plan_s* p, bool need_base, bool need_path, bool need_second) {
    HostStage& g = p->stage;
    const HsShape& sh = p->shape;
    if (!g.ready) {
        // slot size: about 256 MiB of input per slot unless hs_plan_set_host_slot_bytes said otherwise; at least one spectrum
        const long long slot_bytes = p->host_slot_bytes;
        const long long row_bytes = sh.in_stride * 4;
        long long rows = std::max(1ll, slot_bytes / std::max(1ll, row_bytes));
        rows = std::min<long long>(rows, sh.n_spectra);
        g.rows = (int)rows;
        for (int i = 0; i < 2; ++i) {
            if (cudaStreamCreateWithFlags(&g.stream[i], cudaStreamNonBlocking) != cudaSuccess) { free_stage(g); return HS_ERR_ALLOC; }
            if (cudaMalloc(&g.d_in[i], rows * sh.in_stride * 4) != cudaSuccess ||
                cudaMalloc(&g.d_snr[i][0], rows * sh.out_stride * 4) != cudaSuccess ||
                cudaMalloc(&g.d_bh[i][0], rows * sh.out_stride * 4) != cudaSuccess) { (void)cudaGetLastError(); free_stage(g); return HS_ERR_ALLOC; }
        }
        g.ready = true;
    }
    for (int i = 0; i < 2; ++i) {
        if (need_base && !g.d_base[i] && cudaMalloc(&g.d_base[i], (long long)g.rows * sh.in_stride * 4) != cudaSuccess) { (void)cudaGetLastError(); return HS_ERR_ALLOC; }
        if (need_path && !g.d_path[i] && cudaMalloc(&g.d_path[i], (long long)g.rows * sh.out_stride * 4) != cudaSuccess) { (void)cudaGetLastError(); return HS_ERR_ALLOC; }
        if (need_second && !g.d_snr[i][1] && (cudaMalloc(&g.d_snr[i][1], (long long)g.rows * sh.out_stride * 4) != cudaSuccess ||
                                              cudaMalloc(&g.d_bh[i][1], (long long)g.rows * sh.out_stride * 4) != cudaSuccess)) { (void)cudaGetLastError(); return HS_ERR_ALLOC; }
    }
    return HS_OK;
}

struct HostForm {           // one form's host-side arguments (snr == nullptr: the form is not run)
    const float* mu;
    const float* sigma;
    float* snr;
    int32_t* bh;
    uint32_t* path;         // greedy only
};

// Spectra go through the plan's two staging slots in groups of rows: upload ONCE, run the requested forms on the
// slot, download their outputs; the two slots alternate on two streams so copies and kernels overlap.
hs_status run_host(hs_plan_s* p, const float* hx, const float* hb, const HostForm& gr, const HostForm& pr) {
    if (!p || p->two_d || !hx || (!gr.snr && !pr.snr)) return HS_ERR_INVALID_ARG;
    if ((gr.snr && !gr.bh) || (pr.snr && !pr.bh)) return HS_ERR_INVALID_ARG;
    HsStats st_g, st_p;
    hs_status rc = HS_OK;
    if (gr.snr && (rc = fill_stats(p, gr.mu, gr.sigma, &st_g)) != HS_OK) return rc;
    if (pr.snr && (rc = fill_stats(p, pr.mu, pr.sigma, &st_p)) != HS_OK) return rc;
    DeviceGuard guard(p->device);
    HS_CUDA(guard.err);
    const bool both = gr.snr && pr.snr;
    rc = ensure_stage(p, hb != nullptr, gr.snr && gr.path, both);
    if (rc != HS_OK) return rc;
    HostStage& g = p->stage;
    const HsShape& full = p->shape;
    hs_status result = HS_OK;
    int chunk = 0;
    const size_t w = (size_t)full.n_fund * 4, pitch = (size_t)full.out_stride * 4;
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
        int f = 0;
        if (gr.snr) {
            HsIO io{g.d_in[i], hb ? g.d_base[i] : nullptr, g.d_snr[i][f], g.d_bh[i][f], gr.path ? g.d_path[i] : nullptr};
            result = launch_greedy(p, sh, st_g, io, stm);
            if (result != HS_OK) break;
            e = cudaMemcpy2DAsync(gr.snr + (long long)s0 * full.out_stride, pitch, g.d_snr[i][f], pitch, w, rows, cudaMemcpyDeviceToHost, stm);
            if (e == cudaSuccess)
                e = cudaMemcpy2DAsync(gr.bh + (long long)s0 * full.out_stride, pitch, g.d_bh[i][f], pitch, w, rows, cudaMemcpyDeviceToHost, stm);
            if (e == cudaSuccess && gr.path)
                e = cudaMemcpy2DAsync(gr.path + (long long)s0 * full.out_stride, pitch, g.d_path[i], pitch, w, rows, cudaMemcpyDeviceToHost, stm);
            if (e != cudaSuccess) { result = cuda_fail(e); break; }
            ++f;
        }
        if (pr.snr) {
            HsIO io{g.d_in[i], hb ? g.d_base[i] : nullptr, g.d_snr[i][f], g.d_bh[i][f], nullptr};
            result = launch_presto(p, sh, st_p, io, stm);
            if (result != HS_OK) break;
            e = cudaMemcpy2DAsync(pr.snr + (long long)s0 * full.out_stride, pitch, g.d_snr[i][f], pitch, w, rows, cudaMemcpyDeviceToHost, stm);
            if (e == cudaSuccess)
                e = cudaMemcpy2DAsync(pr.bh + (long long)s0 * full.out_stride, pitch, g.d_bh[i][f], pitch, w, rows, cudaMemcpyDeviceToHost, stm);
            if (e != cudaSuccess) { result = cuda_fail(e); break; }
        }
    }
    for (int i = 0; i < 2; ++i) {
        cudaError_t e = cudaStreamSynchronize(g.stream[i]);
        if (e != cudaSuccess && result == HS_OK) result = cuda_fail(e);
    }
    return result;
}

template <int L>
hs_status launch_presto_tile_2d(hs_plan_s* p, const HsStats& st, const HsIO& io, cudaStream_t stream) {
    constexpr int W = 2;
    constexpr int smem = 4 * hs_tile::smem_words(L, W);
    static std::atomic<uint64_t> opted{0};
    HS_CUDA(opt_in_smem(hs_presto_tile_kernel<L, W, false, true>, smem, p->device, opted));
    constexpr int T = hs_tile::TILE * W;
    const HsShape& sh = p->shape;
    dim3 grid((unsigned)((sh.n_fund + T - 1) / T), (unsigned)sh.n_spectra);
    hs_presto_tile_kernel<L, W, false, true><<<grid, 64 * W, smem, stream>>>(sh, st, io);
    p->last_kernel = "hs_presto_tile_kernel<W=2,2d>";
    p->launches += 1;
    HS_CUDA(cudaGetLastError());
    return HS_OK;
}

// threshold + compaction of `rows` output rows whose first spectrum has index s_base; appends to d_out / d_count
hs_status launch_candidates(hs_plan_s* plan, const float* d_snr, const int32_t* d_best_h, long long n_rows, long long s_base,
                            float threshold, hs_candidate* d_out, int64_t capacity, uint64_t* d_count, cudaStream_t stream) {
    const HsShape& sh = plan->shape;
    if (sh.n_fund == 0) return HS_OK;
    const long long n4 = (sh.n_fund + 3) / 4;
    for (long long s0 = 0; s0 < n_rows; s0 += HS_MAX_GRID_Y) {
        const int rows = (int)std::min<long long>(HS_MAX_GRID_Y, n_rows - s0);
        // a few waves of 256-thread CTAs per spectrum row, grid-stride inside the row
        const long long per_row = std::max(1ll, std::min((n4 + 255) / 256, (long long)std::max(1, plan->sm_count * 64 / rows + 1)));
        dim3 grid((unsigned)per_row, (unsigned)rows);
        hs_candidates_kernel<256><<<grid, 256, 0, stream>>>(d_snr + s0 * sh.out_stride, d_best_h + s0 * sh.out_stride, sh.out_stride,
                                                            (int)sh.n_fund, (int)(s_base + s0), threshold, reinterpret_cast<HsCandidate*>(d_out),
                                                            (unsigned long long)capacity, reinterpret_cast<unsigned long long*>(d_count));
        plan->launches += 1;
        HS_CUDA(cudaGetLastError());
    }
    return HS_OK;
}

bool presto_flags_ok(uint32_t flags) { return !((flags & HS_PRESTO_ALL_ORDERS) && !(flags & HS_PRESTO_ALL_HARMONICS)); }

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
    const uint32_t known = HS_GREEDY_NO_FUND_SELECT | HS_GREEDY_NO_DRIFT | HS_PRESTO_ALL_HARMONICS | HS_PRESTO_ALL_ORDERS;
    if (flags & ~known) return HS_ERR_INVALID_ARG;
    if (!presto_flags_ok(flags)) return HS_ERR_INVALID_ARG;
    if (device < 0) return HS_ERR_INVALID_ARG;
    int count = 0;
    HS_CUDA(cudaGetDeviceCount(&count));
    if (device >= count) return HS_ERR_INVALID_ARG;
    int sms = 0;
    HS_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device));
    hs_plan_s* p = new (std::nothrow) hs_plan_s();      // host state only: no device allocation, no sync
    if (!p) return HS_ERR_ALLOC;
    p->shape.n_bins = n_bins;
    p->shape.n_fund = n_fund;
    p->shape.in_stride = in_stride;
    p->shape.out_stride = out_stride;
    p->shape.n_spectra = n_spectra;
    p->shape.H = H;
    p->shape.flags = flags;
    p->tune = 0;
    p->two_d = false;
    p->shape.Z = 0;
    p->device = device;
    p->sm_count = sms;
    p->launches = 0;
    p->last_kernel = "";
    p->host_slot_bytes = 256ll << 20;
    *plan = p;
    return HS_OK;
}

hs_status hs_plan_2d(hs_plan_t* plan, int64_t n_bins, int32_t n_z, int32_t H, int64_t in_stride, int64_t out_stride,
                     uint32_t flags, int32_t device) {
    if (!plan) return HS_ERR_INVALID_ARG;
    *plan = nullptr;
    // k r and 2 k r + H' stay in 32 bits for k <= 16
    if (n_bins < 2 || n_bins > (1ll << 25) || n_z < 1 || !(n_z & 1) || n_z > 65535 || H < 1 || H > 16) return HS_ERR_INVALID_ARG;
    const hs_status rc = hs_plan(plan, n_bins, n_z, H, in_stride, out_stride, 0, flags, device);
    if (rc != HS_OK) return rc;
    (*plan)->two_d = true;
    (*plan)->shape.Z = (n_z - 1) / 2;
    return HS_OK;
}

hs_status hs_run_greedy_2d(hs_plan_t plan, const float* d_plane, const float* mu, const float* sigma,
                           float* d_snr, int32_t* d_best_h, uint32_t* d_path, void* cuda_stream) {
    hs_status rc = check_device_args(plan, d_plane, nullptr, d_snr, d_best_h, d_path);
    if (rc != HS_OK) return rc;
    if (!plan->two_d) return HS_ERR_INVALID_ARG;
    HsStats st;
    rc = fill_stats(plan, mu, sigma, &st);
    if (rc != HS_OK) return rc;
    DeviceGuard guard(plan->device);
    HS_CUDA(guard.err);
    const HsShape& sh = plan->shape;
    HsIO io{d_plane, nullptr, d_snr, d_best_h, d_path, nullptr, nullptr};
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    constexpr int BLOCK = 256, R = 2;
    dim3 grid((unsigned)((sh.n_bins + BLOCK * R - 1) / (BLOCK * R)), (unsigned)sh.n_spectra);
    const bool fs = !(sh.flags & HS_GREEDY_NO_FUND_SELECT), wp = d_path != nullptr, drift = !(sh.flags & HS_GREEDY_NO_DRIFT);
    if (!drift) {
        if (wp) hs_greedy2d_kernel<BLOCK, R, true, true, false><<<grid, BLOCK, 0, stream>>>(sh, st, io);
        else hs_greedy2d_kernel<BLOCK, R, true, false, false><<<grid, BLOCK, 0, stream>>>(sh, st, io);
    } else if (fs && wp) hs_greedy2d_kernel<BLOCK, R, true, true, true><<<grid, BLOCK, 0, stream>>>(sh, st, io);
    else if (fs) hs_greedy2d_kernel<BLOCK, R, true, false, true><<<grid, BLOCK, 0, stream>>>(sh, st, io);
    else if (wp) hs_greedy2d_kernel<BLOCK, R, false, true, true><<<grid, BLOCK, 0, stream>>>(sh, st, io);
    else hs_greedy2d_kernel<BLOCK, R, false, false, true><<<grid, BLOCK, 0, stream>>>(sh, st, io);
    plan->last_kernel = "hs_greedy2d_kernel";
    plan->launches += 1;
    HS_CUDA(cudaGetLastError());
    return HS_OK;
}

hs_status hs_run_presto_2d(hs_plan_t plan, const float* d_plane, const float* mu, const float* sigma,
                           float* d_snr, int32_t* d_best_h, void* cuda_stream) {
    hs_status rc = check_device_args(plan, d_plane, nullptr, d_snr, d_best_h, nullptr);
    if (rc != HS_OK) return rc;
    if (!plan->two_d) return HS_ERR_INVALID_ARG;
    HsStats st;
    rc = fill_stats(plan, mu, sigma, &st);
    if (rc != HS_OK) return rc;
    DeviceGuard guard(plan->device);
    HS_CUDA(guard.err);
    const HsShape& sh = plan->shape;
    HsIO io{d_plane, nullptr, d_snr, d_best_h, nullptr, nullptr, nullptr};
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    if (!(sh.flags & (HS_PRESTO_ALL_HARMONICS | HS_PRESTO_ALL_ORDERS)) && plan->tune != HS_TUNE_GENERIC) {
        switch (floor_log2(sh.H)) {
            case 0: return launch_presto_tile_2d<0>(plan, st, io, stream);
            case 1: return launch_presto_tile_2d<1>(plan, st, io, stream);
            case 2: return launch_presto_tile_2d<2>(plan, st, io, stream);
            case 3: return launch_presto_tile_2d<3>(plan, st, io, stream);
            default: return launch_presto_tile_2d<4>(plan, st, io, stream);
        }
    }
    dim3 grid((unsigned)((sh.n_bins + 255) / 256), (unsigned)sh.n_spectra);
    hs_presto2d_generic_kernel<<<grid, 256, 0, stream>>>(sh, st, io);
    plan->last_kernel = "hs_presto2d_generic_kernel";
    plan->launches += 1;
    HS_CUDA(cudaGetLastError());
    return HS_OK;
}

hs_status hs_plan_set_host_slot_bytes(hs_plan_t plan, int64_t bytes) {
    if (!plan || bytes < 1 || plan->stage.ready) return HS_ERR_INVALID_ARG;     // the slots exist once a *_host call has run
    plan->host_slot_bytes = bytes;
    return HS_OK;
}

hs_status hs_plan_set_tuning(hs_plan_t plan, uint32_t variant) {
    if (!plan || variant > 255u) return HS_ERR_INVALID_ARG;
    plan->tune = variant;
    return HS_OK;
}

hs_status hs_run_greedy(hs_plan_t plan, const float* d_spectra, const float* d_inv_baseline, const float* mu,
                        const float* sigma, float* d_snr, int32_t* d_best_h, uint32_t* d_path, void* cuda_stream) {
    hs_status rc = check_device_args(plan, d_spectra, d_inv_baseline, d_snr, d_best_h, d_path);
    if (rc != HS_OK) return rc;
    if (plan->two_d) return HS_ERR_INVALID_ARG;
    HsStats st;
    rc = fill_stats(plan, mu, sigma, &st);
    if (rc != HS_OK) return rc;
    DeviceGuard guard(plan->device);
    HS_CUDA(guard.err);
    HsIO io{d_spectra, d_inv_baseline, d_snr, d_best_h, d_path};
    return launch_greedy(plan, plan->shape, st, io, (cudaStream_t)cuda_stream);
}

hs_status hs_run_presto(hs_plan_t plan, const float* d_spectra, const float* d_inv_baseline, const float* mu,
                        const float* sigma, float* d_snr, int32_t* d_best_h, void* cuda_stream) {
    hs_status rc = check_device_args(plan, d_spectra, d_inv_baseline, d_snr, d_best_h, nullptr);
    if (rc != HS_OK) return rc;
    if (plan->two_d) return HS_ERR_INVALID_ARG;
    HsStats st;
    rc = fill_stats(plan, mu, sigma, &st);
    if (rc != HS_OK) return rc;
    DeviceGuard guard(plan->device);
    HS_CUDA(guard.err);
    HsIO io{d_spectra, d_inv_baseline, d_snr, d_best_h, nullptr};
    return launch_presto(plan, plan->shape, st, io, (cudaStream_t)cuda_stream);
}

hs_status hs_run_greedy_dstats(hs_plan_t plan, const float* d_spectra, const float* d_inv_baseline, const float* d_mu,
                               const float* d_sigma, float* d_snr, int32_t* d_best_h, uint32_t* d_path, void* cuda_stream) {
    hs_status rc = check_device_args(plan, d_spectra, d_inv_baseline, d_snr, d_best_h, d_path);
    if (rc != HS_OK) return rc;
    if (plan->two_d || !d_mu || !d_sigma || (reinterpret_cast<uintptr_t>(d_mu) & 3u) || (reinterpret_cast<uintptr_t>(d_sigma) & 3u)) return HS_ERR_INVALID_ARG;
    HsStats st;
    std::memset(&st, 0, sizeof(st));
    DeviceGuard guard(plan->device);
    HS_CUDA(guard.err);
    HsIO io{d_spectra, d_inv_baseline, d_snr, d_best_h, d_path, d_mu, d_sigma};
    return launch_greedy(plan, plan->shape, st, io, (cudaStream_t)cuda_stream);
}

hs_status hs_run_presto_dstats(hs_plan_t plan, const float* d_spectra, const float* d_inv_baseline, const float* d_mu,
                               const float* d_sigma, float* d_snr, int32_t* d_best_h, void* cuda_stream) {
    hs_status rc = check_device_args(plan, d_spectra, d_inv_baseline, d_snr, d_best_h, nullptr);
    if (rc != HS_OK) return rc;
    if (plan->two_d || !d_mu || !d_sigma || (reinterpret_cast<uintptr_t>(d_mu) & 3u) || (reinterpret_cast<uintptr_t>(d_sigma) & 3u)) return HS_ERR_INVALID_ARG;
    HsStats st;
    std::memset(&st, 0, sizeof(st));
    DeviceGuard guard(plan->device);
    HS_CUDA(guard.err);
    HsIO io{d_spectra, d_inv_baseline, d_snr, d_best_h, nullptr, d_mu, d_sigma};
    return launch_presto(plan, plan->shape, st, io, (cudaStream_t)cuda_stream);
}

hs_status hs_whiten(hs_plan_t plan, const float* d_spectra, const float* d_inv_baseline, float* d_whitened, void* cuda_stream) {
    if (!plan || plan->two_d || !d_spectra || !d_inv_baseline || !d_whitened) return HS_ERR_INVALID_ARG;
    if (!aligned16(d_spectra) || !aligned16(d_inv_baseline) || !aligned16(d_whitened)) return HS_ERR_INVALID_ARG;
    if ((const void*)d_whitened == (const void*)d_spectra || (const void*)d_whitened == (const void*)d_inv_baseline) return HS_ERR_INVALID_ARG;
    const HsShape& sh = plan->shape;
    DeviceGuard guard(plan->device);
    HS_CUDA(guard.err);
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    for (long long s0 = 0; s0 < sh.n_spectra; s0 += HS_MAX_GRID_Y) {
        const int rows = (int)std::min<long long>(HS_MAX_GRID_Y, sh.n_spectra - s0);
        const long long n4 = std::max<long long>(1, sh.n_bins / 4);
        const long long per_row = std::max(1ll, std::min((n4 + 255) / 256, (long long)std::max(1, plan->sm_count * 32 / rows + 1)));
        dim3 grid((unsigned)per_row, (unsigned)rows);
        hs_whiten_kernel<<<grid, 256, 0, stream>>>(d_spectra + s0 * sh.in_stride, d_inv_baseline + s0 * sh.in_stride,
                                                   d_whitened + s0 * sh.in_stride, sh.in_stride, sh.in_stride, (int)sh.n_bins);
        plan->launches += 1;
        HS_CUDA(cudaGetLastError());
    }
    return HS_OK;
}

int64_t hs_stats_workspace_bytes(hs_plan_t plan, int32_t n_clip) {
    if (!plan || n_clip < 0 || n_clip > 16) return -1;
    return (int64_t)(n_clip + 1) * plan->shape.n_spectra * HS_MAX_H * 3 * (int64_t)sizeof(double);
}

namespace {
int64_t stats_cache_pitch(int64_t count) { return (count + 3) & ~(int64_t)3; }
int64_t stats_cache_offset(int64_t accumulators) { return (accumulators + 255) & ~(int64_t)255; }
}  // namespace

int64_t hs_stats_workspace_bytes_cached(hs_plan_t plan, int32_t n_clip, int64_t n_lo, int64_t n_hi) {
    const int64_t need = hs_stats_workspace_bytes(plan, n_clip);
    if (need < 0) return -1;
    if (n_hi == 0) n_hi = plan->shape.n_bins;
    if (n_lo < 0 || n_hi > plan->shape.n_bins || n_lo > n_hi) return -1;
    return stats_cache_offset(need) + (int64_t)plan->shape.n_spectra * plan->shape.H * stats_cache_pitch(n_hi - n_lo) * (int64_t)sizeof(float);
}

hs_status hs_estimate_stats(hs_plan_t plan, int32_t greedy, const float* d_spectra, const float* d_inv_baseline,
                            int64_t n_lo, int64_t n_hi, float clip_sigma, int32_t n_clip,
                            float* d_mu, float* d_sigma, void* d_work, int64_t work_bytes, void* cuda_stream) {
    if (!plan || plan->two_d || !d_spectra || !d_mu || !d_sigma || !d_work) return HS_ERR_INVALID_ARG;
    const HsShape& sh = plan->shape;
    if (n_hi == 0) n_hi = sh.n_bins;
    if (n_lo < 0 || n_hi > sh.n_bins || n_lo > n_hi || n_clip < 0 || n_clip > 16 || !(clip_sigma > 0.f)) return HS_ERR_INVALID_ARG;
    if (!aligned16(d_spectra) || (d_inv_baseline && !aligned16(d_inv_baseline)) || (reinterpret_cast<uintptr_t>(d_work) & 7u) ||
        (reinterpret_cast<uintptr_t>(d_mu) & 3u) || (reinterpret_cast<uintptr_t>(d_sigma) & 3u))
        return HS_ERR_INVALID_ARG;
    const int64_t need = hs_stats_workspace_bytes(plan, n_clip);
    if (work_bytes < need) return HS_ERR_INVALID_ARG;
    if (!greedy && !presto_flags_ok(sh.flags)) return HS_ERR_INVALID_ARG;
    if (sh.n_bins >= (1ll << 31) - 64 - 1 && !greedy) return HS_ERR_UNSUPPORTED;
    DeviceGuard guard(plan->device);
    HS_CUDA(guard.err);
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    HS_CUDA(cudaMemsetAsync(d_work, 0, (size_t)need, stream));
    double* acc = static_cast<double*>(d_work);
    const long long per_round = (long long)sh.n_spectra * HS_MAX_H * 3;
    const long long count = n_hi - n_lo;
    // cached path: a workspace of hs_stats_workspace_bytes_cached() also holds the sums of the first pass, and the
    // rejection rounds stream them back instead of gathering again (the same fp32 values, so the same results)
    const long long cpad = stats_cache_pitch(count);
    const bool cached = n_clip >= 1 && count > 0 && ((reinterpret_cast<uintptr_t>(d_work) + (uintptr_t)stats_cache_offset(need)) & 15u) == 0 &&
                        work_bytes >= stats_cache_offset(need) + (int64_t)sh.n_spectra * sh.H * cpad * (int64_t)sizeof(float);
    float* cache = cached ? reinterpret_cast<float*>(static_cast<char*>(d_work) + stats_cache_offset(need)) : nullptr;
    if (count > 0) {
        for (int r = 0; r <= n_clip; ++r) {
            for (long long s0 = 0; s0 < sh.n_spectra; s0 += HS_MAX_GRID_Y) {
                HsShape sub = sh;
                sub.n_spectra = (int)std::min<long long>(HS_MAX_GRID_Y, sh.n_spectra - s0);
                const double* prev = r ? acc + (r - 1) * per_round + s0 * HS_MAX_H * 3 : nullptr;
                double* cur = acc + r * per_round + s0 * HS_MAX_H * 3;
                float* csub = cached ? cache + s0 * sh.H * cpad : nullptr;
                if (cached && r == 0) {                      // the one gather: the sums go to the workspace
                    HsIO io{d_spectra + s0 * sh.in_stride, d_inv_baseline ? d_inv_baseline + s0 * sh.in_stride : nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
                    HsStatsArgs a{n_lo, n_hi, (double)clip_sigma, nullptr, nullptr, csub, cpad};
                    dim3 sgrid((unsigned)std::max(1ll, (count + 256 * 2 - 1) / (256 * 2)), (unsigned)sub.n_spectra);   // two groups of 32 bins per warp
                    if (greedy && d_inv_baseline) hs_stats_store_kernel<true, true><<<sgrid, 256, 0, stream>>>(sub, io, a);
                    else if (greedy) hs_stats_store_kernel<true, false><<<sgrid, 256, 0, stream>>>(sub, io, a);
                    else if (d_inv_baseline) hs_stats_store_kernel<false, true><<<sgrid, 256, 0, stream>>>(sub, io, a);
                    else hs_stats_store_kernel<false, false><<<sgrid, 256, 0, stream>>>(sub, io, a);
                    plan->launches += 1;
                    HS_CUDA(cudaGetLastError());
                }
                if (cached) {
                    const long long n4 = std::max(1ll, count / 4);
                    dim3 cgrid((unsigned)std::max(1ll, std::min(64ll, (n4 + 256 * 16 - 1) / (256 * 16))), (unsigned)sh.H, (unsigned)sub.n_spectra);
                    hs_stats_cached_kernel<<<cgrid, 256, 0, stream>>>(csub, cpad, count, sh.H, (double)clip_sigma, prev, cur);
                    plan->launches += 1;
                    HS_CUDA(cudaGetLastError());
                    continue;
                }
                HsIO io{d_spectra + s0 * sh.in_stride, d_inv_baseline ? d_inv_baseline + s0 * sh.in_stride : nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
                HsStatsArgs a{n_lo, n_hi, (double)clip_sigma, prev, cur, csub, cpad};
                const long long want = std::max(1ll, (count + 256 * 2 - 1) / (256 * 2));      // two groups of 32 bins per warp
                dim3 grid((unsigned)want, (unsigned)sub.n_spectra);
                if (greedy && d_inv_baseline) hs_stats_pass_kernel<true, true><<<grid, 256, 0, stream>>>(sub, io, a);
                else if (greedy) hs_stats_pass_kernel<true, false><<<grid, 256, 0, stream>>>(sub, io, a);
                else if (d_inv_baseline) hs_stats_pass_kernel<false, true><<<grid, 256, 0, stream>>>(sub, io, a);
                else hs_stats_pass_kernel<false, false><<<grid, 256, 0, stream>>>(sub, io, a);
                plan->launches += 1;
                HS_CUDA(cudaGetLastError());
            }
        }
    }
    const int total = sh.n_spectra * sh.H;
    hs_stats_finish_kernel<<<(total + 255) / 256, 256, 0, stream>>>(acc + n_clip * per_round, sh.n_spectra, sh.H, d_mu, d_sigma);
    plan->launches += 1;
    plan->last_kernel = cached ? "hs_stats_store_kernel+hs_stats_cached_kernel" : "hs_stats_pass_kernel";
    HS_CUDA(cudaGetLastError());
    return HS_OK;
}

// ------------------------------------------------------------------------------------------
// hs_estimate_stats_static: the statistics step for callers that cannot allocate device memory.
//
// Who that is: code that runs where a cudaMalloc is forbidden or ruinous -- a real-time search pipeline whose
// device memory is carved up once at start-up and then frozen, a plug-in inside a host application that owns the
// allocator and hands out only the input and output buffers, a worker that lives inside a memory pool with no head
// room left (cudaMalloc may then fail, or synchronise the whole device in the middle of an observation).  Such a
// caller can provide the spectra and the [S][H] results, but not the (n_clip + 1) x S x 32 x 3 doubles of
// accumulators hs_estimate_stats wants as d_work.  Here that workspace lives in the library image itself.
//
// g_stats_scratch is a file-scope __device__ array: the CUDA runtime places one copy on EVERY device that loads
// this library and keeps it there until the process exits (HS_STATIC_STATS_MAX_BYTES = 3 MiB per device).  In
// host code the identifier `g_stats_scratch` is only the host-side shadow of that array -- NOT a device address
// (a kernel handed &g_stats_scratch would fault, or scribble over host memory on a system where the GPU can reach
// it); the device address of the current device's copy comes from cudaGetSymbolAddress, asked once per device.
// ------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_stats_scratch[HS_STATIC_STATS_MAX_BYTES];

namespace {
constexpr int HS_SCRATCH_DEVICES = 64;
std::atomic<void*> g_stats_scratch_addr[HS_SCRATCH_DEVICES];     // device address of g_stats_scratch, per device ordinal

// The plan's device must be current (cudaGetSymbolAddress answers for the current device).  The first call on a
// device may load the library's module there, which is why it has to happen outside any stream capture.
hs_status stats_scratch_address(int device, void** out) {
    *out = nullptr;
    if (device >= 0 && device < HS_SCRATCH_DEVICES) {
        void* known = g_stats_scratch_addr[device].load(std::memory_order_acquire);
        if (known) { *out = known; return HS_OK; }
    }
    void* ptr = nullptr;
    HS_CUDA(cudaGetSymbolAddress(&ptr, g_stats_scratch));
    if (!ptr) return cuda_fail(cudaErrorInvalidSymbol);
    if (device >= 0 && device < HS_SCRATCH_DEVICES) g_stats_scratch_addr[device].store(ptr, std::memory_order_release);
    *out = ptr;
    return HS_OK;
}
}  // namespace

hs_status hs_estimate_stats_static(hs_plan_t plan, int32_t greedy, const float* d_spectra, const float* d_inv_baseline,
                                   int64_t n_lo, int64_t n_hi, float clip_sigma, int32_t n_clip,
                                   float* d_mu, float* d_sigma, void* cuda_stream) {
    if (!plan) return HS_ERR_INVALID_ARG;
    const int64_t need = hs_stats_workspace_bytes(plan, n_clip);
    if (need < 0) return HS_ERR_INVALID_ARG;
    if (need > (int64_t)HS_STATIC_STATS_MAX_BYTES) return HS_ERR_TOO_LARGE;     // (n_clip + 1) * n_spectra > HS_STATIC_STATS_MAX_ROWS
    void* scratch = nullptr;
    {
        DeviceGuard guard(plan->device);                 // the symbol address is a per-device answer
        HS_CUDA(guard.err);
        const hs_status rc = stats_scratch_address(plan->device, &scratch);
        if (rc != HS_OK) return rc;
    }
    // From here on this is hs_estimate_stats with the library-owned workspace: it validates the other arguments,
    // clears the `need` bytes it uses with a cudaMemsetAsync ON THE STREAM (the array still holds the last call's
    // sums), and launches the same kernels.  Nothing on this path calls cudaMalloc / cudaFree or a library routine
    // that allocates.
    return hs_estimate_stats(plan, greedy, d_spectra, d_inv_baseline, n_lo, n_hi, clip_sigma, n_clip, d_mu, d_sigma,
                             scratch, need, cuda_stream);
}

hs_status hs_run_greedy_host(hs_plan_t plan, const float* h_spectra, const float* h_inv_baseline, const float* mu,
                             const float* sigma, float* h_snr, int32_t* h_best_h, uint32_t* h_path) {
    if (!h_snr || !h_best_h) return HS_ERR_INVALID_ARG;
    return run_host(plan, h_spectra, h_inv_baseline, HostForm{mu, sigma, h_snr, h_best_h, h_path},
                    HostForm{nullptr, nullptr, nullptr, nullptr, nullptr});
}

hs_status hs_run_presto_host(hs_plan_t plan, const float* h_spectra, const float* h_inv_baseline, const float* mu,
                             const float* sigma, float* h_snr, int32_t* h_best_h) {
    if (!h_snr || !h_best_h) return HS_ERR_INVALID_ARG;
    return run_host(plan, h_spectra, h_inv_baseline, HostForm{nullptr, nullptr, nullptr, nullptr, nullptr},
                    HostForm{mu, sigma, h_snr, h_best_h, nullptr});
}

hs_status hs_run_both_host(hs_plan_t plan, const float* h_spectra, const float* h_inv_baseline,
                           const float* mu_greedy, const float* sigma_greedy, float* h_snr_greedy, int32_t* h_best_h_greedy,
                           uint32_t* h_path,
                           const float* mu_presto, const float* sigma_presto, float* h_snr_presto, int32_t* h_best_h_presto) {
    if (!h_snr_greedy || !h_best_h_greedy || !h_snr_presto || !h_best_h_presto) return HS_ERR_INVALID_ARG;
    return run_host(plan, h_spectra, h_inv_baseline, HostForm{mu_greedy, sigma_greedy, h_snr_greedy, h_best_h_greedy, h_path},
                    HostForm{mu_presto, sigma_presto, h_snr_presto, h_best_h_presto, nullptr});
}

hs_status hs_find_candidates(hs_plan_t plan, const float* d_snr, const int32_t* d_best_h, float threshold,
                             hs_candidate* d_out, int64_t capacity, uint64_t* d_count, void* cuda_stream) {
    static_assert(sizeof(hs_candidate) == sizeof(HsCandidate) && sizeof(hs_candidate) == 16, "candidate layout");
    if (!plan || !d_snr || !d_best_h || !d_count || capacity < 0 || (capacity > 0 && !d_out)) return HS_ERR_INVALID_ARG;
    if (!aligned16(d_snr) || !aligned16(d_best_h) || (d_out && !aligned16(d_out)) || (reinterpret_cast<uintptr_t>(d_count) & 7u))
        return HS_ERR_INVALID_ARG;
    if (!(threshold == threshold)) return HS_ERR_INVALID_ARG;
    DeviceGuard guard(plan->device);
    HS_CUDA(guard.err);
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    HS_CUDA(cudaMemsetAsync(d_count, 0, sizeof(uint64_t), stream));
    return launch_candidates(plan, d_snr, d_best_h, plan->shape.n_spectra, 0, threshold, d_out, capacity, d_count, stream);
}

hs_status hs_search_host(hs_plan_t plan, const float* h_spectra, const float* h_inv_baseline,
                         const float* mu_greedy, const float* sigma_greedy, const float* mu_presto, const float* sigma_presto,
                         float threshold, hs_candidate* h_cand_greedy, int64_t capacity_greedy, uint64_t* h_count_greedy,
                         hs_candidate* h_cand_presto, int64_t capacity_presto, uint64_t* h_count_presto) {
    if (!plan || plan->two_d || !h_spectra || !h_count_greedy || !h_count_presto || capacity_greedy < 0 || capacity_presto < 0 ||
        (capacity_greedy > 0 && !h_cand_greedy) || (capacity_presto > 0 && !h_cand_presto) || !(threshold == threshold))
        return HS_ERR_INVALID_ARG;
    HsStats st_g, st_p;
    hs_status rc = fill_stats(plan, mu_greedy, sigma_greedy, &st_g);
    if (rc != HS_OK) return rc;
    if ((rc = fill_stats(plan, mu_presto, sigma_presto, &st_p)) != HS_OK) return rc;
    DeviceGuard guard(plan->device);
    HS_CUDA(guard.err);
    if ((rc = ensure_stage(plan, h_inv_baseline != nullptr, false, false)) != HS_OK) return rc;
    HostStage& g = plan->stage;
    const HsShape& full = plan->shape;
    // candidate buffers and counters on the device (owned by the plan's host path; grown on demand)
    const int64_t need = capacity_greedy + capacity_presto;
    if (g.cand_cap < need || !g.d_cand_count) {
        if (g.d_cand) cudaFree(g.d_cand);
        g.d_cand = nullptr; g.cand_cap = 0;
        if (!g.d_cand_count && cudaMalloc(&g.d_cand_count, 2 * sizeof(uint64_t)) != cudaSuccess) { (void)cudaGetLastError(); return HS_ERR_ALLOC; }
        if (need > 0 && cudaMalloc(&g.d_cand, (size_t)need * sizeof(HsCandidate)) != cudaSuccess) { (void)cudaGetLastError(); return HS_ERR_ALLOC; }
        g.cand_cap = need;
    }
    HS_CUDA(cudaMemsetAsync(g.d_cand_count, 0, 2 * sizeof(uint64_t), g.stream[0]));
    HS_CUDA(cudaStreamSynchronize(g.stream[0]));                    // both streams append to the same counters
    hs_candidate* d_cg = reinterpret_cast<hs_candidate*>(g.d_cand);
    hs_candidate* d_cp = d_cg ? d_cg + capacity_greedy : nullptr;
    hs_status result = HS_OK;
    int chunk = 0;
    for (int s0 = 0; s0 < full.n_spectra && result == HS_OK; s0 += g.rows, ++chunk) {
        const int i = chunk & 1;
        const int rows = std::min(g.rows, full.n_spectra - s0);
        cudaStream_t stm = g.stream[i];
        HsShape sh = full;
        sh.n_spectra = rows;
        cudaError_t e = cudaMemcpy2DAsync(g.d_in[i], full.in_stride * 4, h_spectra + (long long)s0 * full.in_stride, full.in_stride * 4,
                                          full.n_bins * 4, rows, cudaMemcpyHostToDevice, stm);
        if (e == cudaSuccess && h_inv_baseline)
            e = cudaMemcpy2DAsync(g.d_base[i], full.in_stride * 4, h_inv_baseline + (long long)s0 * full.in_stride, full.in_stride * 4,
                                  full.n_bins * 4, rows, cudaMemcpyHostToDevice, stm);
        if (e != cudaSuccess) { result = cuda_fail(e); break; }
        HsIO io{g.d_in[i], h_inv_baseline ? g.d_base[i] : nullptr, g.d_snr[i][0], g.d_bh[i][0], nullptr, nullptr, nullptr};
        if ((result = launch_greedy(plan, sh, st_g, io, stm)) != HS_OK) break;
        if ((result = launch_candidates(plan, g.d_snr[i][0], g.d_bh[i][0], rows, s0, threshold, d_cg, capacity_greedy,
                                        g.d_cand_count, stm)) != HS_OK) break;
        if ((result = launch_presto(plan, sh, st_p, io, stm)) != HS_OK) break;
        if ((result = launch_candidates(plan, g.d_snr[i][0], g.d_bh[i][0], rows, s0, threshold, d_cp, capacity_presto,
                                        g.d_cand_count + 1, stm)) != HS_OK) break;
    }
    for (int i = 0; i < 2; ++i) {
        cudaError_t e = cudaStreamSynchronize(g.stream[i]);
        if (e != cudaSuccess && result == HS_OK) result = cuda_fail(e);
    }
    if (result != HS_OK) return result;
    uint64_t counts[2] = {0, 0};
    HS_CUDA(cudaMemcpy(counts, g.d_cand_count, sizeof(counts), cudaMemcpyDeviceToHost));
    *h_count_greedy = counts[0];
    *h_count_presto = counts[1];
    const uint64_t ng = std::min<uint64_t>(counts[0], (uint64_t)capacity_greedy), np_ = std::min<uint64_t>(counts[1], (uint64_t)capacity_presto);
    if (ng) HS_CUDA(cudaMemcpy(h_cand_greedy, d_cg, ng * sizeof(hs_candidate), cudaMemcpyDeviceToHost));
    if (np_) HS_CUDA(cudaMemcpy(h_cand_presto, d_cp, np_ * sizeof(hs_candidate), cudaMemcpyDeviceToHost));
    return HS_OK;
}

int64_t hs_launch_count(hs_plan_t plan) { return plan ? plan->launches : -1; }

const char* hs_last_kernel(hs_plan_t plan) { return plan ? plan->last_kernel : ""; }

hs_status hs_destroy(hs_plan_t plan) {
    if (!plan) return HS_OK;
    if (plan->stage.ready) {
        DeviceGuard guard(plan->device);
        free_stage(plan->stage);
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
        case HS_ERR_TOO_LARGE: return "HS_ERR_TOO_LARGE: the request exceeds the fixed scratch capacity of a no-allocation entry point";
    }
    return "unknown hs_status";
}

int32_t hs_last_cuda_error(void) { return g_last_cuda_error; }

}  // extern "C"
