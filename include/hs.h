/* =====================================================================================
 * hs.h -- C-ABI boundary of the B200-native incoherent harmonic sum (arXiv 2202.12817).
 *
 * The library computes, for a batch of fp32 Fourier power spectra (one per time-series /
 * DM trial), the per-bin maximum SNR over harmonic counts and the harmonic
 * count that gave it (eq. 2; "only the highest SNR value is returned for
 * each element n"), with the partial sums formed either
 *
 *   - by the paper's GREEDY algorithm (Alg. 2; eq. 5, PAPER.md:182:
 *     at order h read x[m], x[m+1] with m = h n + d, add the larger, and if it was the
 *     second one grow the drift d; fundamental-bin selection), or
 *   - by the PRESTO-like algorithm (Alg. 1; eq. 4, PAPER.md:138:
 *     X[n] = sum x[round(h n / H')], n the LAST bin of the series, H' in powers of two,
 *     fundamental plus even harmonics).
 *
 * Every step (gather, select, accumulate, normalise, max/argmax, store) runs in the
 * library's sm_100a kernels.  There is no CPU fallback.
 *
 * Symbols and indexing
 *   N = n_bins per spectrum, S = n_spectra, x[s][b] the power of spectrum s at bin b,
 *   H = maximum harmonic order (1..32).  mu[h-1], sigma[h-1] are the mean and standard
 *   deviation of the partial sum at harmonic order h; the library never
 *   estimates them inside hs_run_* ("GetMeanStdev()", is a step of its own: hs_estimate_stats).
 *   Outputs are written for every bin n in [0, n_fund) of every spectrum; for the greedy
 *   form n is the FUNDAMENTAL bin, for the PRESTO form n is the TOP (last-summed) bin
 *   (PAPER.md:140).
 *
 * Exact semantics (readings of the paper):
 *   greedy, per spectrum and n:   d = 0, sum = 0, best = -inf
 *     for h = 1..H:  m = h n + d;  stop if m > N-1;
 *        a = x[m];  b = x[m+1] if m+1 <= N-1 else -inf   (b = -inf at h = 1 under
 *        HS_GREEDY_NO_FUND_SELECT, and always under HS_GREEDY_NO_DRIFT);
 *        if b > a { d += 1; sum += b; path |= 1 << (h-1) } else sum += a;
 *        snr_h = (sum - mu[h-1]) / sigma[h-1];  if snr_h > best { best = snr_h; best_h = h }
 *   PRESTO, per spectrum and n:   best = -inf
 *     for H' in 1,2,4,..<=H (every H' = 1..H under HS_PRESTO_ALL_ORDERS):
 *        sum = sum over h in {1} U {2,4,..,H'} (1..H' under HS_PRESTO_ALL_HARMONICS)
 *              of x[(2 h n + H') / (2 H')]                  (round half up, exact integers)
 *        snr = (sum - mu[H'-1]) / sigma[H'-1];  if snr > best { best = snr; best_h = H' }
 *   With d_inv_baseline != NULL every x[b] above is replaced by the fp32 product
 *   x[b] * inv_baseline[b] (spectrum whitening supplied by the caller).
 *   Sums are accumulated in fp32.  Greedy: in the order written above.  PRESTO (Alg. 1): the harmonic sets are
 *   nested (the terms of H' are those of H'/2 plus the new fractions h/H' with h/2 odd), and the default kernel
 *   forms S_{H'} = S_{H'/2} + (the new terms of H' summed first, by increasing level-local order) -- a different
 *   fp32 association from the loop above, inside the stated tolerance; the coverage kernel adds in the written
 *   order.  ALL_HARMONICS variants: the terms of one H' may be grouped by reduced fraction h/H', each group in
 *   increasing h, groups in increasing denominator.  The SNR is formed as
 *   fma(sum, 1/sigma, -mu/sigma) in fp32, both constants rounded once on the host.  Non-finite
 *   inputs give unspecified results.
 *
 * Memory, ownership, threading
 *   The caller owns every buffer.  d_* pointers are DEVICE pointers on the plan's device;
 *   h_* pointers are HOST pointers; mu and sigma are always HOST arrays of H floats, read
 *   during the call and passed to the kernels by value (no hidden copy, no sync).
 *   Layout: row-major, spectrum s starts at element s*in_stride (inputs) / s*out_stride
 *   (outputs).  Device base pointers must be 16-byte aligned and strides multiples of 4
 *   elements.  No output array may overlap an input array or another output array anywhere in its
 *   [S][stride] extent (checked on the address ranges: HS_ERR_INVALID_ARG).  hs_run_* are asynchronous on the given
 *   CUDA stream (a cudaStream_t passed as void*; NULL = the legacy default stream) and
 *   neither allocate nor block.  hs_run_*_host are synchronous: they return when the host
 *   output arrays are complete.  A plan may be reused for any number of runs but not
 *   concurrently from two host threads.
 *
 * Errors: every entry point returns an hs_status; nothing throws or aborts.  Invalid
 *   arguments are rejected before any launch (HS_ERR_INVALID_ARG), valid but unimplemented
 *   combinations give HS_ERR_UNSUPPORTED, CUDA runtime failures HS_ERR_CUDA
 *   (hs_last_cuda_error() returns the cudaError_t value), allocation failures HS_ERR_ALLOC.
 * ===================================================================================== */
#ifndef HS_B200_H_
#define HS_B200_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hs_plan_s* hs_plan_t;

typedef enum {
    HS_OK = 0,
    HS_ERR_INVALID_ARG = 1,
    HS_ERR_UNSUPPORTED = 2,
    HS_ERR_ALLOC = 3,
    HS_ERR_CUDA = 4,
    HS_ERR_TOO_LARGE = 5      /* hs_estimate_stats_static only: the batch needs more than the built-in scratch array */
} hs_status;

enum {
    /* algorithm flags (plan) */
    HS_GREEDY_NO_FUND_SELECT = 1u << 0, /* order 1 takes x[n] without comparing with x[n+1] (PAPER.md:260 is optional) */
    HS_GREEDY_NO_DRIFT       = 1u << 1, /* simple harmonic sum, eq. 3: the drift stays 0 */
    HS_PRESTO_ALL_HARMONICS  = 1u << 2, /* PRESTO_all: sum every harmonic 1..H' */
    HS_PRESTO_ALL_ORDERS     = 1u << 3  /* with ALL_HARMONICS = PRESTO+: every H' = 1..H */
};

/* Create a plan for a batch shape.
 *   n_bins     N, 2 <= N <= 2^31 - 64
 *   n_spectra  S >= 1
 *   H          maximum harmonic order, 1..32
 *   in_stride  elements between consecutive input spectra (0 = n_bins); >= n_bins, multiple of 4
 *   out_stride elements between consecutive output rows (0 = n_fund rounded up to 4); >= n_fund, multiple of 4
 *   n_fund     outputs are computed for n < n_fund (0 = n_bins); <= n_bins
 *   flags      OR of the enum above; HS_PRESTO_ALL_ORDERS requires HS_PRESTO_ALL_HARMONICS
 *   device     CUDA device ordinal
 * The plan owns only small internal host state (shape, device properties); hs_plan allocates nothing on
 * the device and does not synchronise.  Once a *_host entry point has been used the plan also owns that
 * path's device staging buffers and streams.  n_spectra has no limit other than memory.
 * Every entry point that takes a plan runs on the plan's device whatever device is current, and leaves
 * the caller's current device unchanged. */
hs_status hs_plan(hs_plan_t* plan, int64_t n_bins, int32_t n_spectra, int32_t H,
                  int64_t in_stride, int64_t out_stride, int64_t n_fund,
                  uint32_t flags, int32_t device);

/* Greedy harmonic sum (Alg. 2) on device buffers.
 *   d_spectra       [S][in_stride] fp32 powers (device)
 *   d_inv_baseline  NULL, or [S][in_stride] fp32 per-bin multipliers (device)
 *   mu, sigma       HOST arrays of H floats, entry h-1 for order h; sigma > 0
 *   d_snr           [S][out_stride] fp32 out: max over h of snr_h
 *   d_best_h        [S][out_stride] int32 out: the order h (1..H) attaining it (first maximum)
 *   d_path          NULL, or [S][out_stride] uint32 out: bit h-1 set iff the drift grew at order h
 *   cuda_stream     cudaStream_t */
hs_status hs_run_greedy(hs_plan_t plan, const float* d_spectra, const float* d_inv_baseline,
                        const float* mu, const float* sigma,
                        float* d_snr, int32_t* d_best_h, uint32_t* d_path, void* cuda_stream);

/* PRESTO-like harmonic sum (Alg. 1 and its _all / + variants per the plan flags) on device
 * buffers; arguments as above; best_h is the H' attaining the maximum. */
hs_status hs_run_presto(hs_plan_t plan, const float* d_spectra, const float* d_inv_baseline,
                        const float* mu, const float* sigma,
                        float* d_snr, int32_t* d_best_h, void* cuda_stream);

/* The same two operations with PER-SPECTRUM statistics that already live on the device (the output of
 * hs_estimate_stats, or the caller's own): d_mu, d_sigma are DEVICE arrays [S][H] of fp32, entry [s][h-1] for order h
 * of spectrum s; every CTA forms 1/sigma and -mu/sigma of its spectrum exactly as the host does for the by-value
 * statistics.  The values are never read on the host, so they cannot be rejected as hs_run_* rejects bad host
 * statistics: an entry whose sigma is not a positive finite number, or whose mu is not finite, is replaced ON THE DEVICE
 * by (mu, sigma) = (0, 1) for that spectrum and order (the pair hs_estimate_stats returns for an order without samples),
 * identically in every kernel, so equal inputs give equal outputs whichever kernel variant or tile computes a bin.
 * Otherwise as hs_run_greedy / hs_run_presto: asynchronous, no allocation, no synchronisation. */
hs_status hs_run_greedy_dstats(hs_plan_t plan, const float* d_spectra, const float* d_inv_baseline,
                               const float* d_mu, const float* d_sigma,
                               float* d_snr, int32_t* d_best_h, uint32_t* d_path, void* cuda_stream);
hs_status hs_run_presto_dstats(hs_plan_t plan, const float* d_spectra, const float* d_inv_baseline,
                               const float* d_mu, const float* d_sigma,
                               float* d_snr, int32_t* d_best_h, void* cuda_stream);

/* Spectrum whitening as a pass of its own: d_whitened[s][b] = d_spectra[s][b] * d_inv_baseline[s][b]
 * for b < n_bins, ONE fp32 multiply -- the product the fused path forms (reading R13) -- so that
 * hs_run_*(plan, d_whitened, NULL, ..) returns the bits of hs_run_*(plan, d_spectra, d_inv_baseline, ..) while its
 * gather reads one array instead of two (cfg4: 4.0 + 11.6 ms instead of 26 ms).  d_whitened: device, [S][in_stride],
 * 16-byte aligned, not aliasing the inputs; elements beyond n_bins of a row are not written.  Asynchronous. */
hs_status hs_whiten(hs_plan_t plan, const float* d_spectra, const float* d_inv_baseline, float* d_whitened, void* cuda_stream);

/* The step before the path: "{mu, sigma} = GetMeanStdev()", "the mean and standard deviation ...
 * for partial sum of length H", the pre-processing all algorithms share.  The paper does
 * not define it; reading R14 of DESIGN.md: for every spectrum s and order h, the mean and the population standard
 * deviation over the bins n in [n_lo, n_hi) of the partial sum S_h(n) that the selected form builds at order h
 * (greedy != 0: Alg. 2 with the plan's greedy flags, n the fundamental bin, bins whose order h lies beyond the band
 * edge do not count; greedy == 0: the Alg. 1 family with the plan's PRESTO flags, n the top bin, H' outside the order
 * set get (0, 1)), with the whitening multiplier applied if d_inv_baseline != NULL, followed by n_clip rounds of
 * outlier rejection: round p keeps the sums with lo <= S_h(n) <= hi, lo / hi = mean -/+ clip_sigma * std of round
 * p - 1 rounded to fp32.  An order without samples gets (0, 1); a zero deviation is returned as 1.
 *   n_lo, n_hi   bin range (n_hi = 0: n_bins)
 *   d_mu, d_sigma  [S][H] fp32 out (device): the arguments hs_run_*_dstats take
 *   d_work       device workspace of hs_stats_workspace_bytes(plan, n_clip) bytes, 8-byte aligned (zeroed by the call)
 * S_h is accumulated in fp32 as the coverage kernels do; the moments in fp64 (the order of the fp64 additions is not
 * fixed).  Asynchronous on the stream: n_clip + 1 gather passes over [n_lo, n_hi) and one tiny launch -- or one gather
 * pass and n_clip streaming passes when the workspace has hs_stats_workspace_bytes_cached() bytes (below). */
hs_status hs_estimate_stats(hs_plan_t plan, int32_t greedy, const float* d_spectra, const float* d_inv_baseline,
                            int64_t n_lo, int64_t n_hi, float clip_sigma, int32_t n_clip,
                            float* d_mu, float* d_sigma, void* d_work, int64_t work_bytes, void* cuda_stream);
int64_t hs_stats_workspace_bytes(hs_plan_t plan, int32_t n_clip);   /* -1 on invalid arguments (n_clip in 0..16) */

/* A larger workspace that makes the rejection rounds cheap: hs_stats_workspace_bytes(plan, n_clip) rounded up to 256 bytes
 * plus n_spectra * H * ((n_hi - n_lo) rounded up to 4) floats.  Given at least that many bytes (and n_clip >= 1),
 * hs_estimate_stats writes the sums S_h(n) of its first gather pass into the workspace and rounds 1 .. n_clip stream
 * them back instead of walking every bin's orders again: one gather pass instead of n_clip + 1.  The stored values are
 * the fp32 sums the gather forms, the comparisons and fp64 moments are the same, so the results are those of the
 * small-workspace path (bit-equal where the moments are exact).  cfg4 (1024 x 2^21, bins [N/64, N/32), H = 32): 4 GiB.
 * n_hi = 0 means n_bins; -1 on invalid arguments. */
int64_t hs_stats_workspace_bytes_cached(hs_plan_t plan, int32_t n_clip, int64_t n_lo, int64_t n_hi);

/* hs_estimate_stats for callers that CANNOT ALLOCATE device memory -- the same statistics, the same kernels, but no
 * d_work argument: the accumulators live in an array that is part of the library image.
 *
 * Use it when a cudaMalloc at this point is not an option: a real-time pipeline that partitions device memory once at
 * start-up and must not allocate (or hit the implicit device-wide synchronisation of cudaMalloc / cudaFree) while an
 * observation is running; a plug-in whose host application owns the allocator and passes in nothing but the input and
 * output buffers; a process packed so tightly into a memory pool that a further allocation would fail.  The caller
 * still passes the spectra (and optional multipliers) and the two [S][H] output arrays; everything else is as in
 * hs_estimate_stats, results included (same kernels; fp64 sums in an unspecified order, so bit-equal on exactly
 * representable data and equal to rounding otherwise).
 *
 * Limit: (n_clip + 1) * n_spectra <= HS_STATIC_STATS_MAX_ROWS (4096; e.g. 1024 spectra with three rejection rounds).
 *   Beyond it the call returns HS_ERR_TOO_LARGE and launches nothing -- use hs_estimate_stats with your own workspace,
 *   or split the batch over several plans.
 * Cost: HS_STATIC_STATS_MAX_BYTES (3 MiB) of device memory on every GPU on which this library is loaded, held from
 *   load until the process exits whether or not this entry point is ever called.
 * First call on each device: looks up the device address of the array (one cudaGetSymbolAddress, which may make the
 *   runtime load the library's code on that device).  Make that first call during set-up, BEFORE any CUDA stream capture
 *   is begun; later calls on that device do no such lookup.
 * Sharing: there is ONE array per device, shared by every plan, stream and host thread, and it keeps whatever the last
 *   call left in it.  Each call clears the part it uses on `cuda_stream` before its first kernel, so calls that are
 *   ordered on the device (same stream, or ordered by events) are safe back to back; two calls whose kernels can overlap
 *   on one device (different streams, different host threads, different plans) RACE on the accumulators and return
 *   garbage -- serialise them.
 * The call itself never calls cudaMalloc, cudaFree or any allocating routine; asynchronous on the stream. */
#define HS_STATIC_STATS_MAX_ROWS  4096
#define HS_STATIC_STATS_MAX_BYTES (HS_STATIC_STATS_MAX_ROWS * 32 * 3 * 8)
hs_status hs_estimate_stats_static(hs_plan_t plan, int32_t greedy, const float* d_spectra, const float* d_inv_baseline,
                                   int64_t n_lo, int64_t n_hi, float clip_sigma, int32_t n_clip,
                                   float* d_mu, float* d_sigma, void* cuda_stream);

/* The same two operations with HOST buffers (any host memory; page-locked memory copies
 * fastest).  Spectra are streamed through plan-owned device staging buffers in groups of
 * rows: host->device copy, kernels, device->host copy, overlapped on internal streams.
 * Synchronous.  h_inv_baseline and h_path may be NULL. */
hs_status hs_run_greedy_host(hs_plan_t plan, const float* h_spectra, const float* h_inv_baseline,
                             const float* mu, const float* sigma,
                             float* h_snr, int32_t* h_best_h, uint32_t* h_path);
hs_status hs_run_presto_host(hs_plan_t plan, const float* h_spectra, const float* h_inv_baseline,
                             const float* mu, const float* sigma,
                             float* h_snr, int32_t* h_best_h);

/* Both forms from ONE upload of the spectra: greedy (outputs h_snr_greedy, h_best_h_greedy, optional h_path) and
 * PRESTO (h_snr_presto, h_best_h_presto) with their own statistics; otherwise as the two calls above. */
hs_status hs_run_both_host(hs_plan_t plan, const float* h_spectra, const float* h_inv_baseline,
                           const float* mu_greedy, const float* sigma_greedy,
                           float* h_snr_greedy, int32_t* h_best_h_greedy, uint32_t* h_path,
                           const float* mu_presto, const float* sigma_presto,
                           float* h_snr_presto, int32_t* h_best_h_presto);

/* NEXT-4: 2-D harmonic sums over an f-fdot (acceleration) plane (BASELINE.json configs[4]; the paper only mentions
 * higher-dimensional harmonic sums, and defines no algorithm for them).  Reading R15 of DESIGN.md:
 * the plane is P[z + Z][r], z = -Z .. Z (n_z = 2 Z + 1 rows of n_bins fp32 powers, row stride in_stride); outputs are
 * written for every (z, r) at [z + Z][r] (row stride out_stride).  H <= 16, n_bins <= 2^25, n_z odd.
 *   hs_run_greedy_2d, plan flag HS_GREEDY_NO_DRIFT: the SIMPLE 2-D sum S_h(r, z) = sum_{k <= h} P[k z][k r]
 *     (BASELINE.json's formula at integer (r, z)); order k is evaluated iff k r <= n_bins - 1 and |k z| <= Z, and once
 *     an order is skipped all later ones are; snr_h = (S_h - mu[h-1]) / sigma[h-1], output = the first maximum over h.
 *   hs_run_greedy_2d, no flag: a 2-D GREEDY rule, OURS (not the paper's): drifts d_r = d_z = 0; at order h let
 *     m = h r + d_r, w = h z + d_z (stop if m > n_bins - 1 or |w| > Z); the candidates are P[w][m], P[w][m+1],
 *     P[w+1][m], P[w+1][m+1] (those outside the plane never win; at h = 1 only P[w][m] under
 *     HS_GREEDY_NO_FUND_SELECT); the largest is added, ties going to the first in that order, and d_r / d_z grow by
 *     one if it lies at m+1 / w+1.  d_path (nullable): bit h-1 = r-shift at order h, bit 16+h-1 = z-shift.
 *   hs_run_presto_2d: the PRESTO-like form: the output index (r, z) is the TOP harmonic; for H' in the order set
 *     S = sum over k in {1} U {2,4,..,H'} (1..H' under HS_PRESTO_ALL_HARMONICS) of
 *     P[Round(k z / H')][Round(k r / H')], Round(a / b) = floor((2a + b) / (2b)) (half up, also for negative z).
 * mu, sigma: HOST arrays of H floats.  Asynchronous on the stream.  The 1-D entry points reject a 2-D plan and vice
 * versa; hs_find_candidates accepts both (spectrum = z + Z). */
hs_status hs_plan_2d(hs_plan_t* plan, int64_t n_bins, int32_t n_z, int32_t H,
                     int64_t in_stride, int64_t out_stride, uint32_t flags, int32_t device);
hs_status hs_run_greedy_2d(hs_plan_t plan, const float* d_plane, const float* mu, const float* sigma,
                           float* d_snr, int32_t* d_best_h, uint32_t* d_path, void* cuda_stream);
hs_status hs_run_presto_2d(hs_plan_t plan, const float* d_plane, const float* mu, const float* sigma,
                           float* d_snr, int32_t* d_best_h, void* cuda_stream);

/* One detection (reading R11 of DESIGN.md: a bin whose maximum SNR reaches the threshold). */
typedef struct {
    int32_t spectrum;   /* row s of the batch */
    int32_t bin;        /* n (greedy: the fundamental bin; PRESTO: the top bin) */
    float   snr;        /* d_snr[s][n] */
    int32_t best_h;     /* d_best_h[s][n] */
} hs_candidate;

/* Candidate list of a finished run: every (s, n), n < n_fund, with d_snr[s][n] >= threshold (NaN never
 * qualifies), in unspecified order (sort by (spectrum, bin) for a canonical list).
 *   d_snr, d_best_h  outputs of hs_run_greedy / hs_run_presto of the same plan (device, [S][out_stride])
 *   d_out            device array of `capacity` hs_candidate (16-byte aligned); may be NULL if capacity = 0
 *   d_count          device uint64: set to the number of qualifying bins, which may exceed `capacity`
 *                    (then only `capacity` of them were stored: call again with a larger array)
 * Asynchronous on the stream; one streaming pass over d_snr. */
hs_status hs_find_candidates(hs_plan_t plan, const float* d_snr, const int32_t* d_best_h, float threshold,
                             hs_candidate* d_out, int64_t capacity, uint64_t* d_count, void* cuda_stream);

/* The search as one call on HOST buffers: the spectra are uploaded once (in groups of rows through the plan's staging
 * slots, two streams), both forms run on the device, their outputs are thresholded and compacted THERE, and only the two
 * candidate lists travel back -- the per-bin outputs never leave the device.  Lists as hs_find_candidates defines them
 * (unspecified order; *h_count_* = the number of qualifying bins, which may exceed the capacity: then only `capacity`
 * records were stored).  h_cand_* are HOST arrays.  Synchronous.  The plan owns the device lists it compacts into. */
hs_status hs_search_host(hs_plan_t plan, const float* h_spectra, const float* h_inv_baseline,
                         const float* mu_greedy, const float* sigma_greedy, const float* mu_presto, const float* sigma_presto,
                         float threshold, hs_candidate* h_cand_greedy, int64_t capacity_greedy, uint64_t* h_count_greedy,
                         hs_candidate* h_cand_presto, int64_t capacity_presto, uint64_t* h_count_presto);

/* UNSTABLE, diagnostics only (not part of the method's interface; values may change between versions):
 * selects a kernel variant for the plan's later runs.  0 = the library's choice; 255 = the plain
 * one-thread-per-bin coverage kernels.  Every variant computes the results defined above. */
hs_status hs_plan_set_tuning(hs_plan_t plan, uint32_t variant);

/* UNSTABLE: input bytes per device staging slot of the *_host entry points (default 256 MiB; a slot holds at least one
 * spectrum).  Must be called before the plan's first *_host call, which allocates the slots (HS_ERR_INVALID_ARG after). */
hs_status hs_plan_set_host_slot_bytes(hs_plan_t plan, int64_t bytes);

/* Number of kernels this plan has launched so far (for bench.py's gpu_launches). */
int64_t hs_launch_count(hs_plan_t plan);

/* Name of the kernel variant the plan launched last ("" before the first run): bench.py keys its committed
 * ncu evidence (profiles/) by this name.  Static string. */
const char* hs_last_kernel(hs_plan_t plan);

/* Release the plan and everything it owns.  NULL is accepted. */
hs_status hs_destroy(hs_plan_t plan);

/* Static description of a status code. */
const char* hs_status_string(hs_status s);

/* cudaError_t of the most recent HS_ERR_CUDA on this host thread (0 if none). */
int32_t hs_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* HS_B200_H_ */
