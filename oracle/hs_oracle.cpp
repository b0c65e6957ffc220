// =====================================================================================
// hs_oracle.cpp -- CPU ORACLE for the incoherent 1-D harmonic sum of arXiv 2202.12817.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
// header, table or helper with the CUDA path (paper_2202_12817_b200/csrc, include/hs.h);
// the flag values below are restated here on purpose.
//
// It is a plain, slow, double-precision restatement of the paper's algorithms, one
// fundamental (or top) bin at a time, in the paper's order and notation:
//
//   * eq. 2   SNR = max_H (X_H - mu_H) / sigma_H; only the max and its H
//                               are returned per bin.
//   * Alg. 2 greedy harmonic sum; eq. 5 m = h n + d;
//                               fundamental-bin selection.
//   * eq. 3     simple harmonic sum = greedy with the drift held at 0.
//   * Alg. 1 PRESTO harmonic sum; eq. 4 x[round(h n / H)],
//                               n = LAST bin of the series; H' in powers of two,
//                               fundamental + even harmonics.
//   * PRESTO_all / PRESTO+ (PAPER.md:174, 368): all harmonics / additionally every H' = 1..H.
//
// Neither algorithm reaches a plainly-defined result faster -- both are heuristics that
// choose WHICH bins to add -- so the oracle is the algorithm itself, step by step.
// Inputs are the caller's fp32 powers; all sums and SNRs are formed in fp64.
//
// Readings of the paper adopted here:
//   R1  every bin n in [0, n_fund) gets an output (eq. 12 counts all bins).
//   R2  PRESTO computes the SNR once per H', after the inner loop, with mu[H'], sigma[H'].
//   R3  Round() = round-half-up in exact integers: (2 h n + H') / (2 H').      [parity unpinned]
//   R4  greedy: order h is evaluated iff m = h n + d <= N-1; a missing second bin (m+1 = N)
//       never wins; once an order is skipped all later ones are.                [parity unpinned]
//   R5  H steps in total, harmonic ORDERS 1..H, statistics indexed by order.
//   R6  CompareSNR keeps the first maximum (strict >); best starts at -inf, no clamp at 0,
//       so best_h is in [1, H].                                                 [parity unpinned]
//   R7  fundamental selection on by default; a flag disables it.
//   R8  mu[h-1], sigma[h-1] are inputs (the statistics of the partial sum at order h).
//   R14 GetMeanStdev() ("mean and standard deviation for partial sum of length H", PAPER.md:58;
//       "all algorithms use the same pre-processing steps (mean and standard deviation calculation ...)")
//       is not defined by the paper.  Reading (hs_oracle_estimate_stats below): per spectrum and per order h, the
//       sample mean and the population standard deviation, over the bins n of a caller-chosen range [n_lo, n_hi), of
//       the partial sum S_h(n) that the selected variant forms at order h (bins whose order h is not evaluated do not
//       count), followed by n_clip rounds of outlier rejection: round p keeps the sums with
//       lo <= S_h(n) <= hi, lo/hi = mean -/+ clip * std of round p-1 rounded to fp32.  An order without samples gets
//       (mu, sigma) = (0, 1); a zero standard deviation is returned as 1.
//   R15 (NEXT-4, 2-D harmonic sum over the f-fdot plane; the paper only mentions it; BASELINE.json
//       configs[4] gives S_h(r,z) = sum_{k<=h} P[round(k r), round(k z)]): the plane is P[z + Z][r], z in [-Z, Z];
//       SIMPLE 2-D sum = that formula at integer (r, z); order k is evaluated iff k r <= N-1 and |k z| <= Z, and once an
//       order is skipped all later ones are (as R4).  PRESTO-like 2-D: the output is indexed by the TOP harmonic (r, z)
//       and the terms sit at (Round(k r / H'), Round(k z / H')), Round = round half up = floor((2a + b) / (2b)) also
//       for negative z.  GREEDY 2-D is OURS (the paper defines no 2-D greedy rule): drifts d_r, d_z >= 0; at order h
//       the candidates are the 2 x 2 block P[w..w+1][m..m+1], m = h r + d_r, w = h z + d_z; the largest is added (ties:
//       the first of (m,w), (m+1,w), (m,w+1), (m+1,w+1)) and the drifts follow it; candidates outside the plane never
//       win; path bit h-1 = r-shift at order h, bit 16+h-1 = z-shift (H <= 16).
//   NEXT-2: an optional per-bin multiplier inv_baseline[] whitens the spectrum; the product
//       x*inv_baseline is formed in fp32 (one IEEE multiply -- the kernel's precision --
//       because it decides the greedy comparison), everything after it in fp64.
//
// Pins (tests/test_oracle_pins.py, tests/golden/): P1 identity at H = 1, P2 constant
// spectrum closed form, P3 delta train, P4 the paper's worked index example
// (PAPER.md:170, 172), P5 brute force on tiny spectra (exact rational rounding; path-tree
// enumeration), P6 invariants, P7 exact-integer spectra, P8 Exp(1) noise statistics.
// Parity unpinned by anything the paper prints: R3 (tie rule of Round), R4 (band edge),
// R6 (tie-breaks), R14 (what GetMeanStdev() estimates) and R15 (the 2-D sums: the paper defines none);
// they are fixed by the readings above and pinned against independent restatements only
// (numpy moments of numpy gathers; exact-rational brute force; the z = 0 row = the 1-D sums).
// =====================================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <thread>
#include <vector>

namespace {

// Flag values restated from the boundary's documentation (not included from include/hs.h).
constexpr uint32_t F_NO_FUND_SELECT = 1u << 0;  // greedy: order 1 takes x[n] without looking at x[n+1]
constexpr uint32_t F_NO_DRIFT = 1u << 1;        // greedy: simple harmonic sum, eq. 3
constexpr uint32_t F_ALL_HARMONICS = 1u << 2;   // PRESTO_all
constexpr uint32_t F_ALL_ORDERS = 1u << 3;      // with ALL_HARMONICS: PRESTO+

struct Spectrum {
    const float* x;        // N powers
    const float* invb;     // optional per-bin multiplier (may be null)
    int64_t N;
    // Power at bin m as the method sees it.
    double at(int64_t m) const {
        if (invb) {
            volatile float p = x[m] * invb[m];   // one fp32 multiply (kernel's precision)
            return (double)p;
        }
        return (double)x[m];
    }
};

struct Stats {
    const float* mu;
    const float* sigma;
    double snr(double sum, int order) const {   // eq. 2 term for harmonic order `order` (1-based)
        return (sum - (double)mu[order - 1]) / (double)sigma[order - 1];
    }
};

const double NEG_INF = -std::numeric_limits<double>::infinity();

// ---- Algorithm 2 (greedy) for one fundamental bin n --------------------------------
// snr_h / bin_h (optional, length H): per-order SNR (NaN if the order was not evaluated)
// and the bin that was added at that order (-1 if none).
void greedy_bin(const Spectrum& sp, int H, const Stats& st, uint32_t flags, int64_t n,
                double* best_out, int32_t* besth_out, uint32_t* path_out,
                double* snr_h, int64_t* bin_h) {
    const int64_t N = sp.N;
    int64_t d = 0;          // drift
    double sum = 0.0;
    double best = NEG_INF;  // R6: no clamp at zero
    int32_t bh = 0;
    uint32_t path = 0;
    if (snr_h) for (int h = 0; h < H; ++h) snr_h[h] = std::nan("");
    if (bin_h) for (int h = 0; h < H; ++h) bin_h[h] = -1;
    for (int h = 1; h <= H; ++h) {
        const int64_t m = (int64_t)h * n + d;            // eq. 5
        if (m > N - 1) break;                            // R4
        const double xd = sp.at(m);                      // x_d
        double xd1 = (m + 1 <= N - 1) ? sp.at(m + 1) : NEG_INF;   // x_(d+1); R4
        if (h == 1 && (flags & F_NO_FUND_SELECT)) xd1 = NEG_INF;  // R7
        if (flags & F_NO_DRIFT) xd1 = NEG_INF;                    // eq. 3
        int64_t picked = m;
        if (xd1 > xd) {                                  // strict >, ties stay
            d += 1;
            sum += xd1;
            path |= (1u << (h - 1));
            picked = m + 1;
        } else {
            sum += xd;
        }
        const double s = st.snr(sum, h);                 // CalculateSNR
        if (snr_h) snr_h[h - 1] = s;
        if (bin_h) bin_h[h - 1] = picked;
        if (s > best) { best = s; bh = h; }              // CompareSNR, R6
    }
    *best_out = best;
    *besth_out = bh;
    if (path_out) *path_out = path;
}

// ---- Algorithm 1 (PRESTO family) for one top bin n -----------------------------------
inline bool order_in_set(int Hp, uint32_t flags) {
    if (flags & F_ALL_ORDERS) return true;               // PRESTO+: every H' = 1..H
    return (Hp & (Hp - 1)) == 0;                         // H' = 1, 2, 4, ...
}

inline int64_t presto_index(int h, int Hp, int64_t n) {  // Round(h/H' n), R3
    return (2 * (int64_t)h * n + Hp) / (2 * (int64_t)Hp);
}

void presto_bin(const Spectrum& sp, int H, const Stats& st, uint32_t flags, int64_t n,
                double* best_out, int32_t* besth_out, double* snr_h) {
    double best = NEG_INF;
    int32_t bh = 0;
    if (snr_h) for (int h = 0; h < H; ++h) snr_h[h] = std::nan("");
    for (int Hp = 1; Hp <= H; ++Hp) {
        if (!order_in_set(Hp, flags)) continue;
        // fundamental frequency bin
        double sum = sp.at(presto_index(1, Hp, n));
        if (flags & F_ALL_HARMONICS) {
            for (int h = 2; h <= Hp; ++h) sum += sp.at(presto_index(h, Hp, n));
        } else {
            for (int h = 2; h <= Hp; h += 2) sum += sp.at(presto_index(h, Hp, n));
        }
        const double s = st.snr(sum, Hp);                // R2: once per H'
        if (snr_h) snr_h[Hp - 1] = s;
        if (s > best) { best = s; bh = Hp; }
    }
    *best_out = best;
    *besth_out = bh;
}

bool bad_common(const float* x, int64_t N, int32_t S, int32_t H, const float* mu, const float* sigma) {
    if (!x || !mu || !sigma || N < 2 || S < 1 || H < 1 || H > 32) return true;
    for (int h = 0; h < H; ++h) if (!(sigma[h] > 0.0f)) return true;
    return false;
}

template <class F>
void parallel_for_rows(int32_t S, int64_t n_fund, int n_threads, F&& body) {
    // split (spectrum, bin-range) work items over threads
    if (n_threads < 1) n_threads = 1;
    const int64_t chunk = 1 << 16;
    const int64_t chunks_per_row = (n_fund + chunk - 1) / chunk;
    const int64_t total = (int64_t)S * chunks_per_row;
    auto worker = [&](int t) {
        for (int64_t w = t; w < total; w += n_threads) {
            const int32_t s = (int32_t)(w / chunks_per_row);
            const int64_t lo = (w % chunks_per_row) * chunk;
            const int64_t hi = (lo + chunk < n_fund) ? lo + chunk : n_fund;
            body(s, lo, hi);
        }
    };
    if (n_threads == 1) { worker(0); return; }
    std::vector<std::thread> th;
    for (int t = 0; t < n_threads; ++t) th.emplace_back(worker, t);
    for (auto& t : th) t.join();
}

}  // namespace

extern "C" {

// Greedy harmonic sum (Alg. 2) over a batch.  x: [S][in_stride] fp32 (first N of each row used);
// inv_baseline: same layout or null; mu/sigma: H floats, index h-1; outputs [S][out_stride]:
// snr fp64, best_h int32, path uint32 (nullable; bit h-1 set iff the drift grew at order h).
// Bins n >= n_fund are not written.  Returns 0, or 1 on invalid arguments.
int hs_oracle_greedy(const float* x, const float* inv_baseline, int64_t N, int32_t S, int64_t in_stride,
                     int32_t H, const float* mu, const float* sigma, uint32_t flags, int64_t n_fund,
                     double* snr, int32_t* best_h, uint32_t* path, int64_t out_stride, int32_t n_threads) {
    if (bad_common(x, N, S, H, mu, sigma) || !snr || !best_h) return 1;
    if (in_stride < N || out_stride < n_fund || n_fund < 0 || n_fund > N) return 1;
    const Stats st{mu, sigma};
    parallel_for_rows(S, n_fund, n_threads, [&](int32_t s, int64_t lo, int64_t hi) {
        const Spectrum sp{x + (int64_t)s * in_stride, inv_baseline ? inv_baseline + (int64_t)s * in_stride : nullptr, N};
        for (int64_t n = lo; n < hi; ++n) {
            const int64_t o = (int64_t)s * out_stride + n;
            greedy_bin(sp, H, st, flags, n, &snr[o], &best_h[o], path ? &path[o] : nullptr, nullptr, nullptr);
        }
    });
    return 0;
}

// PRESTO family (Alg. 1) over a batch; same conventions.  Output index n is the TOP bin (R10).
int hs_oracle_presto(const float* x, const float* inv_baseline, int64_t N, int32_t S, int64_t in_stride,
                     int32_t H, const float* mu, const float* sigma, uint32_t flags, int64_t n_fund,
                     double* snr, int32_t* best_h, int64_t out_stride, int32_t n_threads) {
    if (bad_common(x, N, S, H, mu, sigma) || !snr || !best_h) return 1;
    if (in_stride < N || out_stride < n_fund || n_fund < 0 || n_fund > N) return 1;
    if ((flags & F_ALL_ORDERS) && !(flags & F_ALL_HARMONICS)) return 1;
    const Stats st{mu, sigma};
    parallel_for_rows(S, n_fund, n_threads, [&](int32_t s, int64_t lo, int64_t hi) {
        const Spectrum sp{x + (int64_t)s * in_stride, inv_baseline ? inv_baseline + (int64_t)s * in_stride : nullptr, N};
        for (int64_t n = lo; n < hi; ++n) {
            const int64_t o = (int64_t)s * out_stride + n;
            presto_bin(sp, H, st, flags, n, &snr[o], &best_h[o], nullptr);
        }
    });
    return 0;
}

// One bin at a time, with the per-order detail: used for sampled checks at full size and for the
// near-tie sets of the acceptance rule.  rows/bins: `count` (spectrum, bin) pairs.
// snr_h: [count][H] per-order SNR (NaN where the order was not evaluated);
// bin_h: [count][H] bin added at each order (-1 if none) -- nullable.
int hs_oracle_greedy_bins(const float* x, const float* inv_baseline, int64_t N, int64_t in_stride, int32_t H,
                          const float* mu, const float* sigma, uint32_t flags,
                          const int64_t* rows, const int64_t* bins, int64_t count,
                          double* snr, int32_t* best_h, uint32_t* path, double* snr_h, int64_t* bin_h) {
    if (bad_common(x, N, 1, H, mu, sigma) || !rows || !bins || !snr || !best_h) return 1;
    const Stats st{mu, sigma};
    for (int64_t i = 0; i < count; ++i) {
        if (bins[i] < 0 || bins[i] >= N) return 1;
        const Spectrum sp{x + rows[i] * in_stride, inv_baseline ? inv_baseline + rows[i] * in_stride : nullptr, N};
        greedy_bin(sp, H, st, flags, bins[i], &snr[i], &best_h[i], path ? &path[i] : nullptr,
                   snr_h ? snr_h + i * H : nullptr, bin_h ? bin_h + i * H : nullptr);
    }
    return 0;
}

int hs_oracle_presto_bins(const float* x, const float* inv_baseline, int64_t N, int64_t in_stride, int32_t H,
                          const float* mu, const float* sigma, uint32_t flags,
                          const int64_t* rows, const int64_t* bins, int64_t count,
                          double* snr, int32_t* best_h, double* snr_h) {
    if (bad_common(x, N, 1, H, mu, sigma) || !rows || !bins || !snr || !best_h) return 1;
    if ((flags & F_ALL_ORDERS) && !(flags & F_ALL_HARMONICS)) return 1;
    const Stats st{mu, sigma};
    for (int64_t i = 0; i < count; ++i) {
        if (bins[i] < 0 || bins[i] >= N) return 1;
        const Spectrum sp{x + rows[i] * in_stride, inv_baseline ? inv_baseline + rows[i] * in_stride : nullptr, N};
        presto_bin(sp, H, st, flags, bins[i], &snr[i], &best_h[i], snr_h ? snr_h + i * H : nullptr);
    }
    return 0;
}

// R14: the statistics of the partial sums (the reading of GetMeanStdev() in the header).  greedy != 0: Alg. 2 with
// `flags`; else the PRESTO family with `flags` (orders outside its order set get (0, 1)).
// mu, sigma: [S][H] fp32 out; count: [S][H] int64 out (samples kept in the last round; nullable).
int hs_oracle_estimate_stats(const float* x, const float* inv_baseline, int64_t N, int32_t S, int64_t in_stride,
                             int32_t H, uint32_t flags, int32_t greedy, int64_t n_lo, int64_t n_hi,
                             double clip, int32_t n_clip, float* mu, float* sigma, int64_t* count) {
    if (!x || !mu || !sigma || N < 2 || S < 1 || H < 1 || H > 32 || in_stride < N) return 1;
    if (n_lo < 0 || n_hi > N || n_lo > n_hi || n_clip < 0 || !(clip > 0.0)) return 1;
    if (!greedy && (flags & F_ALL_ORDERS) && !(flags & F_ALL_HARMONICS)) return 1;
    std::vector<float> zero(H, 0.0f), one(H, 1.0f);
    const Stats unit{zero.data(), one.data()};               // (sum - 0) / 1 = the partial sum itself
    std::vector<double> sums(H);
    for (int32_t s = 0; s < S; ++s) {
        const Spectrum sp{x + (int64_t)s * in_stride, inv_baseline ? inv_baseline + (int64_t)s * in_stride : nullptr, N};
        std::vector<double> lo(H, NEG_INF), hi(H, -NEG_INF), mean(H, 0.0), sd(H, 0.0);
        std::vector<int64_t> cnt(H, 0);
        for (int p = 0; p <= n_clip; ++p) {
            std::vector<double> a1(H, 0.0), a2(H, 0.0);
            std::fill(cnt.begin(), cnt.end(), 0);
            for (int64_t n = n_lo; n < n_hi; ++n) {
                double best; int32_t bh;
                if (greedy) greedy_bin(sp, H, unit, flags, n, &best, &bh, nullptr, sums.data(), nullptr);
                else presto_bin(sp, H, unit, flags, n, &best, &bh, sums.data());
                for (int h = 0; h < H; ++h) {
                    const double v = sums[h];
                    if (v != v) continue;                    // order not evaluated for this bin
                    if (v < lo[h] || v > hi[h]) continue;    // rejected by the previous round
                    cnt[h] += 1; a1[h] += v; a2[h] += v * v;
                }
            }
            for (int h = 0; h < H; ++h) {
                if (cnt[h] == 0) { mean[h] = 0.0; sd[h] = 0.0; continue; }
                mean[h] = a1[h] / (double)cnt[h];
                const double var = a2[h] / (double)cnt[h] - mean[h] * mean[h];
                sd[h] = var > 0.0 ? std::sqrt(var) : 0.0;
                lo[h] = (double)(float)(mean[h] - clip * sd[h]);
                hi[h] = (double)(float)(mean[h] + clip * sd[h]);
            }
        }
        for (int h = 0; h < H; ++h) {
            mu[(int64_t)s * H + h] = cnt[h] ? (float)mean[h] : 0.0f;
            sigma[(int64_t)s * H + h] = (cnt[h] && sd[h] > 0.0) ? (float)sd[h] : 1.0f;
            if (count) count[(int64_t)s * H + h] = cnt[h];
        }
    }
    return 0;
}

// ---- R15: 2-D harmonic sums over an f-fdot plane P[n_z][stride], n_z = 2 Z + 1 (NEXT-4) ----------------------------
namespace {
inline int64_t floor_div(int64_t a, int64_t b) { int64_t q = a / b; if ((a % b != 0) && ((a < 0) != (b < 0))) --q; return q; }
inline int64_t round_half_up(int64_t a, int64_t b) { return floor_div(2 * a + b, 2 * b); }   // Round(a / b), b > 0

struct Plane {
    const float* p; int64_t N, stride; int32_t Z;
    double at(int64_t z, int64_t r) const { return (double)p[(z + Z) * stride + r]; }
};

// snr_h (nullable): the SNR of every order, NaN for the orders that were not evaluated -- for the near-tie rule of the
// parity tests only; nothing of the sum depends on it
void greedy2d_bin(const Plane& pl, int H, const Stats& st, uint32_t flags, int64_t r, int64_t z,
                  double* best_out, int32_t* besth_out, uint32_t* path_out, double* snr_h = nullptr) {
    if (snr_h) for (int h = 0; h < H; ++h) snr_h[h] = std::numeric_limits<double>::quiet_NaN();
    int64_t dr = 0, dz = 0;
    double sum = 0.0, best = NEG_INF;
    int32_t bh = 0;
    uint32_t path = 0;
    for (int h = 1; h <= H; ++h) {
        const int64_t m = (int64_t)h * r + dr, w = (int64_t)h * z + dz;
        if (m > pl.N - 1 || w < -pl.Z || w > pl.Z) break;
        const bool drift = !(flags & F_NO_DRIFT) && !(h == 1 && (flags & F_NO_FUND_SELECT));
        const bool r1 = drift && m + 1 <= pl.N - 1, z1 = drift && w + 1 <= pl.Z;
        const double c[4] = {pl.at(w, m), r1 ? pl.at(w, m + 1) : NEG_INF, z1 ? pl.at(w + 1, m) : NEG_INF,
                             (r1 && z1) ? pl.at(w + 1, m + 1) : NEG_INF};
        int pick = 0;
        for (int k = 1; k < 4; ++k) if (c[k] > c[pick]) pick = k;      // strict >: the first maximum stays
        if (pick & 1) { dr += 1; path |= 1u << (h - 1); }
        if (pick & 2) { dz += 1; path |= 1u << (16 + h - 1); }
        sum += c[pick];
        const double s = st.snr(sum, h);
        if (snr_h) snr_h[h - 1] = s;
        if (s > best) { best = s; bh = h; }
    }
    *best_out = best; *besth_out = bh;
    if (path_out) *path_out = path;
}

void presto2d_bin(const Plane& pl, int H, const Stats& st, uint32_t flags, int64_t r, int64_t z,
                  double* best_out, int32_t* besth_out, double* snr_h = nullptr) {
    if (snr_h) for (int h = 0; h < H; ++h) snr_h[h] = std::numeric_limits<double>::quiet_NaN();
    double best = NEG_INF;
    int32_t bh = 0;
    for (int Hp = 1; Hp <= H; ++Hp) {
        if (!order_in_set(Hp, flags)) continue;
        double sum = pl.at(round_half_up(z, Hp), round_half_up(r, Hp));
        const int step = (flags & F_ALL_HARMONICS) ? 1 : 2;
        for (int k = 2; k <= Hp; k += step) sum += pl.at(round_half_up((int64_t)k * z, Hp), round_half_up((int64_t)k * r, Hp));
        const double s = st.snr(sum, Hp);
        if (snr_h) snr_h[Hp - 1] = s;
        if (s > best) { best = s; bh = Hp; }
    }
    *best_out = best; *besth_out = bh;
}
}  // namespace

// The two 2-D forms for selected (row zi = z + Z, column r) pairs, with the SNR of every order ([count][H], NaN where an
// order was not evaluated): what the parity tests need to apply the near-tie rule on a plane.
int hs_oracle_2d_bins(const float* plane, int64_t N, int32_t n_z, int64_t stride, int32_t H, const float* mu, const float* sigma,
                      uint32_t flags, int32_t greedy, const int64_t* zi, const int64_t* r, int64_t count,
                      double* snr, int32_t* best_h, double* snr_h) {
    if (bad_common(plane, N, n_z, H, mu, sigma) || H > 16 || !(n_z & 1) || !zi || !r || !snr || !best_h || !snr_h || stride < N) return 1;
    if (!greedy && (flags & F_ALL_ORDERS) && !(flags & F_ALL_HARMONICS)) return 1;
    const Stats st{mu, sigma};
    const Plane pl{plane, N, stride, (n_z - 1) / 2};
    for (int64_t i = 0; i < count; ++i) {
        if (zi[i] < 0 || zi[i] >= n_z || r[i] < 0 || r[i] >= N) return 1;
        if (greedy) greedy2d_bin(pl, H, st, flags, r[i], zi[i] - pl.Z, &snr[i], &best_h[i], nullptr, snr_h + i * H);
        else presto2d_bin(pl, H, st, flags, r[i], zi[i] - pl.Z, &snr[i], &best_h[i], snr_h + i * H);
    }
    return 0;
}

// plane: [n_z][stride] fp32, n_z odd; outputs [n_z][out_stride], only rows zi_lo <= z + Z < zi_hi are computed and
// written (the sums still read the whole plane); H <= 16.  Returns 0, or 1 on invalid arguments.
int hs_oracle_greedy_2d(const float* plane, int64_t N, int32_t n_z, int64_t stride, int32_t H, const float* mu, const float* sigma,
                        uint32_t flags, double* snr, int32_t* best_h, uint32_t* path, int64_t out_stride, int32_t n_threads,
                        int32_t zi_lo, int32_t zi_hi) {
    if (bad_common(plane, N, n_z, H, mu, sigma) || H > 16 || !(n_z & 1) || !snr || !best_h || stride < N || out_stride < N) return 1;
    if (zi_lo < 0 || zi_hi > n_z || zi_lo > zi_hi) return 1;
    const Stats st{mu, sigma};
    const Plane pl{plane, N, stride, (n_z - 1) / 2};
    parallel_for_rows(zi_hi - zi_lo, N, n_threads, [&](int32_t row, int64_t lo, int64_t hi) {
        const int32_t zi = zi_lo + row;
        for (int64_t r = lo; r < hi; ++r) {
            const int64_t o = (int64_t)zi * out_stride + r;
            greedy2d_bin(pl, H, st, flags, r, (int64_t)zi - pl.Z, &snr[o], &best_h[o], path ? &path[o] : nullptr);
        }
    });
    return 0;
}

int hs_oracle_presto_2d(const float* plane, int64_t N, int32_t n_z, int64_t stride, int32_t H, const float* mu, const float* sigma,
                        uint32_t flags, double* snr, int32_t* best_h, int64_t out_stride, int32_t n_threads,
                        int32_t zi_lo, int32_t zi_hi) {
    if (bad_common(plane, N, n_z, H, mu, sigma) || H > 16 || !(n_z & 1) || !snr || !best_h || stride < N || out_stride < N) return 1;
    if ((flags & F_ALL_ORDERS) && !(flags & F_ALL_HARMONICS)) return 1;
    if (zi_lo < 0 || zi_hi > n_z || zi_lo > zi_hi) return 1;
    const Stats st{mu, sigma};
    const Plane pl{plane, N, stride, (n_z - 1) / 2};
    parallel_for_rows(zi_hi - zi_lo, N, n_threads, [&](int32_t row, int64_t lo, int64_t hi) {
        const int32_t zi = zi_lo + row;
        for (int64_t r = lo; r < hi; ++r) {
            const int64_t o = (int64_t)zi * out_stride + r;
            presto2d_bin(pl, H, st, flags, r, (int64_t)zi - pl.Z, &snr[o], &best_h[o]);
        }
    });
    return 0;
}

int64_t hs_oracle_round_half_up(int64_t a, int64_t b) { return round_half_up(a, b); }

// Index helpers exposed so the pins can check them against the paper's worked example
// (bin 800 is the last element of fundamental 100 at H = 8 and of 200 at H = 4).
int64_t hs_oracle_presto_index(int32_t h, int32_t Hp, int64_t n) { return presto_index(h, Hp, n); }
int32_t hs_oracle_presto_order_in_set(int32_t Hp, uint32_t flags) { return order_in_set(Hp, flags) ? 1 : 0; }

int32_t hs_oracle_hardware_threads(void) {
    unsigned n = std::thread::hardware_concurrency();
    return n ? (int32_t)n : 1;
}

}  // extern "C"
