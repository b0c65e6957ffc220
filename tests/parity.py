"""GPU-vs-oracle acceptance rules (SURVEY.md 8(c) 'GPU-vs-oracle acceptance', north_star checks a-c).

(a) greedy path bit-exact everywhere (it depends only on comparisons of identical fp32 inputs);
    best_h equal to the oracle's, or any order whose ORACLE snr lies within
    tol = 2e-5 * max(1, |best|, mu_H/sigma_H) of the oracle's best (near-tie set);
(b) |snr_gpu - snr_ref| <= 1e-5 |snr_ref| where snr_ref >= 1, else <= 1e-5 (|S| + mu)/sigma
    (a pure relative bound is unattainable where S ~ mu cancels; fp32 accumulation of <= 32
    positive terms carries <~ 2e-6 relative error on S);
(c) candidate sets {(s, n, best_h): snr >= T} equal, except bins whose oracle snr is within tol of T.
"""
import numpy as np

REL = 1e-5


def _tol(best, mu, sg):
    return 2e-5 * np.maximum(np.maximum(1.0, np.abs(best)), float(mu[-1]) / float(sg[-1]))


def _check_common(snr_ref, bh_ref, snr_gpu, bh_gpu, mu, sg, per_order_fn, T):
    mu = np.asarray(mu, np.float64)
    sg = np.asarray(sg, np.float64)
    snr_gpu = snr_gpu.astype(np.float64)
    assert np.all(np.isfinite(snr_gpu)), "non-finite snr from the GPU"
    tol = _tol(snr_ref, mu, sg)
    # (a) best_h: equal, or inside the oracle's near-tie set
    bad = np.argwhere(bh_gpu != bh_ref)
    if bad.size:
        assert np.all((bh_gpu[bad[:, 0], bad[:, 1]] >= 1) & (bh_gpu[bad[:, 0], bad[:, 1]] <= mu.size))
        snr_h = per_order_fn(bad[:, 0], bad[:, 1])                 # oracle per-order snr [k, H]
        got = snr_h[np.arange(bad.shape[0]), bh_gpu[bad[:, 0], bad[:, 1]] - 1]
        ok = got >= snr_ref[bad[:, 0], bad[:, 1]] - tol[bad[:, 0], bad[:, 1]]
        assert np.all(ok), f"best_h outside the near-tie set at {bad[~ok][:5]}"
    # (b) snr
    S = snr_ref * sg[bh_ref - 1] + mu[bh_ref - 1]
    bound = np.where(snr_ref >= 1.0, REL * np.abs(snr_ref), REL * (np.abs(S) + mu[bh_ref - 1]) / sg[bh_ref - 1])
    err = np.abs(snr_gpu - snr_ref)
    assert np.all(err <= bound), f"snr error {err.max()} exceeds bound at {np.argwhere(err > bound)[:5]}"
    # (c) candidates
    if T is not None:
        near = np.abs(snr_ref - T) <= tol
        cg = (snr_gpu >= T) & ~near
        cr = (snr_ref >= T) & ~near
        assert np.array_equal(cg, cr), "candidate lists differ"
        sel = cr & (bh_gpu == bh_ref)
        assert np.count_nonzero(cr & ~sel) <= np.count_nonzero(bh_gpu != bh_ref)
    return dict(max_err=float(err.max()), bh_mismatch=int(bad.shape[0]))


def check_greedy(oracle, x, H, mu, sg, flags, snr_gpu, bh_gpu, path_gpu, inv_baseline=None, T=10.0, n_fund=None):
    snr_ref, bh_ref, path_ref = oracle.greedy(x, H, mu, sg, flags, inv_baseline=inv_baseline, n_fund=n_fund)
    if path_gpu is not None:
        assert np.array_equal(path_gpu.view(np.uint32), path_ref), "greedy path differs"   # (a) bit-exact

    def per_order(rows, bins):
        return oracle.greedy_bins(x, H, mu, sg, rows, bins, flags, inv_baseline=inv_baseline)["snr_h"]

    return _check_common(snr_ref, bh_ref, snr_gpu, bh_gpu, mu, sg, per_order, T)


def check_presto(oracle, x, H, mu, sg, flags, snr_gpu, bh_gpu, inv_baseline=None, T=10.0, n_fund=None):
    snr_ref, bh_ref = oracle.presto(x, H, mu, sg, flags, inv_baseline=inv_baseline, n_fund=n_fund)

    def per_order(rows, bins):
        return oracle.presto_bins(x, H, mu, sg, rows, bins, flags, inv_baseline=inv_baseline)["snr_h"]

    return _check_common(snr_ref, bh_ref, snr_gpu, bh_gpu, mu, sg, per_order, T)
