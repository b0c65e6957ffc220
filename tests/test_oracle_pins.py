"""Pins for the CPU oracle (oracle/hs_oracle.cpp) -- nothing here touches the CUDA path.

Each test fixes the oracle to something other than itself: values the paper prints
(tests/golden/), closed forms, brute-force enumeration with independent (exact rational)
index arithmetic, library routines (numpy gathers/cumsum) for the special cases that reduce
to them, and invariants the paper states.  Pin numbers follow SURVEY.md section 8(c).
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest
import torch

from paper_2202_12817_b200 import inputs

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")

NO_FUND_SELECT, NO_DRIFT, ALL_HARMONICS, ALL_ORDERS = 1, 2, 4, 8


def _rows(path):
    out = []
    with open(path) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                out.append([int(t) for t in line.split()])
    return out


def _lin_stats(H, mu1=1.0, sig1=1.0):
    """mu_h = h mu1, sigma_h = sqrt(h) sig1 (statistics of a sum of h iid terms)."""
    h = np.arange(1, H + 1, dtype=np.float64)
    return (h * mu1).astype(np.float32), (np.sqrt(h) * sig1).astype(np.float32)


# ------------------------------------------------------------------------------------------
# P4  the paper's worked index example and order set
# ------------------------------------------------------------------------------------------
def test_p4_paper_index_example(oracle_mod):
    for h, Hp, n, want in _rows(os.path.join(GOLDEN, "presto_index_example.txt")):
        assert oracle_mod.presto_index(h, Hp, n) == want


def test_p4_paper_order_set(oracle_mod):
    (want,) = _rows(os.path.join(GOLDEN, "presto_orders_H32.txt"))
    assert oracle_mod.presto_orders(32) == want
    assert oracle_mod.presto_orders(32, ALL_HARMONICS) == want            # PRESTO_all keeps the order set
    assert oracle_mod.presto_orders(32, ALL_HARMONICS | ALL_ORDERS) == list(range(1, 33))  # PRESTO+
    assert oracle_mod.presto_orders(12) == [1, 2, 4, 8]


def test_p4_presto_harmonic_set_decoded_from_sums(oracle_mod):
    """Alg. 1 adds the fundamental and the EVEN harmonics only:
    HARM(8) = {1,2,4,6,8}.  x[b] = 8^b makes every sum a base-8 numeral whose digits are the
    multiplicities of the bins that were added; expected bins come from exact Fractions."""
    N = 17
    x = np.array([8.0 ** b for b in range(N)], dtype=np.float32)
    H = 8
    mu = np.zeros(H, np.float32)
    sg = np.ones(H, np.float32)
    for flags, harm in ((0, lambda Hp: [1] + list(range(2, Hp + 1, 2))),
                        (ALL_HARMONICS, lambda Hp: list(range(1, Hp + 1)))):
        for n in range(N):
            r = oracle_mod.presto_bins(x, H, mu, sg, [0], [n], flags)
            for Hp in (1, 2, 4, 8):
                digits = [0] * N
                for h in harm(Hp):
                    digits[math.floor(Fraction(h * n, Hp) + Fraction(1, 2))] += 1
                want = sum(c * 8 ** b for b, c in enumerate(digits))
                assert r["snr_h"][0, Hp - 1] == float(want), (flags, n, Hp)
            for Hp in (3, 5, 6, 7):
                assert math.isnan(r["snr_h"][0, Hp - 1])


# ------------------------------------------------------------------------------------------
# P1  H = 1 is the identity up to normalisation
# ------------------------------------------------------------------------------------------
def test_p1_identity(oracle_mod):
    rng = np.random.default_rng(11)
    x = rng.exponential(1.0, (3, 257)).astype(np.float32)
    mu = np.array([0.75], np.float32)
    sg = np.array([1.5], np.float32)
    ident = (x.astype(np.float64) - 0.75) / 1.5
    s, b = oracle_mod.presto(x, 1, mu, sg)
    assert np.array_equal(s, ident) and np.all(b == 1)
    s, b, p = oracle_mod.greedy(x, 1, mu, sg, NO_FUND_SELECT)
    assert np.array_equal(s, ident) and np.all(b == 1) and np.all(p == 0)
    # default greedy: the larger of x[n], x[n+1]; x[N] is absent (R4)
    s, b, p = oracle_mod.greedy(x, 1, mu, sg)
    nxt = np.concatenate([x[:, 1:], np.full((3, 1), -np.inf, np.float32)], axis=1)
    assert np.array_equal(s, (np.maximum(x, nxt).astype(np.float64) - 0.75) / 1.5)
    assert np.array_equal(p, (nxt > x).astype(np.uint32))
    assert np.all(b == 1)


# ------------------------------------------------------------------------------------------
# P2  constant spectrum: closed form, sqrt(N_harm) gain
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("c", [3.0, 1.0, 0.25])
def test_p2_constant_spectrum(oracle_mod, c):
    N, H = 200, 8
    x = np.full((1, N), c, np.float32)
    mu, sg = _lin_stats(H, 1.0, 0.5)
    s, b, p = oracle_mod.greedy(x, H, mu, sg)
    assert np.all(p == 0)                                   # ties stay: never shifts
    n = np.arange(N)
    k = np.where(n == 0, H, np.minimum(H, (N - 1) // np.maximum(n, 1)))   # evaluated orders
    if c > 1.0:
        assert np.array_equal(b[0], k)
        want = np.sqrt(k.astype(np.float32).astype(np.float64)) * (c - 1.0) / 0.5
        assert np.allclose(s[0], want, rtol=1e-6)           # sigma_h is an fp32 input
    elif c == 1.0:
        assert np.all(s[0] == 0.0) and np.all(b == 1)       # all orders tie at 0: the first wins
    else:
        assert np.all(b == 1) and np.allclose(s[0], (c - 1.0) / 0.5)
    # PRESTO_all: S = H' c exactly; PRESTO (Alg. 1): 1 or 1 + H'/2 terms
    s, b = oracle_mod.presto(x, H, mu, sg, ALL_HARMONICS)
    if c > 1.0:
        assert np.all(b == 8) and np.allclose(s, math.sqrt(8) * (c - 1.0) / 0.5, rtol=1e-6)
    r = oracle_mod.presto_bins(x, H, np.zeros(H, np.float32), np.ones(H, np.float32), [0] * 3, [5, 77, 199])
    for Hp, terms in ((1, 1), (2, 2), (4, 3), (8, 5)):
        assert np.all(r["snr_h"][:, Hp - 1] == terms * c)


# ------------------------------------------------------------------------------------------
# P3  delta train
# ------------------------------------------------------------------------------------------
def test_p3_delta_train_greedy(oracle_mod):
    N, f0, K, A, H = 4096, 37, 8, 10.0, 16
    x = inputs.delta_train(N, f0, K, A).numpy()[None, :]
    mu, sg = _lin_stats(H)
    s, b, p = oracle_mod.greedy(x, H, mu, sg, NO_FUND_SELECT)
    assert int(np.argmax(s[0])) == f0 and np.count_nonzero(s[0] == s[0].max()) == 1
    assert b[0, f0] == K and p[0, f0] == 0
    assert s[0, f0] == pytest.approx((K * A - K) / math.sqrt(K), rel=1e-6)      # (A-1) sqrt(K)
    # with fundamental selection bin f0-1 follows the train too (drift grows at every order)
    s, b, p = oracle_mod.greedy(x, H, mu, sg)
    top = np.flatnonzero(s[0] == s[0].max())
    assert set(top.tolist()) == {f0 - 1, f0}
    assert p[0, f0] == 0 and p[0, f0 - 1] == (1 << K) - 1 and b[0, f0 - 1] == K


def test_p3_delta_train_presto(oracle_mod):
    N, f0, K, A, H = 4096, 37, 8, 10.0, 16
    x = inputs.delta_train(N, f0, K, A).numpy()[None, :]
    mu, sg = _lin_stats(H)                                  # "h, sqrt(h)" statistics
    for flags in (ALL_HARMONICS, ALL_HARMONICS | ALL_ORDERS):
        s, b = oracle_mod.presto(x, H, mu, sg, flags)
        assert int(np.argmax(s[0])) == K * f0               # R10: indexed by the TOP harmonic
        assert b[0, K * f0] == K
        assert s[0, K * f0] == pytest.approx((A - 1.0) * math.sqrt(K), rel=1e-6)
    # Alg. 1 proper (even harmonics, term-count statistics): at n = K f0 the even harmonics of
    # f0/2 are all K harmonics of f0, so H' = 2K wins with (A K - (1+K)) / sqrt(1+K).
    mu_t, sg_t = (t.numpy() for t in inputs.exp1_stats("presto", H))
    s, b = oracle_mod.presto(x, H, mu_t, sg_t)
    assert b[0, K * f0] == 2 * K
    assert s[0, K * f0] == pytest.approx((A * K - (1 + K)) / math.sqrt(1 + K), rel=1e-6)
    assert s[0, K * f0] == pytest.approx(23.6666666, rel=1e-6)


# ------------------------------------------------------------------------------------------
# P5  brute force on tiny spectra
# ------------------------------------------------------------------------------------------
def _tiny(seed, N):
    # many exact ties on purpose (values 0..5) so the tie rules are exercised
    return np.random.default_rng(seed).integers(0, 6, N).astype(np.float32)


@pytest.mark.parametrize("flags", [0, ALL_HARMONICS, ALL_HARMONICS | ALL_ORDERS])
def test_p5_presto_bruteforce_exact_rational(oracle_mod, flags):
    """eq. 4 with python Fractions for the index and exact integer sums (N <= 64, all H <= 8)."""
    for seed, N in ((1, 7), (2, 33), (3, 64)):
        x = _tiny(seed, N)
        for H in range(1, 9):
            mu = (0.5 * np.arange(1, H + 1)).astype(np.float32)     # exact in fp32
            sg = (2.0 ** (np.arange(H) % 3)).astype(np.float32)     # powers of two
            s, b = oracle_mod.presto(x, H, mu, sg, flags)
            for n in range(N):
                best, bh = -math.inf, 0
                for Hp in range(1, H + 1):
                    if not (flags & ALL_ORDERS) and (Hp & (Hp - 1)):
                        continue
                    hs = range(1, Hp + 1) if flags & ALL_HARMONICS else [1] + list(range(2, Hp + 1, 2))
                    tot = sum(Fraction(float(x[math.floor(Fraction(h * n, Hp) + Fraction(1, 2))])) for h in hs)
                    snr = (tot - Fraction(float(mu[Hp - 1]))) / Fraction(float(sg[Hp - 1]))
                    if snr > best:
                        best, bh = snr, Hp
                assert s[0, n] == float(best) and b[0, n] == bh, (seed, H, n)


def _path_tree(y, n, H, flags):
    """All monotone drift paths of fundamental n through the values y (Fig. 4).
    Returns (locally greedy paths [(bits, partial sums)], best partial sum over all paths per order)."""
    N = len(y)
    greedy_paths, best_sum_at = [], [-math.inf] * H
    for bits in range(1 << H):
        d, tot, in_tree, locally_greedy, sums = 0, 0.0, True, True, []
        for h in range(1, H + 1):
            m = h * n + d
            step = (bits >> (h - 1)) & 1
            if m > N - 1:                       # band edge: the path ends here (R4)
                in_tree = in_tree and (bits >> (h - 1)) == 0   # canonical: no later steps
                break
            second = float(y[m + 1]) if m + 1 <= N - 1 else None
            if h == 1 and (flags & NO_FUND_SELECT):
                second = None                   # the tree has a single child here (R7)
            if step and second is None:
                in_tree = False
                break
            want = 1 if (second is not None and second > float(y[m])) else 0
            locally_greedy = locally_greedy and (step == want)
            tot += second if step else float(y[m])
            d += step
            sums.append(tot)
        if not in_tree:
            continue
        for i, t in enumerate(sums):
            best_sum_at[i] = max(best_sum_at[i], t)
        if locally_greedy:
            greedy_paths.append((bits, sums))
    return greedy_paths, best_sum_at


def _check_against_tree(res, y, N, H, flags, mu, sg, tag):
    for n in range(N):
        greedy_paths, best_sum_at = _path_tree(y, n, H, flags)
        assert len(greedy_paths) == 1, (tag, n)
        bits, sums = greedy_paths[0]
        assert res["path"][n] == bits, (tag, n)
        got = res["snr_h"][n] * sg + mu           # partial sums back from the per-order SNRs
        for i, t in enumerate(sums):
            assert got[i] == t and t <= best_sum_at[i]
        assert np.all(np.isnan(res["snr_h"][n][len(sums):]))
        snrs = [(t - mu[i]) / sg[i] for i, t in enumerate(sums)]
        assert res["snr"][n] == max(snrs)
        assert res["best_h"][n] == 1 + snrs.index(max(snrs))      # first maximum (R6)


@pytest.mark.parametrize("flags", [0, NO_FUND_SELECT])
def test_p5_greedy_bruteforce_path_tree(oracle_mod, flags):
    """Enumerate all 2^H monotone drift paths of the tree (Fig. 4).  Exactly one
    of them is 'locally greedy' (each step takes the larger child, ties stay); the oracle must
    return that one, and its partial sums can never beat the best path."""
    for seed, N, H in ((5, 40, 5), (6, 64, 6), (7, 23, 4)):
        x = _tiny(seed, N)
        mu = np.arange(1, H + 1).astype(np.float32)
        sg = np.ones(H, np.float32)
        res = oracle_mod.greedy_bins(x, H, mu, sg, [0] * N, list(range(N)), flags)
        _check_against_tree(res, x, N, H, flags, mu, sg, seed)


# ------------------------------------------------------------------------------------------
# R13 / NEXT-2  the whitening multiplier: every x[b] is replaced by the fp32 product x[b] * inv_baseline[b]
# ("whitening" happens before the sum; PAPER.md:264 same pre-processing for all algorithms)
# ------------------------------------------------------------------------------------------
def test_r13_inv_baseline_power_of_two_equals_premultiplied(oracle_mod):
    """With power-of-two multipliers the product is exact in fp32, so running on (x, ib) must equal
    running on the pre-multiplied spectrum bit for bit -- and differ from ignoring ib."""
    rng = np.random.default_rng(41)
    S, N, H = 3, 1500, 8
    x = rng.exponential(1.0, (S, N)).astype(np.float32)
    ib = (2.0 ** rng.integers(-3, 4, (S, N))).astype(np.float32)
    y = x * ib                                                # exact
    assert np.array_equal(y.astype(np.float64), x.astype(np.float64) * ib.astype(np.float64))
    mu, sg = (t.numpy() for t in inputs.exp1_stats("greedy", H))
    bins = np.arange(0, N, 3)
    rows = bins % S
    for flags in (0, NO_FUND_SELECT, NO_DRIFT):
        a = oracle_mod.greedy(x, H, mu, sg, flags, inv_baseline=ib)
        b = oracle_mod.greedy(y, H, mu, sg, flags)
        c = oracle_mod.greedy(x, H, mu, sg, flags)
        for u, v in zip(a, b):
            assert np.array_equal(u, v)
        assert not np.array_equal(a[0], c[0])                 # the multiplier is not ignored
        ra = oracle_mod.greedy_bins(x, H, mu, sg, rows, bins, flags, inv_baseline=ib)
        rb = oracle_mod.greedy_bins(y, H, mu, sg, rows, bins, flags)
        for k in ("snr", "best_h", "path", "bin_h"):
            assert np.array_equal(ra[k], rb[k]), k
        assert np.array_equal(ra["snr_h"], rb["snr_h"], equal_nan=True)
        assert np.array_equal(ra["snr"], a[0][rows, bins])
    for flags in (0, ALL_HARMONICS, ALL_HARMONICS | ALL_ORDERS):
        mu, sg = (t.numpy() for t in inputs.exp1_stats("presto" if flags == 0 else "presto_plus", H))
        a = oracle_mod.presto(x, H, mu, sg, flags, inv_baseline=ib)
        b = oracle_mod.presto(y, H, mu, sg, flags)
        c = oracle_mod.presto(x, H, mu, sg, flags)
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
        assert not np.array_equal(a[0], c[0])
        ra = oracle_mod.presto_bins(x, H, mu, sg, rows, bins, flags, inv_baseline=ib)
        rb = oracle_mod.presto_bins(y, H, mu, sg, rows, bins, flags)
        assert np.array_equal(ra["snr"], rb["snr"]) and np.array_equal(ra["best_h"], rb["best_h"])
        assert np.array_equal(ra["snr_h"], rb["snr_h"], equal_nan=True)


@pytest.mark.parametrize("flags", [0, NO_FUND_SELECT])
def test_r13_inv_baseline_flips_comparisons_path_tree(oracle_mod, flags):
    """Small-integer x and ib (products exact): the multiplier must change WHICH child is larger; the
    oracle's path is the unique locally greedy path of the tree over the products, which differs from
    the tree over x alone."""
    for seed, N, H in ((8, 40, 5), (9, 57, 6)):
        rng = np.random.default_rng(seed)
        x = rng.integers(1, 6, N).astype(np.float32)
        ib = rng.integers(1, 5, N).astype(np.float32)
        y = [float(a) * float(b) for a, b in zip(x, ib)]       # exact small integers
        mu = np.arange(1, H + 1).astype(np.float32)
        sg = np.ones(H, np.float32)
        res = oracle_mod.greedy_bins(x, H, mu, sg, [0] * N, list(range(N)), flags, inv_baseline=ib)
        _check_against_tree(res, y, N, H, flags, mu, sg, seed)
        plain = oracle_mod.greedy_bins(x, H, mu, sg, [0] * N, list(range(N)), flags)
        assert np.count_nonzero(plain["path"] != res["path"]) >= 8          # comparisons really flipped


def test_r13_inv_baseline_product_is_one_fp32_multiply(oracle_mod):
    """The product that decides the comparison is rounded to fp32 (reading R13): two fp64-distinct
    products that round to the same fp32 value tie, and a tie stays."""
    a, ia = np.float32(1.0 + 2.0 ** -23), np.float32(3.0)    # exact product 3 + 1.5 ulp: rounds (to even) to 3 + 2 ulp
    b, ib_ = np.float32(3.0 + 2.0 ** -21), np.float32(1.0)   # 3 + 2 ulp
    pa64, pb64 = float(a) * float(ia), float(b) * float(ib_)
    assert pb64 > pa64 and np.float32(a * ia) == np.float32(b * ib_)       # fp64: second larger; fp32: tie
    x = np.array([a, b, 0.0, 0.0], np.float32)
    ib = np.array([ia, ib_, 1.0, 1.0], np.float32)
    r = oracle_mod.greedy_bins(x, 1, [0.0], [1.0], [0], [0], inv_baseline=ib)
    assert r["path"][0] == 0 and r["bin_h"][0, 0] == 0
    assert r["snr"][0] == float(np.float32(a * ia))


# ------------------------------------------------------------------------------------------
# Special cases that reduce to library routines
# ------------------------------------------------------------------------------------------
def test_simple_hs_equals_numpy_gather_cumsum(oracle_mod):
    """NO_DRIFT greedy is eq. 3, X[n] = sum_h x[h n]: numpy fancy indexing + cumsum."""
    rng = np.random.default_rng(21)
    N, H = 5000, 16
    x = rng.exponential(1.0, N).astype(np.float32)
    mu, sg = _lin_stats(H)
    bins = np.arange(1, (N - 1) // H + 1)                      # all H orders inside the band
    res = oracle_mod.greedy_bins(x, H, mu, sg, np.zeros_like(bins), bins, NO_DRIFT)
    idx = bins[:, None] * np.arange(1, H + 1)[None, :]
    S = np.cumsum(x[idx].astype(np.float64), axis=1)
    snr_h = (S - mu.astype(np.float64)) / sg.astype(np.float64)
    assert np.allclose(res["snr_h"], snr_h, rtol=1e-13, atol=1e-13)
    assert np.array_equal(res["best_h"], 1 + np.argmax(snr_h, axis=1))
    assert np.all(res["path"] == 0)
    assert np.array_equal(res["bin_h"], idx)


def test_presto_all_on_exact_multiples_equals_simple_hs(oracle_mod):
    """When H' divides n, h n / H' is an integer, so PRESTO_all at top bin n = H' f adds exactly
    x[h f], h = 1..H' -- the simple harmonic sum of fundamental f (eq. 3 vs eq. 4)."""
    rng = np.random.default_rng(22)
    N, H = 4096, 8
    x = rng.exponential(1.0, N).astype(np.float32)
    mu, sg = _lin_stats(H)
    f = np.arange(1, (N - 1) // H + 1)
    simple = oracle_mod.greedy_bins(x, H, mu, sg, np.zeros_like(f), f, NO_DRIFT)
    for Hp in (1, 2, 4, 8):
        pa = oracle_mod.presto_bins(x, H, mu, sg, np.zeros_like(f), f * Hp, ALL_HARMONICS)
        assert np.allclose(pa["snr_h"][:, Hp - 1], simple["snr_h"][:, Hp - 1], rtol=1e-13, atol=1e-13)


# ------------------------------------------------------------------------------------------
# P6  invariants
# ------------------------------------------------------------------------------------------
def test_p6_greedy_invariants(oracle_mod):
    w = inputs.workload("cfg1")
    x = inputs.generate_row(w, 0).numpy()
    N, H = x.size, 8
    mu, sg = (t.numpy() for t in inputs.exp1_stats("greedy", H))
    bins = np.arange(0, N, 7)
    for flags in (0, NO_FUND_SELECT):
        r = oracle_mod.greedy_bins(x, H, mu, sg, np.zeros_like(bins), bins, flags)
        for h in range(1, H + 1):
            d_h = np.array([bin(int(p) & ((1 << h) - 1)).count("1") for p in r["path"]])
            assert np.all(d_h <= (h if flags == 0 else h - 1))
            ev = r["bin_h"][:, h - 1] >= 0
            assert np.array_equal(r["bin_h"][ev, h - 1], (h * bins + d_h)[ev])  # eq. 5
            assert np.all(r["bin_h"][ev, h - 1] <= N - 1)
            # R4: evaluated iff h n + d_{h-1} <= N-1
            d_prev = np.array([bin(int(p) & ((1 << (h - 1)) - 1)).count("1") for p in r["path"]])
            assert np.array_equal(ev, h * bins + d_prev <= N - 1)
        assert np.all((r["best_h"] >= 1) & (r["best_h"] <= H))
        s1 = r["snr_h"][:, 0] * sg[0] + mu[0]
        assert np.all(s1 >= x[bins] - 1e-6)                                     # S_1 >= x[n]


def test_p6_presto_depends_only_on_bins_up_to_n(oracle_mod):
    rng = np.random.default_rng(31)
    N, H = 3000, 16
    x = rng.exponential(1.0, N).astype(np.float32)
    mu, sg = (t.numpy() for t in inputs.exp1_stats("presto", H))
    s0, b0 = oracle_mod.presto(x, H, mu, sg)
    cut = 1777
    y = x.copy()
    y[cut + 1:] = 1e6
    s1, b1 = oracle_mod.presto(y, H, mu, sg)
    assert np.array_equal(s0[0, :cut + 1], s1[0, :cut + 1]) and np.array_equal(b0[0, :cut + 1], b1[0, :cut + 1])


def test_p6_power_of_two_scaling_and_batch_independence(oracle_mod):
    rng = np.random.default_rng(32)
    S, N, H = 4, 2048, 8
    x = rng.exponential(1.0, (S, N)).astype(np.float32)
    mu, sg = (t.numpy() for t in inputs.exp1_stats("greedy", H))
    s0, b0, p0 = oracle_mod.greedy(x, H, mu, sg)
    s1, b1, p1 = oracle_mod.greedy(x * 4, H, mu * 4, sg * 4)
    assert np.array_equal(s0, s1) and np.array_equal(b0, b1) and np.array_equal(p0, p1)
    for r in range(S):
        sr, br, pr = oracle_mod.greedy(x[r], H, mu, sg, n_threads=1)
        assert np.array_equal(sr[0], s0[r]) and np.array_equal(br[0], b0[r]) and np.array_equal(pr[0], p0[r])
    mu, sg = (t.numpy() for t in inputs.exp1_stats("presto", H))
    q0, c0 = oracle_mod.presto(x, H, mu, sg)
    q1, c1 = oracle_mod.presto(x * 0.5, H, mu * 0.5, sg * 0.5)
    assert np.array_equal(q0, q1) and np.array_equal(c0, c1)
    # n_fund limits the outputs, values unchanged
    q2, c2 = oracle_mod.presto(x, H, mu, sg, n_fund=100)
    assert q2.shape == (S, 100) and np.array_equal(q2, q0[:, :100])


def test_r4_band_edge(oracle_mod):
    """Order h is evaluated iff h n + d <= N-1; the absent bin N never wins."""
    N, H = 101, 4
    x = np.zeros(N, np.float32)
    x[100] = 5.0
    mu = np.zeros(H, np.float32)
    sg = np.ones(H, np.float32)
    r = oracle_mod.greedy_bins(x, H, mu, sg, [0] * 4, [25, 50, 100, 99], NO_FUND_SELECT)
    # n = 25: orders 1..4 land on 25, 50, 75, 100 (m = 100 = N-1 evaluated, second bin absent)
    assert np.array_equal(r["bin_h"][0], [25, 50, 75, 100]) and r["snr"][0] == 5.0 and r["best_h"][0] == 4
    # n = 50: order 2 at m = 100, order 3 would be 150 > N-1: skipped
    assert np.array_equal(r["bin_h"][1], [50, 100, -1, -1]) and r["best_h"][1] == 2
    # n = 100: only the fundamental; with selection on, x[N] is absent and cannot win
    assert np.array_equal(r["bin_h"][2], [100, -1, -1, -1])
    r2 = oracle_mod.greedy_bins(x, H, mu, sg, [0, 0], [100, 99])
    assert r2["path"][0] == 0 and r2["snr"][0] == 5.0
    # n = 99 with selection: picks bin 100 (drift 1); order 2 would start at 199 > N-1
    assert r2["path"][1] == 1 and np.array_equal(r2["bin_h"][1], [100, -1, -1, -1])


# ------------------------------------------------------------------------------------------
# P8  statistics of the partial sums on Exp(1) noise match the closed forms
# ------------------------------------------------------------------------------------------
def test_p8_noise_statistics(oracle_mod):
    H, N = 16, 1 << 20
    w = inputs.Workload("noise", 1, N, H, seed=77)
    x = inputs.generate_row(w, 0).numpy()
    assert abs(x.mean() - 1.0) < 5.0 / math.sqrt(N) and abs(x.var() - 1.0) < 0.02   # Exp(1)
    bins = np.arange(64, N // (H + 1), 3)
    cnt = bins.size
    zeros = np.zeros_like(bins)

    def check(res, variant, mu, sg, orders):
        for h in orders:
            S = res["snr_h"][:, h - 1] * sg[h - 1] + mu[h - 1]
            var = float(sg[h - 1]) ** 2
            assert abs(S.mean() - mu[h - 1]) < 6.0 * math.sqrt(var / cnt), (variant, h)
            assert abs(S.var() / var - 1.0) < 0.06, (variant, h)

    mu, sg = (t.numpy().astype(np.float64) for t in inputs.exp1_stats("greedy", H))
    check(oracle_mod.greedy_bins(x, H, mu, sg, zeros, bins), "greedy", mu, sg, range(1, H + 1))
    mu, sg = (t.numpy().astype(np.float64) for t in inputs.exp1_stats("greedy", H, fund_select=False))
    check(oracle_mod.greedy_bins(x, H, mu, sg, zeros, bins, NO_FUND_SELECT), "greedy_nofs", mu, sg, range(1, H + 1))
    mu, sg = (t.numpy().astype(np.float64) for t in inputs.exp1_stats("simple", H))
    check(oracle_mod.greedy_bins(x, H, mu, sg, zeros, bins, NO_DRIFT), "simple", mu, sg, range(1, H + 1))
    top = bins * H       # PRESTO outputs are indexed by the top bin; keep the bins distinct
    mu, sg = (t.numpy().astype(np.float64) for t in inputs.exp1_stats("presto", H))
    check(oracle_mod.presto_bins(x, H, mu, sg, zeros, top), "presto", mu, sg, (1, 2, 4, 8, 16))
    mu, sg = (t.numpy().astype(np.float64) for t in inputs.exp1_stats("presto_plus", H))
    check(oracle_mod.presto_bins(x, H, mu, sg, zeros, top, ALL_HARMONICS | ALL_ORDERS), "presto_plus", mu, sg, range(1, H + 1))


# ------------------------------------------------------------------------------------------
# P9 (soft, paper-stated): on a noiseless pulse train greedy recovers what PRESTO+ recovers
# and the simple sum loses; scalloping keeps sinc(1/2) = 0.637
# of the amplitude for a half-bin offset ("up to 36% loss").
# ------------------------------------------------------------------------------------------
def test_p9_noiseless_pulse_train_soft(oracle_mod):
    N, H = 1 << 14, 16
    p = inputs.Pulsar(0, 200.5, 0.04, 8.0, 0.3)
    re = torch.zeros(N, dtype=torch.float64)
    im = torch.zeros(N, dtype=torch.float64)
    inputs._inject(re, im, p)
    x = (re * re + im * im).to(torch.float32).numpy()
    assert x[200] / 64.0 == pytest.approx((2.0 / math.pi) ** 2, rel=1e-6)     # |sinc(1/2)|^2 of the power
    mu, sg = _lin_stats(H, 0.0, 1.0)
    g, _, _ = oracle_mod.greedy(x, H, mu, sg)
    s, _, _ = oracle_mod.greedy(x, H, mu, sg, NO_DRIFT)
    pp, _ = oracle_mod.presto(x, H, mu, sg, ALL_HARMONICS | ALL_ORDERS)
    assert g.max() >= 0.97 * pp.max()
    # at the fundamental itself the drift-free sum walks off the peak after a few orders
    assert s[0, 199:202].max() < 0.9 * g[0, 199:202].max()


def test_argument_validation(oracle_mod):
    x = np.ones(16, np.float32)
    with pytest.raises(ValueError):
        oracle_mod.greedy(x, 2, [1, 2], [1, 0])            # sigma must be > 0
    with pytest.raises(ValueError):
        oracle_mod.presto(x, 2, [1, 2], [1, 1], ALL_ORDERS)  # ALL_ORDERS needs ALL_HARMONICS
    with pytest.raises(ValueError):
        oracle_mod.greedy(x, 33, np.ones(33), np.ones(33))


def test_candidates_definition_brute_force():
    """R11: the candidate list is the plain threshold definition; pinned by a Python loop on a tiny array
    (ties at the threshold count, NaN does not)."""
    import oracle
    snr = np.array([[1.0, 10.0, np.nan, 12.5], [9.999, 10.0001, -3.0, 1e9]], np.float32)
    bh = np.array([[1, 2, 3, 4], [5, 6, 7, 8]], np.int32)
    want = [(s, n, int(bh[s, n])) for s in range(2) for n in range(4) if float(snr[s, n]) >= 10.0]
    got, vals = oracle.candidates(snr, bh, 10.0)
    assert [tuple(r) for r in got.tolist()] == want == [(0, 1, 2), (0, 3, 4), (1, 1, 6), (1, 3, 8)]
    assert vals.tolist() == [float(snr[s, n]) for s, n, _ in want]


# ------------------------------------------------------------------------------------------
# R14: the reading of GetMeanStdev() -- oracle.estimate_stats
# ------------------------------------------------------------------------------------------
def _simple_sums_numpy(x, H, n_lo, n_hi):
    """S_h(n) = sum_{k<=h} x[k n] (eq. 3) by gather + cumsum; NaN where h n > N - 1.  Independent of the oracle."""
    N = x.shape[0]
    n = np.arange(n_lo, n_hi)
    out = np.full((n.size, H), np.nan)
    run = np.zeros(n.size)
    alive = np.ones(n.size, bool)
    for h in range(1, H + 1):
        alive &= h * n <= N - 1
        run[alive] += x[(h * n)[alive]].astype(np.float64)
        out[alive, h - 1] = run[alive]
    return out


def test_r14_stats_simple_variant_equals_numpy_moments(oracle_mod):
    """Exact-integer spectra, simple harmonic sum: mean / population std / count of S_h over a range that crosses the
    band edges N/h, against numpy moments of numpy gathers (nothing of the oracle is re-used)."""
    H, N = 16, 6000
    x = inputs.integer_spectra(71, 3, N, 50).numpy()
    n_lo, n_hi = 5, 2500
    mu, sg, cnt = oracle_mod.estimate_stats(x, H, NO_DRIFT | NO_FUND_SELECT, True, n_lo, n_hi)
    for s in range(3):
        sums = _simple_sums_numpy(x[s], H, n_lo, n_hi)
        for h in range(H):
            v = sums[:, h][~np.isnan(sums[:, h])]
            assert cnt[s, h] == v.size == np.count_nonzero((h + 1) * np.arange(n_lo, n_hi) <= N - 1)
            assert mu[s, h] == np.float32(v.mean())
            assert abs(float(sg[s, h]) - v.std()) <= 1e-6 * v.std()


def test_r14_stats_clipping_rounds(oracle_mod):
    """Outlier rejection: a few enormous bins; each round keeps the sums inside mean -/+ clip std of the round before
    (fp32-rounded limits).  Re-done in numpy for the simple variant."""
    H, N, clip = 8, 40000, 2.5
    x = inputs.integer_spectra(72, 1, N, 20).numpy()
    x[0, ::997] += 5000.0
    n_lo, n_hi = 100, 4000
    sums = _simple_sums_numpy(x[0], H, n_lo, n_hi)
    for n_clip in (0, 1, 3):
        mu, sg, cnt = oracle_mod.estimate_stats(x, H, NO_DRIFT | NO_FUND_SELECT, True, n_lo, n_hi, clip=clip, n_clip=n_clip)
        for h in range(H):
            v = sums[:, h]
            keep = np.ones(v.size, bool)
            for _ in range(n_clip + 1):
                m, sd = v[keep].mean(), v[keep].std()
                stats = (m, sd, int(keep.sum()))
                lo, hi = np.float32(m - clip * sd), np.float32(m + clip * sd)
                keep = (v >= lo) & (v <= hi)
            assert cnt[0, h] == stats[2]
            assert mu[0, h] == np.float32(stats[0]) and abs(float(sg[0, h]) - stats[1]) <= 1e-6 * stats[1]
        if n_clip:
            assert cnt[0, 0] < n_hi - n_lo and mu[0, 0] < 15.0          # the outliers are gone: mean of U{0..20} = 10


def test_r14_stats_closed_forms_and_degenerate_cases(oracle_mod):
    """Exp(1) noise: greedy mean 1.5 h, variance 1.25 h; PRESTO (Alg. 1) t terms; PRESTO_all H' terms (SURVEY.md 8(c)
    statistics paragraph) within sampling error.  Constant spectrum: mean h c, sigma returned as 1.  Orders outside
    the PRESTO order set: (0, 1) with no samples."""
    H = 16
    x = inputs.generate(inputs.Workload("n", 2, 1 << 19, H, seed=91)).numpy()
    n_lo, n_hi = 2000, 30000
    k = n_hi - n_lo
    mu, sg, cnt = oracle_mod.estimate_stats(x, H, 0, True, n_lo, n_hi)
    h = np.arange(1, H + 1)
    assert np.all(cnt == k)
    # neighbouring n share bins, so the sums are correlated: bounds in relative terms, not in iid standard errors
    assert np.all(np.abs(mu / (1.5 * h) - 1.0) <= 0.02)
    assert np.all(np.abs(sg ** 2 / (1.25 * h) - 1.0) <= 0.08)
    mu, sg, cnt = oracle_mod.estimate_stats(x, H, 0, False, n_lo, n_hi)
    for Hp in range(1, H + 1):
        if Hp & (Hp - 1):
            assert np.all(cnt[:, Hp - 1] == 0) and np.all(mu[:, Hp - 1] == 0.0) and np.all(sg[:, Hp - 1] == 1.0)
        else:
            t = 1.0 if Hp == 1 else 1.0 + Hp // 2
            assert np.all(np.abs(mu[:, Hp - 1] / t - 1.0) <= 0.03)
            assert np.all(np.abs(sg[:, Hp - 1] ** 2 / t - 1.0) <= 0.12)
    mu, sg, cnt = oracle_mod.estimate_stats(x, H, ALL_HARMONICS, False, n_lo, n_hi)
    for Hp in (1, 2, 4, 8, 16):
        assert np.all(np.abs(mu[:, Hp - 1] / Hp - 1.0) <= 0.03)
    c = np.full((1, 5000), 3.0, np.float32)
    mu, sg, cnt = oracle_mod.estimate_stats(c, 8, 0, True, 10, 500)
    assert np.array_equal(mu[0], 3.0 * np.arange(1, 9)) and np.all(sg == 1.0)


def test_r14_stats_apply_the_whitening_multiplier(oracle_mod):
    """whitening precedes the statistics.  With power-of-two multipliers on an exact-integer spectrum
    the product x * ib is exact, so estimate_stats(x, inv_baseline=ib) must equal estimate_stats(x * ib) bit for bit
    (greedy, simple and PRESTO forms, with rejection rounds), must differ from estimate_stats(x), and -- for the simple
    variant -- must equal numpy moments of numpy gathers of the product (nothing of the oracle re-used)."""
    H, S, N = 12, 2, 9000
    x = inputs.integer_spectra(73, S, N, 40).numpy()
    x[:, ::613] += 2000.0
    rng = np.random.default_rng(5)
    ib = (2.0 ** rng.integers(-1, 3, size=(S, N))).astype(np.float32)          # 0.5, 1, 2, 4
    prod = (x * ib).astype(np.float32)
    assert np.array_equal(prod.astype(np.float64), x.astype(np.float64) * ib.astype(np.float64))
    n_lo, n_hi = 7, 3000
    for greedy, flags in ((True, 0), (True, NO_DRIFT | NO_FUND_SELECT), (False, 0), (False, ALL_HARMONICS)):
        for n_clip in (0, 2):
            with_ib = oracle_mod.estimate_stats(x, H, flags, greedy, n_lo, n_hi, clip=2.5, n_clip=n_clip, inv_baseline=ib)
            of_prod = oracle_mod.estimate_stats(prod, H, flags, greedy, n_lo, n_hi, clip=2.5, n_clip=n_clip)
            plain = oracle_mod.estimate_stats(x, H, flags, greedy, n_lo, n_hi, clip=2.5, n_clip=n_clip)
            for a, b in zip(with_ib, of_prod):
                assert np.array_equal(a, b), (greedy, flags, n_clip)
            assert not np.array_equal(with_ib[0][:, 0], plain[0][:, 0]), (greedy, flags, n_clip)
    mu, sg, cnt = oracle_mod.estimate_stats(x, H, NO_DRIFT | NO_FUND_SELECT, True, n_lo, n_hi, inv_baseline=ib)
    for s in range(S):
        sums = _simple_sums_numpy(prod[s], H, n_lo, n_hi)
        for h in range(H):
            v = sums[:, h][~np.isnan(sums[:, h])]
            assert cnt[s, h] == v.size
            assert mu[s, h] == np.float32(v.mean()) and abs(float(sg[s, h]) - v.std()) <= 1e-6 * v.std()


def limits_spectrum():
    """Eight sums that sit exactly ON the rejection limits (reading R14: a round keeps lo <= S_h(n) <= hi).
    Order 1 of the simple sum is x[n] itself: six bins of 10, one of 6, one of 14 -> mean 10, E[x^2] = 104,
    variance 4, deviation 2 (all exact); with clip = 2 the limits are exactly 6 and 14, the two extreme samples."""
    x = np.zeros((1, 64), np.float32)
    x[0, 8:16] = [10, 6, 10, 10, 14, 10, 10, 10]
    return x, 8, 16, 2.0


def test_r14_rejection_limits_are_inclusive(oracle_mod):
    """DESIGN.md R14: round p keeps lo <= S <= hi.  Samples equal to a limit stay: the second round counts all eight
    sums and returns (10, 2); an exclusive comparison would drop the 6 and the 14 and return count 6, sigma 1
    (zero deviation).  Limits moved slightly inwards do reject them (the comparison is really made)."""
    x, n_lo, n_hi, clip = limits_spectrum()
    for n_clip in (0, 1, 2):
        mu, sg, cnt = oracle_mod.estimate_stats(x, 1, NO_DRIFT | NO_FUND_SELECT, True, n_lo, n_hi, clip=clip, n_clip=n_clip)
        assert cnt[0, 0] == 8 and mu[0, 0] == 10.0 and sg[0, 0] == 2.0, n_clip
    tight = 1.999                                                        # limits 6.002 and 13.998: just inside 6 and 14
    mu, sg, cnt = oracle_mod.estimate_stats(x, 1, NO_DRIFT | NO_FUND_SELECT, True, n_lo, n_hi, clip=tight, n_clip=1)
    assert cnt[0, 0] == 6 and mu[0, 0] == 10.0 and sg[0, 0] == 1.0


# ------------------------------------------------------------------------------------------
# R15 (NEXT-4): 2-D harmonic sums over an f-fdot plane -- oracle.greedy_2d / oracle.presto_2d
# ------------------------------------------------------------------------------------------
def _int_plane(seed, nz, N, max_val=50):
    return inputs.integer_spectra(seed, nz, N, max_val).numpy()


def test_r15_round_half_up_exact_rational(oracle_mod):
    from fractions import Fraction
    for b in (1, 2, 3, 4, 8, 16):
        for a in range(-70, 71):
            assert oracle_mod.round_half_up(a, b) == math.floor(Fraction(a, b) + Fraction(1, 2)), (a, b)


def test_r15_row_z0_reproduces_the_1d_sums(oracle_mod):
    """z = 0: k z = 0 for every k, so the 2-D simple sum and the 2-D PRESTO-like sums of that row are the 1-D sums of
    the row P[Z] (bit for bit: same terms in the same order)."""
    H, nz, N = 16, 7, 5000
    P = _int_plane(5, nz, N)
    Z = nz // 2
    mu, sg = (np.arange(1, H + 1, dtype=np.float32) * 3, np.sqrt(np.arange(1, H + 1)).astype(np.float32))
    s2, b2, p2 = oracle_mod.greedy_2d(P, H, mu, sg, NO_DRIFT)
    s1, b1, p1 = oracle_mod.greedy(P[Z], H, mu, sg, NO_DRIFT)
    assert np.array_equal(s2[Z], s1[0]) and np.array_equal(b2[Z], b1[0]) and not p2.any()
    for flags in (0, ALL_HARMONICS, ALL_HARMONICS | ALL_ORDERS):
        s2, b2 = oracle_mod.presto_2d(P, H, mu, sg, flags)
        s1, b1 = oracle_mod.presto(P[Z], H, mu, sg, flags)
        assert np.array_equal(s2[Z], s1[0]) and np.array_equal(b2[Z], b1[0])


def test_r15_brute_force_tiny_plane(oracle_mod):
    """Independent restatement in plain Python (exact rational rounding, argmax over an explicit candidate list)."""
    from fractions import Fraction
    H, nz, N = 6, 9, 40
    Z = nz // 2
    P = _int_plane(6, nz, N, 9).astype(np.float64)
    mu = np.array([2.0 * h for h in range(1, H + 1)], np.float32)
    sg = np.array([2.0 ** (h % 3) for h in range(1, H + 1)], np.float32)
    rnd = lambda a, b: math.floor(Fraction(a, b) + Fraction(1, 2))
    for flags in (0, NO_FUND_SELECT, NO_DRIFT):
        s, b, p = oracle_mod.greedy_2d(P.astype(np.float32), H, mu, sg, flags)
        for z in range(-Z, Z + 1):
            for r in range(N):
                dr = dz = 0; tot = 0.0; best = -math.inf; bh = 0; path = 0
                for h in range(1, H + 1):
                    m, w = h * r + dr, h * z + dz
                    if m > N - 1 or abs(w) > Z:
                        break
                    cand = [(P[w + Z, m], 0, 0)]
                    if not (flags & NO_DRIFT) and not (h == 1 and flags & NO_FUND_SELECT):
                        if m + 1 < N: cand.append((P[w + Z, m + 1], 1, 0))
                        if w + 1 <= Z: cand.append((P[w + 1 + Z, m], 0, 1))
                        if m + 1 < N and w + 1 <= Z: cand.append((P[w + 1 + Z, m + 1], 1, 1))
                    v, sr, sz = max(cand, key=lambda t: t[0])          # max() keeps the first of equal values
                    dr += sr; dz += sz; tot += v
                    path |= (sr << (h - 1)) | (sz << (16 + h - 1))
                    snr = (tot - float(mu[h - 1])) / float(sg[h - 1])
                    if snr > best: best, bh = snr, h
                assert (s[z + Z, r], b[z + Z, r], p[z + Z, r]) == (best, bh, path), (flags, z, r)
    for flags in (0, ALL_HARMONICS, ALL_HARMONICS | ALL_ORDERS):
        s, b = oracle_mod.presto_2d(P.astype(np.float32), H, mu, sg, flags)
        orders = [Hp for Hp in range(1, H + 1) if flags & ALL_ORDERS or Hp & (Hp - 1) == 0]
        for z in range(-Z, Z + 1):
            for r in range(N):
                best, bh = -math.inf, 0
                for Hp in orders:
                    ks = range(1, Hp + 1) if flags & ALL_HARMONICS else [1] + list(range(2, Hp + 1, 2))
                    tot = sum(P[rnd(k * z, Hp) + Z, rnd(k * r, Hp)] for k in ks)
                    snr = (tot - float(mu[Hp - 1])) / float(sg[Hp - 1])
                    if snr > best: best, bh = snr, Hp
                assert (s[z + Z, r], b[z + Z, r]) == (best, bh), (flags, z, r)


def test_r15_drifting_delta_train_and_truncation(oracle_mod):
    """A train of K deltas at (k r0, k z0) (BASELINE.json configs[4]: S_h(r,z) = sum P[k r, k z]): the simple 2-D sum
    peaks at (r0, z0) with best_h = K and snr (A-1) sqrt(K); at fractional (r0 + e, z0 + f) the bins are
    (floor(k (r0 + e)), floor(k (z0 + f))) and the 2-D greedy rule follows them; PRESTO_all 2-D peaks at the top
    harmonic (K r0, K z0).  Constant plane: best_h = number of evaluated orders = min(H, (N-1)//r, Z//|z|)."""
    H, nz, N, K, A = 16, 41, 3000, 8, 10.0
    Z = nz // 2
    mu = np.arange(1, H + 1, dtype=np.float32)
    sg = np.sqrt(np.arange(1, H + 1)).astype(np.float32)
    r0, z0 = 150, -2
    P = np.zeros((nz, N), np.float32)
    for k in range(1, K + 1):
        P[k * z0 + Z, k * r0] = A
    s, b, p = oracle_mod.greedy_2d(P, H, mu, sg, NO_DRIFT)
    assert (np.unravel_index(np.argmax(s), s.shape)) == (z0 + Z, r0) and b[z0 + Z, r0] == K
    assert abs(s[z0 + Z, r0] - (A - 1) * math.sqrt(K)) < 1e-5           # sigma is the fp32 sqrt
    s, b = oracle_mod.presto_2d(P, H, mu, sg, ALL_HARMONICS)
    assert (np.unravel_index(np.argmax(s), s.shape)) == (K * z0 + Z, K * r0) and b[K * z0 + Z, K * r0] == K
    e, f = 0.37, 0.55
    P = np.zeros((nz, N), np.float32)
    want = 0
    for k in range(1, K + 1):
        P[math.floor(k * (z0 + f)) + Z, math.floor(k * (r0 + e))] = A
    for k in range(1, K + 1):
        if math.floor(k * e) > math.floor((k - 1) * e): want |= 1 << (k - 1)
        if math.floor(k * f) > math.floor((k - 1) * f): want |= 1 << (16 + k - 1)
    s, b, p = oracle_mod.greedy_2d(P, H, mu, sg, 0)
    assert b[z0 + Z, r0] == K and abs(s[z0 + Z, r0] - (A - 1) * math.sqrt(K)) < 1e-5
    assert (p[z0 + Z, r0] & ((1 << K) - 1 | ((1 << K) - 1) << 16)) == want
    sS, _, _ = oracle_mod.greedy_2d(P, H, mu, sg, NO_DRIFT)
    assert sS[z0 + Z, r0] < s[z0 + Z, r0]                       # the simple sum loses the drifting harmonics
    C = np.full((nz, N), 3.0, np.float32)
    s, b, p = oracle_mod.greedy_2d(C, H, mu, sg, 0)
    assert not p.any()                                          # ties stay on the first candidate
    for z in (-20, -7, -1, 0, 3, 20):
        for r in (0, 1, 100, 187, 1499, 2999):
            n_r = H if r == 0 else min(H, (N - 1) // r)
            n_z = H if z == 0 else min(H, Z // abs(z))
            assert b[z + Z, r] == min(n_r, n_z), (z, r)


def test_r15_bins_entry_agrees_with_the_plane_functions_and_exposes_every_order(oracle_mod):
    """oracle.bins_2d (per-order SNRs for the near-tie rule of the GPU tests) against what is already pinned: its snr and
    best_h equal greedy_2d / presto_2d at the same (z, r); best is the FIRST maximum of its per-order list (strict >);
    the orders that are NaN are exactly those the definition does not evaluate (k r > N - 1 or |k z| > Z for the simple
    sum; orders outside the set {1, 2, 4, ..} for the PRESTO-like form); and for the simple sum the per-order values are
    the cumulative sums of P[k z][k r] written out in numpy."""
    H, nz, N = 8, 9, 300
    Z = (nz - 1) // 2
    P = _int_plane(31, nz, N, 40)
    mu = np.array([2.0 * h for h in range(1, H + 1)], np.float32)
    sg = np.array([2.0 ** (h % 3) for h in range(1, H + 1)], np.float32)
    zi, r = np.meshgrid(np.arange(nz), np.arange(N), indexing="ij")
    zi, r = zi.ravel(), r.ravel()
    for greedy, flags in ((True, 0), (True, NO_DRIFT), (False, 0), (False, ALL_HARMONICS)):
        full = oracle_mod.greedy_2d(P, H, mu, sg, flags) if greedy else oracle_mod.presto_2d(P, H, mu, sg, flags)
        b = oracle_mod.bins_2d(P, H, mu, sg, zi, r, flags, greedy)
        assert np.array_equal(b["snr"], full[0].ravel()) and np.array_equal(b["best_h"], full[1].ravel())
        sh = b["snr_h"]
        filled = np.where(np.isnan(sh), -np.inf, sh)
        assert np.array_equal(filled.max(axis=1), b["snr"])
        assert np.array_equal(filled.argmax(axis=1) + 1, b["best_h"])            # numpy's argmax is the first maximum
        if not greedy:
            in_set = np.array([(flags & ALL_ORDERS) or (h & (h - 1)) == 0 for h in range(1, H + 1)])
            assert np.all(np.isnan(sh[:, ~in_set])) and not np.any(np.isnan(sh[:, in_set]))
        if greedy and flags == NO_DRIFT:
            z = zi - Z
            run = np.zeros(zi.size); alive = np.ones(zi.size, bool)
            for k in range(1, H + 1):
                alive &= (k * r <= N - 1) & (np.abs(k * z) <= Z)
                run[alive] += P[(k * z + Z)[alive], (k * r)[alive]]
                want = (run - float(mu[k - 1])) / float(sg[k - 1])
                assert np.array_equal(np.isnan(sh[:, k - 1]), ~alive)
                assert np.array_equal(sh[alive, k - 1], want[alive])

