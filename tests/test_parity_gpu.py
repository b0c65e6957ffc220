"""GPU parity: the CUDA path (through the C-ABI, via the thin binding) against the CPU oracle on
the same seeded inputs.  Acceptance rules in tests/parity.py."""
import math

import numpy as np
import pytest
import torch

from paper_2202_12817_b200 import inputs

pytestmark = pytest.mark.gpu

NO_FUND_SELECT, NO_DRIFT, ALL_HARMONICS, ALL_ORDERS = 1, 2, 4, 8
GENERIC = 255                # hs_plan_set_tuning value that forces the coverage kernels


@pytest.fixture(scope="module")
def hs():
    from paper_2202_12817_b200 import binding
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    binding.load()                      # fails loudly if libhs_b200.so is missing
    return binding


def run_greedy(hs, x, H, mu, sg, flags=0, inv_baseline=None, n_fund=0, want_path=True, in_stride=0, out_stride=0, tune=0):
    x = torch.as_tensor(x)
    if x.ndim == 1:
        x = x[None, :]
    S, N = x.shape
    istr = in_stride or ((N + 3) & ~3)
    nf = n_fund or N
    ostr = out_stride or ((nf + 3) & ~3)
    dx = torch.zeros((S, istr), dtype=torch.float32, device="cuda")
    dx[:, :N] = x.cuda()
    db = None
    if inv_baseline is not None:
        db = torch.ones((S, istr), dtype=torch.float32, device="cuda")
        db[:, :N] = torch.as_tensor(inv_baseline).reshape(S, N).cuda()
    snr = torch.full((S, ostr), float("nan"), dtype=torch.float32, device="cuda")
    bh = torch.full((S, ostr), -7, dtype=torch.int32, device="cuda")
    path = torch.full((S, ostr), -7, dtype=torch.int32, device="cuda") if want_path else None
    plan = hs.hs_plan(N, S, H, istr, ostr, n_fund, flags, 0)
    try:
        hs.hs_plan_set_tuning(plan, tune)
        hs.hs_run_greedy(plan, dx, db, mu, sg, snr, bh, path)
        torch.cuda.synchronize()
        assert hs.hs_launch_count(plan) >= 1
    finally:
        hs.hs_destroy(plan)
    # nothing outside [0, n_fund) is written
    assert torch.all(torch.isnan(snr[:, nf:])) and torch.all(bh[:, nf:] == -7)
    return (snr[:, :nf].cpu().numpy(), bh[:, :nf].cpu().numpy(),
            path[:, :nf].cpu().numpy() if want_path else None)


def run_presto(hs, x, H, mu, sg, flags=0, inv_baseline=None, n_fund=0, in_stride=0, out_stride=0, tune=0):
    x = torch.as_tensor(x)
    if x.ndim == 1:
        x = x[None, :]
    S, N = x.shape
    istr = in_stride or ((N + 3) & ~3)
    nf = n_fund or N
    ostr = out_stride or ((nf + 3) & ~3)
    dx = torch.zeros((S, istr), dtype=torch.float32, device="cuda")
    dx[:, :N] = x.cuda()
    db = None
    if inv_baseline is not None:
        db = torch.ones((S, istr), dtype=torch.float32, device="cuda")
        db[:, :N] = torch.as_tensor(inv_baseline).reshape(S, N).cuda()
    snr = torch.full((S, ostr), float("nan"), dtype=torch.float32, device="cuda")
    bh = torch.full((S, ostr), -7, dtype=torch.int32, device="cuda")
    plan = hs.hs_plan(N, S, H, istr, ostr, n_fund, flags, 0)
    try:
        hs.hs_plan_set_tuning(plan, tune)
        hs.hs_run_presto(plan, dx, db, mu, sg, snr, bh)
        torch.cuda.synchronize()
    finally:
        hs.hs_destroy(plan)
    assert torch.all(torch.isnan(snr[:, nf:])) and torch.all(bh[:, nf:] == -7)
    return snr[:, :nf].cpu().numpy(), bh[:, :nf].cpu().numpy()


def _int_stats(H):
    """Integer means and power-of-two sigmas: every SNR is exact in fp32 and fp64 (pin P7)."""
    mu = np.array([3 * h for h in range(1, H + 1)], np.float32)
    sg = np.array([2.0 ** ((h % 4) - 1) for h in range(1, H + 1)], np.float32)
    return mu, sg


# ------------------------------------------------------------------------------------------
# P7: exact-integer spectra -> bit-for-bit agreement (index parity), all kernels, ragged shapes
# ------------------------------------------------------------------------------------------
SHAPES = [(1, 2), (1, 3), (2, 33), (3, 257), (2, 1000), (1, 4099), (5, 70001), (2, 1 << 17)]


# hs_plan_set_tuning values: 0 = the library's choice, 255 = coverage kernels, others = alternative tile shapes
GREEDY_TUNES = [0, 3, 4, 255]        # 4 = tiles in ascending order (hs_greedy_tile_kernel<128,4,false>)
PRESTO_TUNES = [0, 50, 52, 53, 255]


@pytest.mark.parametrize("tune", GREEDY_TUNES)
@pytest.mark.parametrize("H", [1, 8, 13, 32])
def test_greedy_exact_integer(hs, oracle_mod, tune, H):
    mu, sg = _int_stats(H)
    for S, N in SHAPES:
        x = inputs.integer_spectra(100 + N, S, N, 255).numpy()
        for flags in (0, NO_FUND_SELECT):
            s_ref, b_ref, p_ref = oracle_mod.greedy(x, H, mu, sg, flags)
            s, b, p = run_greedy(hs, x, H, mu, sg, flags, tune=tune)
            assert np.array_equal(p.view(np.uint32), p_ref), (S, N, flags)
            assert np.array_equal(b, b_ref), (S, N, flags)
            assert np.array_equal(s.astype(np.float64), s_ref), (S, N, flags)


@pytest.mark.parametrize("tune", PRESTO_TUNES)
@pytest.mark.parametrize("H", [1, 2, 4, 8, 13, 16, 32])
def test_presto_exact_integer(hs, oracle_mod, tune, H):
    mu, sg = _int_stats(H)
    for S, N in SHAPES:
        x = inputs.integer_spectra(200 + N, S, N, 255).numpy()
        s_ref, b_ref = oracle_mod.presto(x, H, mu, sg)
        s, b = run_presto(hs, x, H, mu, sg, tune=tune)
        assert np.array_equal(b, b_ref), (S, N)
        assert np.array_equal(s.astype(np.float64), s_ref), (S, N)


@pytest.mark.parametrize("tune", [t for t in PRESTO_TUNES if t != 255])
@pytest.mark.parametrize("H", [8, 32])
def test_presto_many_tiles_per_cta(hs, oracle_mod, tune, H):
    """Many tiles per row and many rows (one CTA per tile: several waves of CTAs, 8 resident per SM, on every SM),
    ragged rows and rows that start on odd 16-byte units (N = 150001: in_stride = 150004 words, so odd rows are not
    32-byte aligned), against the oracle bit for bit on exact-integer spectra."""
    mu, sg = _int_stats(H)
    S, N = 48, 150001
    x = inputs.integer_spectra(300 + H, S, N, 255).numpy()
    s_ref, b_ref = oracle_mod.presto(x, H, mu, sg)
    s, b = run_presto(hs, x, H, mu, sg, tune=tune)
    assert np.array_equal(b, b_ref)
    assert np.array_equal(s.astype(np.float64), s_ref)


@pytest.mark.parametrize("tune", [0, 255])
@pytest.mark.parametrize("flags", [NO_DRIFT, NO_DRIFT | NO_FUND_SELECT])
def test_simple_hs_exact_integer(hs, oracle_mod, flags, tune):
    H = 16
    mu, sg = _int_stats(H)
    x = inputs.integer_spectra(7, 3, 5003, 255).numpy()
    s_ref, b_ref, p_ref = oracle_mod.greedy(x, H, mu, sg, flags)
    s, b, p = run_greedy(hs, x, H, mu, sg, flags, tune=tune)
    assert np.all(p == 0) and np.array_equal(b, b_ref) and np.array_equal(s.astype(np.float64), s_ref)


@pytest.mark.parametrize("tune", [0, 1, 2, 255])    # library choice / Farey kernel forced / staged kernel forced / generic kernel
@pytest.mark.parametrize("flags", [ALL_HARMONICS, ALL_HARMONICS | ALL_ORDERS])
@pytest.mark.parametrize("H", [1, 2, 5, 16, 27, 32])
def test_presto_variants_exact_integer(hs, oracle_mod, flags, H, tune):
    mu, sg = _int_stats(H)
    for S, N in ((2, 6007), (1, 2), (3, 257), (2, 70001)):
        x = inputs.integer_spectra(8 + N, S, N, 255).numpy()
        s_ref, b_ref = oracle_mod.presto(x, H, mu, sg, flags)
        s, b = run_presto(hs, x, H, mu, sg, flags, tune=tune)
        assert np.array_equal(b, b_ref) and np.array_equal(s.astype(np.float64), s_ref), (S, N)


def test_strides_and_n_fund(hs, oracle_mod):
    H = 8
    mu, sg = _int_stats(H)
    S, N = 3, 5000
    x = inputs.integer_spectra(9, S, N, 255).numpy()
    for tune in (0, 255):
        s_ref, b_ref, p_ref = oracle_mod.greedy(x, H, mu, sg, 0, n_fund=1234)
        s, b, p = run_greedy(hs, x, H, mu, sg, 0, n_fund=1234, in_stride=5008, out_stride=1300, tune=tune)
        assert np.array_equal(p.view(np.uint32), p_ref) and np.array_equal(b, b_ref) and np.array_equal(s.astype(np.float64), s_ref)
        q_ref, c_ref = oracle_mod.presto(x, H, mu, sg, 0, n_fund=777)
        q, c = run_presto(hs, x, H, mu, sg, 0, n_fund=777, in_stride=5120, out_stride=780, tune=tune)
        assert np.array_equal(c, c_ref) and np.array_equal(q.astype(np.float64), q_ref)
    # without the optional path output
    s2, b2, _ = run_greedy(hs, x, H, mu, sg, 0, want_path=False)
    s_ref, b_ref, _ = oracle_mod.greedy(x, H, mu, sg, 0)
    assert np.array_equal(b2, b_ref) and np.array_equal(s2.astype(np.float64), s_ref)


# ------------------------------------------------------------------------------------------
# The BASELINE.json configurations: tolerance-based acceptance (a)-(c)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("tune", [0, 255])
def test_cfg1_both_variants(hs, oracle_mod, tune):
    from parity import check_greedy, check_presto
    w = inputs.workload("cfg1")
    x = inputs.generate(w).numpy()
    mu, sg = (t.numpy() for t in inputs.exp1_stats("greedy", w.H))
    s, b, p = run_greedy(hs, x, w.H, mu, sg, tune=tune)
    r = check_greedy(oracle_mod, x, w.H, mu, sg, 0, s, b, p, T=10.0)
    # the injected pulsar (r = 1000.5) is detected at its fundamental
    top = int(np.argmax(s[0]))
    assert top in (1000, 1001) and s[0, top] > 10.0
    mu, sg = (t.numpy() for t in inputs.exp1_stats("presto", w.H))
    s, b = run_presto(hs, x, w.H, mu, sg, tune=tune)
    check_presto(oracle_mod, x, w.H, mu, sg, 0, s, b, T=10.0)
    assert r["bh_mismatch"] < 10


def test_cfg2_all_rows(hs, oracle_mod):
    """configs[1] at its full size: all 64 spectra x 2^20 bins, H = 16, every output against the oracle."""
    from parity import check_greedy, check_presto
    w = inputs.workload("cfg2")
    x = torch.stack([inputs.generate_row(w, s, "cuda") for s in range(w.n_spectra)]).cpu().numpy()
    assert x.shape == (64, 1 << 20)
    mu, sg = (t.numpy() for t in inputs.exp1_stats("greedy", w.H))
    s, b, p = run_greedy(hs, x, w.H, mu, sg)
    check_greedy(oracle_mod, x, w.H, mu, sg, 0, s, b, p, T=10.0)
    mu, sg = (t.numpy() for t in inputs.exp1_stats("presto", w.H))
    s, b = run_presto(hs, x, w.H, mu, sg)
    check_presto(oracle_mod, x, w.H, mu, sg, 0, s, b, T=10.0)


def test_noise_all_flags_tolerance(hs, oracle_mod):
    from parity import check_greedy, check_presto
    H = 32
    w = inputs.Workload("n", 2, 300001, H, seed=41, n_pulsars=3, r_range=(50.0, 5000.0), duty_range=(0.02, 0.1),
                        amp_range=(6.0, 12.0))
    x = inputs.generate(w).numpy()
    for flags, variant, fs in ((0, "greedy", True), (NO_FUND_SELECT, "greedy", False), (NO_DRIFT, "simple", True)):
        mu, sg = (t.numpy() for t in inputs.exp1_stats(variant, H, fs))
        s, b, p = run_greedy(hs, x, H, mu, sg, flags)
        check_greedy(oracle_mod, x, H, mu, sg, flags, s, b, p, T=8.0)
    for flags, variant in ((0, "presto"), (ALL_HARMONICS, "presto_all"), (ALL_HARMONICS | ALL_ORDERS, "presto_plus")):
        mu, sg = (t.numpy() for t in inputs.exp1_stats(variant, H))
        s, b = run_presto(hs, x, H, mu, sg, flags)
        check_presto(oracle_mod, x, H, mu, sg, flags, s, b, T=8.0)


def test_inv_baseline_red_noise(hs, oracle_mod):
    """configs[3] content at reduced size (NEXT-2): red-noise trend, block-median baseline."""
    from parity import check_greedy, check_presto
    H = 32
    w = inputs.Workload("red", 2, 1 << 17, H, seed=4, n_pulsars=2, r_range=(100.0, 4000.0), duty_range=(0.02, 0.1),
                        amp_range=(8.0, 12.0), red_noise=True)
    xt = inputs.generate(w)
    ib = inputs.block_median_inv_baseline(xt).numpy()
    x = xt.numpy()
    for tune in (0, 3, 255):                 # tuned tile kernels with the multiplier, and the generic kernel
        for flags, fs in ((0, True), (NO_FUND_SELECT, False)):
            mu, sg = (t.numpy() for t in inputs.exp1_stats("greedy", H, fs))
            s, b, p = run_greedy(hs, x, H, mu, sg, flags, inv_baseline=ib, tune=tune)
            check_greedy(oracle_mod, x, H, mu, sg, flags, s, b, p, inv_baseline=ib, T=10.0)
    mu, sg = (t.numpy() for t in inputs.exp1_stats("presto", H))
    s, b = run_presto(hs, x, H, mu, sg, 0, inv_baseline=ib)
    check_presto(oracle_mod, x, H, mu, sg, 0, s, b, inv_baseline=ib, T=10.0)


@pytest.mark.parametrize("tune", [0, 3, 255])
def test_inv_baseline_exact_integer(hs, oracle_mod, tune):
    """Integer powers times power-of-two multipliers: every product, sum and SNR is exact (pin P7 with R13)."""
    H = 32
    mu, sg = _int_stats(H)
    S, N = 3, 30011
    x = inputs.integer_spectra(31, S, N, 63).numpy()
    rng = np.random.default_rng(5)
    ib = (2.0 ** rng.integers(-1, 3, size=(S, N))).astype(np.float32)
    for flags in (0, NO_FUND_SELECT):
        s_ref, b_ref, p_ref = oracle_mod.greedy(x, H, mu, sg, flags, inv_baseline=ib)
        s, b, p = run_greedy(hs, x, H, mu, sg, flags, inv_baseline=ib, tune=tune)
        assert np.array_equal(p.view(np.uint32), p_ref) and np.array_equal(b, b_ref)
        assert np.array_equal(s.astype(np.float64), s_ref)


def _gpu_candidates(hs, plan, snr, bh, T, capacity):
    out = torch.full((max(capacity, 1), 4), -1, dtype=torch.int32, device="cuda")
    cnt = torch.full((1,), -5, dtype=torch.int64, device="cuda")
    hs.hs_find_candidates(plan, snr, bh, T, out if capacity else None, cnt)
    torch.cuda.synchronize()
    k = int(cnt.item())
    got = out[:min(k, capacity)].cpu().numpy()
    order = np.lexsort((got[:, 1], got[:, 0]))
    return k, got[order]


def test_candidates_list(hs, oracle_mod):
    """NEXT-3 / north_star check (c): the candidate list produced on the GPU.  Exact against the plain definition
    applied to the same GPU outputs (integer / selection work), and equal to the oracle's list away from the threshold."""
    w = inputs.workload("cfg1")
    H, T = w.H, 10.0
    x = inputs.generate(w)
    S, N = x.shape
    mu, sg = inputs.exp1_stats("greedy", H)
    dx = x.cuda()
    for n_fund, ostr in ((0, 0), (50001, 50004)):
        nf = n_fund or N
        ostride = ostr or N
        snr = torch.empty((S, ostride), dtype=torch.float32, device="cuda")
        bh = torch.empty((S, ostride), dtype=torch.int32, device="cuda")
        plan = hs.hs_plan(N, S, H, 0, ostride, n_fund, 0, 0)
        try:
            hs.hs_run_greedy(plan, dx, None, mu, sg, snr, bh, None)
            snr[:, nf:] = 1e9                                       # nothing outside [0, n_fund) may be reported
            k, got = _gpu_candidates(hs, plan, snr, bh, T, 1 << 16)
            ref, ref_snr = oracle_mod.candidates(snr[:, :nf].cpu().numpy(), bh[:, :nf].cpu().numpy(), T)
            assert k == ref.shape[0] > 0
            assert np.array_equal(got[:, [0, 1, 3]].astype(np.int64), ref)
            assert np.array_equal(got[:, 2].copy().view(np.float32).astype(np.float64), ref_snr)
            # against the oracle's own outputs: equal except bins whose oracle snr is within tol of T
            s_ref, b_ref, _ = oracle_mod.greedy(x.numpy(), H, mu.numpy(), sg.numpy(), 0, n_fund=nf)
            oref, _ = oracle_mod.candidates(s_ref, b_ref, T)
            near = {(r, c) for r, c in zip(*np.nonzero(np.abs(s_ref - T) <= 2e-5 * max(1.0, T)))}
            a = {(int(r), int(c)) for r, c, _ in ref} - near
            b = {(int(r), int(c)) for r, c, _ in oref} - near
            assert a == b
            # capacity smaller than the list: the count is still the full count, nothing is written past capacity
            k2, got2 = _gpu_candidates(hs, plan, snr, bh, T, 3)
            assert k2 == k and got2.shape[0] == 3
            k3, _ = _gpu_candidates(hs, plan, snr, bh, T, 0)
            assert k3 == k
            k4, got4 = _gpu_candidates(hs, plan, snr, bh, 1e30, 8)
            assert k4 == 0 and got4.shape[0] == 0
        finally:
            hs.hs_destroy(plan)


def test_candidates_dense_and_batch(hs, oracle_mod):
    """Every bin a hit (threshold -inf) and a ragged multi-spectrum batch: count and content exact."""
    S, N, H = 5, 70001, 8
    mu, sg = _int_stats(H)
    x = inputs.integer_spectra(77, S, N, 255)
    snr = torch.empty((S, N + 3), dtype=torch.float32, device="cuda")
    bh = torch.empty((S, N + 3), dtype=torch.int32, device="cuda")
    dx = torch.zeros((S, N + 3), dtype=torch.float32, device="cuda")
    dx[:, :N] = x.cuda()
    plan = hs.hs_plan(N, S, H, N + 3, N + 3, 0, 0, 0)
    try:
        hs.hs_run_presto(plan, dx, None, mu, sg, snr, bh)
        for T in (-1e30, 40.0):
            k, got = _gpu_candidates(hs, plan, snr, bh, T, S * N)
            ref, ref_snr = oracle_mod.candidates(snr[:, :N].cpu().numpy(), bh[:, :N].cpu().numpy(), T)
            assert k == ref.shape[0]
            assert np.array_equal(got[:, [0, 1, 3]].astype(np.int64), ref)
            assert np.array_equal(got[:, 2].copy().view(np.float32).astype(np.float64), ref_snr)
    finally:
        hs.hs_destroy(plan)


def test_sensitivity_loss_workload(hs, oracle_mod):
    """NEXT-3: the paper's noiseless sensitivity-loss experiment (eq. 10-11) as a second workload:
    51 von Mises pulse trains stepping across one bin, 156 251 bins each (ragged), H = 32.  Parity against the oracle
    for every variant, and the statements of the text as soft checks (figures 9-11 are not in PAPER.md)."""
    from parity import check_greedy, check_presto
    from paper_2202_12817_b200 import sensitivity as se
    n_c, H = 500, 32
    xt, _ = se.von_mises_spectra(n_c=n_c, device="cuda")
    x = xt.cpu().numpy()
    S, N = x.shape
    assert (S, N) == (51, 156251)
    # scalloping: a half-bin offset keeps |sinc(pi/2)|^2 = 0.405 of the bin-centred power
    assert abs(x[25, n_c] / x[0, n_c] - (2.0 / np.pi) ** 2) < 0.01
    mu = np.zeros(H, np.float32)
    root = np.sqrt(np.arange(1, H + 1)).astype(np.float32)
    pterms = np.sqrt([1.0 if h == 1 else 1.0 + h / 2.0 for h in range(1, H + 1)]).astype(np.float32)
    loss, rsnr0 = {}, {}
    for name, flags in (("greedy", 0), ("greedy_nofs", NO_FUND_SELECT), ("simple", NO_DRIFT)):
        s, b, p = run_greedy(hs, x, H, mu, root, flags)
        check_greedy(oracle_mod, x, H, mu, root, flags, s, b, p, T=None)
        loss[name] = se.loss_curve(torch.from_numpy(s)).numpy()
        rsnr0[name] = s[0, 10:].max()
    for name, flags, sg in (("presto", 0, pterms), ("presto_all", ALL_HARMONICS, root), ("presto_plus", ALL_HARMONICS | ALL_ORDERS, root)):
        s, b = run_presto(hs, x, H, mu, sg, flags)
        check_presto(oracle_mod, x, H, mu, sg, flags, s, b, T=None)
        loss[name] = se.loss_curve(torch.from_numpy(s)).numpy()
        rsnr0[name] = s[0, 10:].max()
    g, sm = loss["greedy"], loss["simple"]
    assert abs(g[50] - 1.0) < 1e-3 and abs(sm[50] - 1.0) < 1e-3          # next bin centre: no loss
    assert np.abs(g - g[::-1]).max() < 0.01                             # drift tracked: symmetric about the bin border
    assert np.abs(loss["greedy_nofs"] - loss["greedy_nofs"][::-1]).max() > 0.1   # without fundamental selection it is not
    assert g.min() > 0.65 and sm.min() < 0.5                            # simple HS loses about half
    assert abs(rsnr0["greedy"] / rsnr0["presto_plus"] - 1.0) < 1e-4     # same maximum RSNR as PRESTO+ 
    assert rsnr0["presto"] < rsnr0["presto_all"] <= rsnr0["presto_plus"] * (1 + 1e-6)


# ------------------------------------------------------------------------------------------
# Host-buffer entry points (the e2e leg of bench.py) and error behaviour
# ------------------------------------------------------------------------------------------
def test_host_entry_points(hs, oracle_mod):
    H = 16
    mu, sg = _int_stats(H)
    S, N = 9, 40000
    x = inputs.integer_spectra(10, S, N, 255)
    hx = x.pin_memory()
    snr = torch.empty((S, N), dtype=torch.float32).pin_memory()
    bh = torch.empty((S, N), dtype=torch.int32).pin_memory()
    path = torch.empty((S, N), dtype=torch.int32).pin_memory()
    plan = hs.hs_plan(N, S, H, N, N, 0, 0, 0)
    try:
        hs.hs_run_greedy_host(plan, hx, None, mu, sg, snr, bh, path)
        s_ref, b_ref, p_ref = oracle_mod.greedy(x.numpy(), H, mu, sg)
        assert np.array_equal(path.numpy().view(np.uint32), p_ref) and np.array_equal(bh.numpy(), b_ref)
        assert np.array_equal(snr.numpy().astype(np.float64), s_ref)
        hs.hs_run_presto_host(plan, hx, None, mu, sg, snr, bh)
        q_ref, c_ref = oracle_mod.presto(x.numpy(), H, mu, sg)
        assert np.array_equal(bh.numpy(), c_ref) and np.array_equal(snr.numpy().astype(np.float64), q_ref)
        assert hs.hs_launch_count(plan) >= 2
    finally:
        hs.hs_destroy(plan)


def test_error_behaviour(hs):
    N, S, H = 1024, 2, 8
    x = torch.ones((S, N), device="cuda")
    snr = torch.empty((S, N), device="cuda")
    bh = torch.empty((S, N), dtype=torch.int32, device="cuda")
    mu, sg = _int_stats(H)
    plan = hs.hs_plan(N, S, H)
    try:
        bad_sg = sg.copy(); bad_sg[3] = 0.0
        with pytest.raises(hs.HsError) as e:
            hs.hs_run_greedy(plan, x, None, mu, bad_sg, snr, bh)
        assert e.value.status == hs.HS_ERR_INVALID_ARG
        with pytest.raises(hs.HsError):
            hs.hs_run_presto(plan, x.view(-1)[1:-3].view(-1), None, mu, sg, snr, bh)     # misaligned pointer
        with pytest.raises(hs.HsError):
            hs.hs_run_greedy(plan, x, None, mu, sg, snr, snr.view(torch.int32))           # aliasing outputs
        # overlapping but unequal ranges: the output starts inside the input array / inside the other output
        big = torch.empty(3 * S * N, device="cuda")
        for bad_x, bad_snr, bad_bh in ((big[:S * N].view(S, N), big[N:N + S * N].view(S, N), bh),
                                       (x, big[:S * N].view(S, N), big[4:4 + S * N].view(S, N).view(torch.int32))):
            with pytest.raises(hs.HsError) as e:
                hs.hs_run_greedy(plan, bad_x, None, mu, sg, bad_snr, bad_bh)
            assert e.value.status == hs.HS_ERR_INVALID_ARG
            with pytest.raises(hs.HsError):
                hs.hs_run_presto(plan, bad_x, None, mu, sg, bad_snr, bad_bh)
        hs.hs_run_greedy(plan, big[:S * N].view(S, N), None, mu, sg, big[S * N:2 * S * N].view(S, N), bh)   # adjacent, not overlapping: fine
        hs.hs_plan_set_host_slot_bytes(plan, 1 << 20)
        with pytest.raises(hs.HsError):
            hs.hs_plan_set_host_slot_bytes(plan, 0)
        hs.hs_run_greedy(plan, x, None, mu, sg, snr, bh)                                   # the plan is still usable
        torch.cuda.synchronize()
        assert torch.all(bh >= 1)
    finally:
        hs.hs_destroy(plan)
    with pytest.raises(hs.HsError):
        hs.hs_plan(N, S, 64)


# ------------------------------------------------------------------------------------------
# Full size, in the launch configuration bench.py times (configs[2]: 256 x 2^22, H = 32)
# ------------------------------------------------------------------------------------------
def test_cfg3_full_size_sampled_rows(hs, oracle_mod):
    """The whole 4 GiB batch goes through one hs_run_* call each (exactly what bench.py times);
    rows the oracle can afford are compared element by element, every row is checked for the
    properties that hold at any size."""
    from parity import check_greedy, check_presto
    w = inputs.workload("cfg3")
    S, N, H = w.n_spectra, w.n_bins, w.H
    free, _ = torch.cuda.mem_get_info()
    if free < 20 * (1 << 30):
        pytest.skip("needs 20 GiB of device memory")
    x = inputs.generate(w, "cuda")
    snr = torch.empty((S, N), dtype=torch.float32, device="cuda")
    bh = torch.empty((S, N), dtype=torch.int32, device="cuda")
    path = torch.empty((S, N), dtype=torch.int32, device="cuda")
    pulsar_rows = sorted({p.spectrum for p in w.pulsars})
    rows = [0, pulsar_rows[0], pulsar_rows[len(pulsar_rows) // 2], S - 1]
    xs = x[rows].cpu().numpy()
    plan = hs.hs_plan(N, S, H)
    try:
        mu, sg = (t.numpy() for t in inputs.exp1_stats("greedy", H))
        hs.hs_run_greedy(plan, x, None, mu, sg, snr, bh, path)
        torch.cuda.synchronize()
        assert int(bh.min()) >= 1 and int(bh.max()) <= H and bool(torch.isfinite(snr).all())
        # S_1 >= x[n]  <=>  best >= (x[n] - mu_1)/sigma_1 (P6), at every bin of every row
        floor1 = (x - float(mu[0])) / float(sg[0])
        assert bool((snr >= floor1 - 1e-5 * (floor1.abs() + 1)).all())
        del floor1
        # bins n >= N/2 evaluate order 1 only: best_h = 1 and path in {0, 1}
        assert bool((bh[:, N // 2 + 1:] == 1).all()) and int(path[:, N // 2 + 1:].max()) <= 1
        check_greedy(oracle_mod, xs, H, mu, sg, 0, snr[rows].cpu().numpy(), bh[rows].cpu().numpy(),
                     path[rows].cpu().numpy(), T=10.0)
        mu, sg = (t.numpy() for t in inputs.exp1_stats("presto", H))
        hs.hs_run_presto(plan, x, None, mu, sg, snr, bh)
        torch.cuda.synchronize()
        assert int(bh.min()) >= 1 and int(bh.max()) <= H and bool(torch.isfinite(snr).all())
        # H' = 1 is always a candidate: best >= (x[n] - mu_1)/sigma_1
        floor1 = (x - float(mu[0])) / float(sg[0])
        assert bool((snr >= floor1 - 1e-5 * (floor1.abs() + 1)).all())
        del floor1
        check_presto(oracle_mod, xs, H, mu, sg, 0, snr[rows].cpu().numpy(), bh[rows].cpu().numpy(), T=10.0)
    finally:
        hs.hs_destroy(plan)


def _sample_bins(N, rng, k=6000):
    edges = np.concatenate([np.arange(0, 64), np.arange(N - 64, N)] +
                           [np.arange(max(0, N // d - 40), min(N, N // d + 40)) for d in (2, 3, 4, 8, 16, 31, 32, 33, 64)])
    return np.unique(np.concatenate([edges, rng.integers(0, N, size=k), rng.integers(0, max(1, N // 32), size=k)]))


@pytest.mark.parametrize("kind,N,kernel", [
    ("greedy", (1 << 30) + 7, "hs_greedy_tile_kernel"),            # 32-bit h n close to its limit
    ("presto", (1 << 26) - 70, "hs_presto_tile_kernel"),           # 32 N just below 2^31
    ("presto", (1 << 26) + 8, "hs_presto_generic_kernel"),         # just past the rows kernel's limit
    ("greedy", (1 << 31) - (1 << 17), "hs_greedy_tile_kernel"),    # the last N the tile kernel takes
    ("greedy", (1 << 31) - 64, "hs_greedy_generic_kernel"),        # the largest N hs_plan accepts: 64-bit offsets
])
def test_maximum_sizes_sampled(hs, oracle_mod, kind, N, kernel):
    """Largest rows the fast paths accept and the first sizes past each fast-path limit (which kernel ran is
    asserted through hs_last_kernel).  Exact-integer spectra, so sampled outputs must equal the oracle's bit for
    bit (the oracle computes the sampled bins one by one)."""
    free, _ = torch.cuda.mem_get_info()
    if free < 30 * (1 << 30):
        pytest.skip("needs 30 GiB of device memory")
    H = 32
    mu, sg = _int_stats(H)
    rng = np.random.default_rng(11)
    if True:
        g = torch.Generator(device="cuda"); g.manual_seed(5)
        istr = (N + 3) & ~3
        x = torch.zeros((1, istr), dtype=torch.float32, device="cuda")
        step = 1 << 28                                             # in pieces: no 8 GiB temporaries
        for a in range(0, N, step):
            b = min(N, a + step)
            x[0, a:b] = torch.randint(0, 256, (b - a,), generator=g, device="cuda", dtype=torch.int32).to(torch.float32)
        snr = torch.empty((1, istr), dtype=torch.float32, device="cuda")
        bh = torch.empty((1, istr), dtype=torch.int32, device="cuda")
        path = torch.empty((1, istr), dtype=torch.int32, device="cuda") if kind == "greedy" else None
        plan = hs.hs_plan(N, 1, H, istr, istr, 0, 0, 0)
        try:
            if kind == "greedy":
                hs.hs_run_greedy(plan, x, None, mu, sg, snr, bh, path)
            else:
                hs.hs_run_presto(plan, x, None, mu, sg, snr, bh)
            torch.cuda.synchronize()
            assert hs.hs_last_kernel(plan).startswith(kernel), hs.hs_last_kernel(plan)
        finally:
            hs.hs_destroy(plan)
        bins = _sample_bins(N, rng)
        idx = torch.from_numpy(bins).cuda()
        xh = x[0, :N].cpu().numpy()[None, :]
        rows = np.zeros_like(bins)
        if kind == "greedy":
            ref = oracle_mod.greedy_bins(xh, H, mu, sg, rows, bins)
            assert np.array_equal(path[0, idx].cpu().numpy().view(np.uint32), ref["path"])
        else:
            ref = oracle_mod.presto_bins(xh, H, mu, sg, rows, bins)
        assert np.array_equal(bh[0, idx].cpu().numpy(), ref["best_h"])
        assert np.array_equal(snr[0, idx].cpu().numpy().astype(np.float64), ref["snr"])
        del x, snr, bh, path, xh
        torch.cuda.empty_cache()


# ------------------------------------------------------------------------------------------
# All rows of the headline batch: tuned kernels against the coverage kernels (which the oracle vouches for
# element by element in the tests above), so that the oracle-checked rows vouch for the rest
# ------------------------------------------------------------------------------------------
def test_cfg3_all_rows_tuned_vs_generic(hs, oracle_mod):
    """cfg3 content, all 256 rows, one launch each.  Greedy: the tile kernel and hs_greedy_generic_kernel add the
    same fp32 terms in the same order, so snr, best_h and path must be equal bit for bit.  PRESTO: the rows kernel
    adds level by level (hs.h "Precision"), so snr agrees within the fp32 accumulation bound and best_h may differ
    only where the two maxima are within that bound; on exact-integer spectra of the same shape it is bit for bit."""
    w = inputs.workload("cfg3")
    S, N, H = w.n_spectra, w.n_bins, w.H
    free, _ = torch.cuda.mem_get_info()
    if free < 32 * (1 << 30):
        pytest.skip("needs 32 GiB of device memory")
    x = inputs.generate(w, "cuda")
    out = [torch.empty((S, N), dtype=torch.float32 if k % 3 == 0 else torch.int32, device="cuda") for k in range(6)]
    plan = hs.hs_plan(N, S, H)
    try:
        mu, sg = (t.numpy() for t in inputs.exp1_stats("greedy", H))
        hs.hs_plan_set_tuning(plan, 0)
        hs.hs_run_greedy(plan, x, None, mu, sg, out[0], out[1], out[2])
        assert hs.hs_last_kernel(plan).startswith("hs_greedy_tile_kernel")
        hs.hs_plan_set_tuning(plan, GENERIC)
        hs.hs_run_greedy(plan, x, None, mu, sg, out[3], out[4], out[5])
        assert hs.hs_last_kernel(plan).startswith("hs_greedy_generic_kernel")
        torch.cuda.synchronize()
        assert torch.equal(out[2], out[5]) and torch.equal(out[1], out[4])
        assert torch.equal(out[0].view(torch.int32), out[3].view(torch.int32))
        mu, sg = (t.numpy() for t in inputs.exp1_stats("presto", H))
        for content in ("cfg3", "integer"):
            if content == "integer":
                g = torch.Generator(device="cuda"); g.manual_seed(9)
                for s in range(S):
                    x[s] = torch.randint(0, 64, (N,), generator=g, device="cuda", dtype=torch.int32).to(torch.float32)
                mu, sg = _int_stats(H)
            hs.hs_plan_set_tuning(plan, 0)
            hs.hs_run_presto(plan, x, None, mu, sg, out[0], out[1])
            assert hs.hs_last_kernel(plan).startswith("hs_presto_tile_kernel")
            hs.hs_plan_set_tuning(plan, GENERIC)
            hs.hs_run_presto(plan, x, None, mu, sg, out[3], out[4])
            assert hs.hs_last_kernel(plan).startswith("hs_presto_generic_kernel")
            torch.cuda.synchronize()
            if content == "integer":
                assert torch.equal(out[1], out[4]) and torch.equal(out[0].view(torch.int32), out[3].view(torch.int32))
                rng = np.random.default_rng(3)
                rows = np.repeat(np.array([0, 100, S - 1]), 2000)
                bins = np.tile(_sample_bins(N, rng, 900)[:2000], 3)
                hrows = {r: x[r].cpu().numpy() for r in (0, 100, S - 1)}
                for r in (0, 100, S - 1):
                    bsel = bins[rows == r]
                    ref = oracle_mod.presto_bins(hrows[r][None, :], H, mu, sg, np.zeros_like(bsel), bsel)
                    idx = torch.from_numpy(bsel).cuda()
                    assert np.array_equal(out[1][r, idx].cpu().numpy(), ref["best_h"])
                    assert np.array_equal(out[0][r, idx].cpu().numpy().astype(np.float64), ref["snr"])
            else:
                err = (out[0] - out[3]).abs()
                bound = 1e-5 * (out[3].abs() + float(mu[-1]) / float(sg[-1]) + 1.0)
                assert bool((err <= bound).all())
                mism = int((out[1] != out[4]).sum())
                assert mism <= 1e-4 * S * N, mism          # near-ties only (their snr already agree within the bound)
            del_err = None
    finally:
        hs.hs_destroy(plan)


# ------------------------------------------------------------------------------------------
# configs[3] at its real size: 1024 x 2^21 = 2^31 elements per array, row offsets beyond int32
# ------------------------------------------------------------------------------------------
def test_cfg4_full_size(hs, oracle_mod):
    """One hs_run_greedy call over the whole cfg4 batch with its whitening multiplier (reading R13).  Rows 0, 511,
    512 and 1023 (element offsets below, at and beyond 2^31) are compared with the oracle element by element
    (path bit-exact), and every row of the tile kernel is compared bit for bit with the generic 64-bit kernel."""
    from parity import check_greedy
    w = inputs.workload("cfg4")
    S, N, H = w.n_spectra, w.n_bins, w.H
    assert S * N == 1 << 31
    free, _ = torch.cuda.mem_get_info()
    if free < 72 * (1 << 30):
        pytest.skip("needs 72 GiB of device memory")
    x = inputs.generate(w, "cuda")
    ib = torch.empty_like(x)
    for s0 in range(0, S, 64):
        ib[s0:s0 + 64] = inputs.block_median_inv_baseline(x[s0:s0 + 64])
    out = [torch.empty((S, N), dtype=torch.float32 if k % 3 == 0 else torch.int32, device="cuda") for k in range(6)]
    mu, sg = (t.numpy() for t in inputs.exp1_stats("greedy", H))
    plan = hs.hs_plan(N, S, H)
    try:
        hs.hs_run_greedy(plan, x, ib, mu, sg, out[0], out[1], out[2])
        assert hs.hs_last_kernel(plan).startswith("hs_greedy_tile_kernel")
        hs.hs_plan_set_tuning(plan, GENERIC)
        hs.hs_run_greedy(plan, x, ib, mu, sg, out[3], out[4], out[5])
        assert hs.hs_last_kernel(plan).startswith("hs_greedy_generic_kernel")
        torch.cuda.synchronize()
    finally:
        hs.hs_destroy(plan)
    assert torch.equal(out[2], out[5]) and torch.equal(out[1], out[4])
    assert torch.equal(out[0].view(torch.int32), out[3].view(torch.int32))
    rows = [0, 511, 512, S - 1]
    check_greedy(oracle_mod, x[rows].cpu().numpy(), H, mu, sg, 0, out[0][rows].cpu().numpy(), out[1][rows].cpu().numpy(),
                 out[2][rows].cpu().numpy(), inv_baseline=ib[rows].cpu().numpy(), T=10.0)


# ------------------------------------------------------------------------------------------
# NEXT-2: hs_estimate_stats (reading R14 of GetMeanStdev) and the per-spectrum statistics entry points
# ------------------------------------------------------------------------------------------
def _gpu_stats(hs, x, H, flags, greedy, n_lo, n_hi, clip, n_clip, inv_baseline=None, cached=False):
    S, N = x.shape
    istr = (N + 3) & ~3
    dx = torch.zeros((S, istr), dtype=torch.float32, device="cuda")
    dx[:, :N] = torch.as_tensor(x).cuda()
    db = None
    if inv_baseline is not None:
        db = torch.ones((S, istr), dtype=torch.float32, device="cuda")
        db[:, :N] = torch.as_tensor(inv_baseline).cuda()
    mu = torch.full((S, H), float("nan"), dtype=torch.float32, device="cuda")
    sg = torch.full((S, H), float("nan"), dtype=torch.float32, device="cuda")
    plan = hs.hs_plan(N, S, H, istr, istr, 0, flags, 0)
    try:
        nbytes = hs.hs_stats_workspace_bytes_cached(plan, n_clip, n_lo, n_hi) if cached else hs.hs_stats_workspace_bytes(plan, n_clip)
        # own bounds check (no sanitizer on this pool): 32 guard words on either side of the workspace must survive
        nw = (nbytes + 7) // 8
        store = torch.full((nw + 64,), -12345.0, dtype=torch.float64, device="cuda")
        work = store[32:32 + nw]
        hs.hs_estimate_stats(plan, greedy, dx, db, n_lo, n_hi, clip, n_clip, mu, sg, work)
        torch.cuda.synchronize()
        assert torch.all(store[:32] == -12345.0) and torch.all(store[32 + nw:] == -12345.0), "write outside the workspace"
        assert ("hs_stats_cached_kernel" in hs.hs_last_kernel(plan)) == (cached and n_clip >= 1 and n_hi > n_lo)
        last = work[:(n_clip + 1) * S * 96].view(n_clip + 1, S, 32, 3)[n_clip, :, :H, 0].cpu().numpy().astype(np.int64)
    finally:
        hs.hs_destroy(plan)
    return mu.cpu().numpy(), sg.cpu().numpy(), last


@pytest.mark.parametrize("greedy,flags", [(True, 0), (True, NO_FUND_SELECT), (True, NO_DRIFT), (False, 0),
                                          (False, ALL_HARMONICS), (False, ALL_HARMONICS | ALL_ORDERS)])
def test_estimate_stats_exact_integer(hs, oracle_mod, greedy, flags):
    """Exact-integer spectra: the fp32 partial sums equal the oracle's fp64 ones, every fp64 moment is an exact
    integer sum whatever the order of the additions, so counts, means and deviations must equal the oracle's exactly,
    rounds of outlier rejection included; the range crosses the greedy band edges."""
    H, S, N = 13, 3, 50001
    x = inputs.integer_spectra(81, S, N, 40).numpy()
    x[:, ::501] += 3000.0                                  # outliers for the rejection rounds
    for n_lo, n_hi, n_clip in ((0, N, 0), (77, 9000, 2), (1000, 1001, 0), (5, 5, 1)):
        mu_r, sg_r, cnt_r = oracle_mod.estimate_stats(x, H, flags, greedy, n_lo, n_hi, clip=2.5, n_clip=n_clip)
        for cached in (False, True):        # True: one gather pass, the rejection rounds stream the stored sums
            mu, sg, cnt = _gpu_stats(hs, x, H, flags, greedy, n_lo, n_hi, 2.5, n_clip, cached=cached)
            assert np.array_equal(cnt, cnt_r), (n_lo, n_hi, n_clip, cached)
            assert np.array_equal(mu, mu_r) and np.array_equal(sg, sg_r), (n_lo, n_hi, n_clip, cached)


def test_estimate_stats_red_noise_and_dstats_run(hs, oracle_mod):
    """cfg4 content at reduced size: statistics of the whitened greedy sums with two rejection rounds against the
    oracle (fp32 vs fp64 partial sums: relative 1e-5; a sum within rounding of a limit may be kept on one side only),
    then hs_run_greedy_dstats / hs_run_presto_dstats with per-spectrum statistics against the oracle run row by row."""
    from parity import check_greedy, check_presto
    H = 32
    w = inputs.Workload("red", 3, 1 << 17, H, seed=4, n_pulsars=2, r_range=(100.0, 4000.0), duty_range=(0.02, 0.1),
                        amp_range=(8.0, 12.0), red_noise=True)
    xt = inputs.generate(w)
    ib = inputs.block_median_inv_baseline(xt).numpy()
    x = xt.numpy()
    S, N = x.shape
    n_lo, n_hi = N // 64, N // 32
    for greedy in (True, False):
        mu_r, sg_r, cnt_r = oracle_mod.estimate_stats(x, H, 0, greedy, n_lo, n_hi, clip=3.0, n_clip=2, inv_baseline=ib)
        mu_c, sg_c, cnt_c = _gpu_stats(hs, x, H, 0, greedy, n_lo, n_hi, 3.0, 2, inv_baseline=ib, cached=True)
        mu, sg, cnt = _gpu_stats(hs, x, H, 0, greedy, n_lo, n_hi, 3.0, 2, inv_baseline=ib)
        # the cached path compares the same fp32 sums with the same limits: identical counts unless a limit itself moved
        # by the rounding of the fp64 additions' order
        assert np.all(np.abs(cnt_c - cnt) <= 1) and np.allclose(mu_c, mu, rtol=1e-6, atol=0) and np.allclose(sg_c, sg, rtol=1e-5, atol=0)
        assert np.all(np.abs(cnt - cnt_r) <= 2)
        assert np.allclose(mu, mu_r, rtol=1e-5, atol=0) and np.allclose(sg, sg_r, rtol=1e-4, atol=0)
        if greedy:      # whitened noise: each step adds about the larger of two Exp(1)
            h = np.arange(1, H + 1)
            assert np.all(np.abs(mu / (1.5 * h) - 1.0) < 0.1)
        # the estimated statistics drive the run: per-spectrum mu / sigma from device memory
        dmu, dsg = torch.from_numpy(mu).cuda(), torch.from_numpy(sg).cuda()
        dx, db = torch.from_numpy(x).cuda(), torch.from_numpy(ib).cuda()
        for tune in (0, GENERIC):
            snr = torch.empty((S, N), dtype=torch.float32, device="cuda")
            bh = torch.empty((S, N), dtype=torch.int32, device="cuda")
            path = torch.empty((S, N), dtype=torch.int32, device="cuda")
            plan = hs.hs_plan(N, S, H)
            try:
                hs.hs_plan_set_tuning(plan, tune)
                if greedy:
                    hs.hs_run_greedy_dstats(plan, dx, db, dmu, dsg, snr, bh, path)
                else:
                    hs.hs_run_presto_dstats(plan, dx, db, dmu, dsg, snr, bh)
                torch.cuda.synchronize()
            finally:
                hs.hs_destroy(plan)
            for s in range(S):
                if greedy:
                    check_greedy(oracle_mod, x[s:s + 1], H, mu[s], sg[s], 0, snr[s:s + 1].cpu().numpy(), bh[s:s + 1].cpu().numpy(),
                                 path[s:s + 1].cpu().numpy(), inv_baseline=ib[s:s + 1], T=10.0)
                else:
                    check_presto(oracle_mod, x[s:s + 1], H, mu[s], sg[s], 0, snr[s:s + 1].cpu().numpy(), bh[s:s + 1].cpu().numpy(),
                                 inv_baseline=ib[s:s + 1], T=10.0)


def test_dstats_equals_by_value_statistics(hs, oracle_mod):
    """The same statistics for every spectrum through the device arrays and through the host arrays: identical bits
    (tile kernels without the multiplier, all tile shapes of the by-value path are the default one here)."""
    H, S, N = 32, 4, 70004                                  # rows start on odd 16-byte units
    x = inputs.generate(inputs.Workload("n", S, N, H, seed=12)).cuda()
    out = [torch.empty((S, N + 4), dtype=torch.float32 if k % 2 == 0 else torch.int32, device="cuda") for k in range(4)]
    plan = hs.hs_plan(N, S, H, N, N + 4, 0, 0, 0)
    try:
        for form in ("greedy", "presto"):
            mu, sg = inputs.exp1_stats(form, H)
            dmu, dsg = mu.repeat(S, 1).cuda(), sg.repeat(S, 1).cuda()
            if form == "greedy":
                hs.hs_run_greedy(plan, x, None, mu, sg, out[0], out[1], None)
                hs.hs_run_greedy_dstats(plan, x, None, dmu, dsg, out[2], out[3], None)
            else:
                hs.hs_run_presto(plan, x, None, mu, sg, out[0], out[1])
                hs.hs_run_presto_dstats(plan, x, None, dmu, dsg, out[2], out[3])
            torch.cuda.synchronize()
            assert torch.equal(out[0][:, :N].view(torch.int32), out[2][:, :N].view(torch.int32)) and torch.equal(out[1][:, :N], out[3][:, :N])
    finally:
        hs.hs_destroy(plan)


def test_dstats_unusable_entries_become_zero_one(hs, oracle_mod):
    """include/hs.h (hs_run_*_dstats): a device-side sigma that is not positive and finite, or a non-finite mu, is
    replaced by (0, 1) for that spectrum and order, in every kernel.  Against hs_run_* with the repaired statistics
    passed by value, row by row, bit for bit; the row crosses the streaming top band (order 1 only) and the gather
    bands, and the coverage kernels must agree with the tile kernels."""
    H, S, N = 16, 3, 40000
    x = inputs.generate(inputs.Workload("n", S, N, H, seed=21)).cuda()
    for form in ("greedy", "presto"):
        mu, sg = inputs.exp1_stats(form, H)
        dmu, dsg = mu.repeat(S, 1).clone(), sg.repeat(S, 1).clone()
        dsg[0, 0] = 0.0; dsg[0, 3] = -2.0; dsg[1, 1] = float("nan"); dsg[1, 7] = float("inf")
        dmu[2, 0] = float("nan"); dmu[2, 15] = float("-inf")
        bad = ~((dsg > 0) & torch.isfinite(dsg) & torch.isfinite(dmu))
        fmu, fsg = dmu.clone(), dsg.clone()
        fmu[bad] = 0.0; fsg[bad] = 1.0
        for tune in (0, GENERIC):
            got = [torch.empty((S, N), dtype=torch.float32, device="cuda"), torch.empty((S, N), dtype=torch.int32, device="cuda")]
            plan = hs.hs_plan(N, S, H)
            plan1 = hs.hs_plan(N, 1, H)
            try:
                hs.hs_plan_set_tuning(plan, tune); hs.hs_plan_set_tuning(plan1, tune)
                run_d = hs.hs_run_greedy_dstats if form == "greedy" else hs.hs_run_presto_dstats
                args = (None,) if form == "greedy" else ()
                run_d(plan, x, None, dmu.cuda(), dsg.cuda(), got[0], got[1], *args)
                torch.cuda.synchronize()
                assert torch.all(got[1] >= 1) and not torch.any(torch.isnan(got[0]))
                for s in range(S):
                    ref = [torch.empty((1, N), dtype=torch.float32, device="cuda"), torch.empty((1, N), dtype=torch.int32, device="cuda")]
                    run_v = hs.hs_run_greedy if form == "greedy" else hs.hs_run_presto
                    run_v(plan1, x[s:s + 1].contiguous(), None, fmu[s], fsg[s], ref[0], ref[1], *args)
                    torch.cuda.synchronize()
                    assert torch.equal(got[0][s].view(torch.int32), ref[0][0].view(torch.int32)) and torch.equal(got[1][s], ref[1][0]), (form, tune, s)
            finally:
                hs.hs_destroy(plan); hs.hs_destroy(plan1)


def test_estimate_stats_rejection_limits_inclusive(hs, oracle_mod):
    """Reading R14: a round keeps lo <= S_h(n) <= hi.  The constructed spectrum of the CPU pin
    (tests/test_oracle_pins.py::limits_spectrum: eight order-1 sums, mean 10, deviation 2, clip 2 -> the limits are
    exactly the samples 6 and 14): the device compares its fp32 sum with the fp32-rounded limits, the oracle its fp64
    sum -- here both are exact, so a wrong comparison direction or limit rounding on either side shows as a count of 6."""
    from test_oracle_pins import limits_spectrum
    x, n_lo, n_hi, clip = limits_spectrum()
    for n_clip in (0, 1, 2):
        for greedy, flags in ((True, NO_DRIFT | NO_FUND_SELECT), (False, 0)):       # order 1 of both forms is x[n]
            mu_r, sg_r, cnt_r = oracle_mod.estimate_stats(x, 1, flags, greedy, n_lo, n_hi, clip=clip, n_clip=n_clip)
            for cached in (False, True):
                mu, sg, cnt = _gpu_stats(hs, x, 1, flags, greedy, n_lo, n_hi, clip, n_clip, cached=cached)
                assert cnt[0, 0] == cnt_r[0, 0] == 8 and mu[0, 0] == mu_r[0, 0] == 10.0 and sg[0, 0] == sg_r[0, 0] == 2.0
    for cached in (False, True):
        mu, sg, cnt = _gpu_stats(hs, x, 1, NO_DRIFT | NO_FUND_SELECT, True, n_lo, n_hi, 1.999, 1, cached=cached)
        assert cnt[0, 0] == 6 and mu[0, 0] == 10.0 and sg[0, 0] == 1.0


# ------------------------------------------------------------------------------------------
# NEXT-4 (reading R15): 2-D harmonic sums over an f-fdot plane
# ------------------------------------------------------------------------------------------
def _run_2d(hs, P, H, mu, sg, flags, form, tune=0, want_path=True):
    P = torch.as_tensor(P)
    nz, N = P.shape
    istr = (N + 3) & ~3
    dP = torch.zeros((nz, istr), dtype=torch.float32, device="cuda")
    dP[:, :N] = P.cuda()
    snr = torch.full((nz, istr), float("nan"), dtype=torch.float32, device="cuda")
    bh = torch.full((nz, istr), -7, dtype=torch.int32, device="cuda")
    path = torch.full((nz, istr), -7, dtype=torch.int32, device="cuda") if (want_path and form == "greedy") else None
    plan = hs.hs_plan_2d(N, nz, H, istr, istr, flags, 0)
    try:
        hs.hs_plan_set_tuning(plan, tune)
        if form == "greedy":
            hs.hs_run_greedy_2d(plan, dP, mu, sg, snr, bh, path)
        else:
            hs.hs_run_presto_2d(plan, dP, mu, sg, snr, bh)
        torch.cuda.synchronize()
        kern = hs.hs_last_kernel(plan)
    finally:
        hs.hs_destroy(plan)
    assert torch.all(torch.isnan(snr[:, N:])) and torch.all(bh[:, N:] == -7)
    return snr[:, :N].cpu().numpy(), bh[:, :N].cpu().numpy(), (path[:, :N].cpu().numpy() if path is not None else None), kern


PLANES = [(1, 2), (1, 700), (3, 3), (5, 4099), (41, 1000), (201, 3001), (9, 70001)]


@pytest.mark.parametrize("H", [1, 2, 5, 8, 16])
def test_2d_exact_integer(hs, oracle_mod, H):
    """Exact-integer planes, ragged shapes: greedy 2-D (ours) / simple 2-D / PRESTO-like 2-D family against the oracle
    bit for bit (snr, best_h, path), tile kernel and coverage kernel."""
    mu, sg = _int_stats(H)
    for nz, N in PLANES:
        P = inputs.integer_spectra(500 + N + nz, nz, N, 255).numpy()
        for flags in (0, NO_FUND_SELECT, NO_DRIFT):
            s_ref, b_ref, p_ref = oracle_mod.greedy_2d(P, H, mu, sg, flags)
            s, b, p, _ = _run_2d(hs, P, H, mu, sg, flags, "greedy")
            assert np.array_equal(p.view(np.uint32), p_ref), (nz, N, flags)
            assert np.array_equal(b, b_ref) and np.array_equal(s.astype(np.float64), s_ref), (nz, N, flags)
        for flags, tunes in ((0, (0, GENERIC)), (ALL_HARMONICS, (0,)), (ALL_HARMONICS | ALL_ORDERS, (0,))):
            s_ref, b_ref = oracle_mod.presto_2d(P, H, mu, sg, flags)
            for tune in tunes:
                s, b, _, kern = _run_2d(hs, P, H, mu, sg, flags, "presto", tune=tune)
                assert kern.startswith("hs_presto_tile_kernel" if (flags == 0 and tune == 0) else "hs_presto2d_generic_kernel")
                assert np.array_equal(b, b_ref) and np.array_equal(s.astype(np.float64), s_ref), (nz, N, flags, tune)


def _check_2d(snr_ref, bh_ref, snr, bh, mu, sg, T=10.0, per_order=None, rows=None):
    """tests/parity.py rules for a plane.  Where best_h differs from the oracle's, the order the GPU chose must lie in the
    oracle's near-tie set: its ORACLE snr (per_order(zi, r) -> [k, H], oracle.bins_2d) within tol of the oracle's best."""
    from parity import REL, _tol
    mu = np.asarray(mu, np.float64); sg = np.asarray(sg, np.float64)
    snr = snr.astype(np.float64)
    tol = _tol(snr_ref, mu, sg)
    S = snr_ref * sg[bh_ref - 1] + mu[bh_ref - 1]
    bound = np.where(snr_ref >= 1.0, REL * np.abs(snr_ref), REL * (np.abs(S) + mu[bh_ref - 1]) / sg[bh_ref - 1])
    err = np.abs(snr - snr_ref)
    assert np.all(err <= bound), err.max()
    bad = bh != bh_ref
    assert np.all(err[bad] <= tol[bad])
    if per_order is not None and bad.any():
        at = np.argwhere(bad)
        assert np.all((bh[bad] >= 1) & (bh[bad] <= mu.size))
        zi = at[:, 0] if rows is None else np.asarray(rows)[at[:, 0]]
        snr_h = per_order(zi, at[:, 1])
        got = snr_h[np.arange(at.shape[0]), bh[bad] - 1]                 # NaN (order not evaluated) fails the comparison
        assert np.all(got >= snr_ref[bad] - tol[bad]), "best_h outside the oracle's near-tie set"
    near = np.abs(snr_ref - T) <= tol
    assert np.array_equal((snr >= T) & ~near, (snr_ref >= T) & ~near)
    return int(bad.sum())


def test_2d_cfg5_content_reduced(hs, oracle_mod):
    """configs[4] content (Exp(1) plane with drifting signals) at 41 x 2^16, H = 16: all three forms within the
    tolerances of tests/parity.py; the greedy path is bit-exact; every injected signal is a candidate of the greedy form."""
    H = 16
    w = inputs.PlaneWorkload("p", 41, 1 << 16, H, seed=5, n_signals=4)
    P = inputs.generate_plane(w, "cuda").cpu().numpy()
    Z = 20
    for flags, variant in ((0, "greedy"), (NO_DRIFT, "simple")):
        mu, sg = (t.numpy() for t in inputs.exp1_stats("simple", H))      # any statistics do: parity does not depend on them
        s_ref, b_ref, p_ref = oracle_mod.greedy_2d(P, H, mu, sg, flags)
        s, b, p, _ = _run_2d(hs, P, H, mu, sg, flags, "greedy")
        assert np.array_equal(p.view(np.uint32), p_ref)
        _check_2d(s_ref, b_ref, s, b, mu, sg, per_order=lambda zi, r: oracle_mod.bins_2d(P, H, mu, sg, zi, r, flags, True)["snr_h"])
        if flags == 0:
            for sgn in w.signals:
                r0, z0 = int(math.floor(sgn.r)), int(math.floor(sgn.z))
                assert s[z0 + Z - 1:z0 + Z + 2, r0 - 1:r0 + 2].max() > 10.0
    for flags, variant in ((0, "presto"), (ALL_HARMONICS, "presto_all")):
        mu, sg = (t.numpy() for t in inputs.exp1_stats(variant, H))
        s_ref, b_ref = oracle_mod.presto_2d(P, H, mu, sg, flags)
        s, b, _, _ = _run_2d(hs, P, H, mu, sg, flags, "presto")
        _check_2d(s_ref, b_ref, s, b, mu, sg, per_order=lambda zi, r: oracle_mod.bins_2d(P, H, mu, sg, zi, r, flags, False)["snr_h"])


def test_2d_cfg5_full_size_sampled_rows(hs, oracle_mod):
    """configs[4] at its real size (201 x 2^21, H = 16) through one call per form, as bench.py --workload cfg5 times it;
    rows z = -100, -6, -1, 0, 1, 3, 50, 100 against the oracle (which reads the whole plane but computes those rows)."""
    w = inputs.plane_workload("cfg5")
    H, nz, N = w.H, w.n_z, w.n_bins
    free, _ = torch.cuda.mem_get_info()
    if free < 12 * (1 << 30):
        pytest.skip("needs 12 GiB of device memory")
    dP = inputs.generate_plane(w, "cuda")
    P = dP.cpu().numpy()
    snr = torch.empty((nz, N), dtype=torch.float32, device="cuda")
    bh = torch.empty((nz, N), dtype=torch.int32, device="cuda")
    path = torch.empty((nz, N), dtype=torch.int32, device="cuda")
    rows = [0, 94, 99, 100, 101, 103, 150, 200]
    plan = hs.hs_plan_2d(N, nz, H)
    try:
        mu, sg = (t.numpy() for t in inputs.exp1_stats("simple", H))
        hs.hs_run_greedy_2d(plan, dP, mu, sg, snr, bh, path)
        torch.cuda.synchronize()
        assert int(bh.min()) >= 1 and int(bh.max()) <= H and bool(torch.isfinite(snr).all())
        for zi in rows:
            s_ref, b_ref, p_ref = oracle_mod.greedy_2d(P, H, mu, sg, 0, rows=(zi, zi + 1))
            assert np.array_equal(path[zi].cpu().numpy().view(np.uint32), p_ref[zi])
            _check_2d(s_ref[zi:zi + 1], b_ref[zi:zi + 1], snr[zi:zi + 1].cpu().numpy(), bh[zi:zi + 1].cpu().numpy(), mu, sg, rows=[zi],
                      per_order=lambda z_, r_: oracle_mod.bins_2d(P, H, mu, sg, z_, r_, 0, True)["snr_h"])
        mu, sg = (t.numpy() for t in inputs.exp1_stats("presto", H))
        hs.hs_run_presto_2d(plan, dP, mu, sg, snr, bh)
        torch.cuda.synchronize()
        assert hs.hs_last_kernel(plan).startswith("hs_presto_tile_kernel")
        assert int(bh.min()) >= 1 and int(bh.max()) <= H and bool(torch.isfinite(snr).all())
        for zi in rows:
            s_ref, b_ref = oracle_mod.presto_2d(P, H, mu, sg, 0, rows=(zi, zi + 1))
            _check_2d(s_ref[zi:zi + 1], b_ref[zi:zi + 1], snr[zi:zi + 1].cpu().numpy(), bh[zi:zi + 1].cpu().numpy(), mu, sg, rows=[zi],
                      per_order=lambda z_, r_: oracle_mod.bins_2d(P, H, mu, sg, z_, r_, 0, False)["snr_h"])
    finally:
        hs.hs_destroy(plan)


def test_2d_plans_and_1d_entry_points_do_not_mix(hs):
    mu, sg = _int_stats(8)
    x = torch.ones((3, 1024), device="cuda"); snr = torch.empty_like(x); bh = torch.empty((3, 1024), dtype=torch.int32, device="cuda")
    p2 = hs.hs_plan_2d(1024, 3, 8)
    p1 = hs.hs_plan(1024, 3, 8)
    try:
        with pytest.raises(hs.HsError):
            hs.hs_run_greedy(p2, x, None, mu, sg, snr, bh)
        with pytest.raises(hs.HsError):
            hs.hs_run_presto_2d(p1, x, mu, sg, snr, bh)
        with pytest.raises(hs.HsError):
            hs.hs_plan_2d(1024, 4, 8)            # n_z must be odd
        with pytest.raises(hs.HsError):
            hs.hs_plan_2d(1024, 3, 32)           # H <= 16
    finally:
        hs.hs_destroy(p1); hs.hs_destroy(p2)


def test_whiten_pass_equals_fused_multiplier(hs, oracle_mod):
    """hs_whiten then hs_run_*(y, NULL) returns the bits of hs_run_*(x, inv_baseline) (reading R13: one fp32 multiply),
    ragged rows included; nothing beyond n_bins of a row is written."""
    H, S, N = 32, 3, 50001
    istr = (N + 3) & ~3
    w = inputs.Workload("red", S, N, H, seed=4, n_pulsars=2, r_range=(100.0, 1500.0), duty_range=(0.02, 0.1), amp_range=(8.0, 12.0), red_noise=True)
    x = torch.zeros((S, istr), device="cuda"); x[:, :N] = inputs.generate(w, "cuda")
    ib = torch.ones((S, istr), device="cuda"); ib[:, :N] = inputs.block_median_inv_baseline(x[:, :N].contiguous())
    y = torch.full((S, istr), float("nan"), device="cuda")
    out = [torch.empty((S, istr), dtype=torch.float32 if k % 2 == 0 else torch.int32, device="cuda") for k in range(4)]
    plan = hs.hs_plan(N, S, H, istr, istr, 0, 0, 0)
    try:
        hs.hs_whiten(plan, x, ib, y)
        torch.cuda.synchronize()
        assert torch.equal(y[:, :N], x[:, :N] * ib[:, :N]) and bool(torch.isnan(y[:, N:]).all())
        mu, sg = inputs.exp1_stats("greedy", H)
        hs.hs_run_greedy(plan, x, ib, mu, sg, out[0], out[1])
        hs.hs_run_greedy(plan, y, None, mu, sg, out[2], out[3])
        torch.cuda.synchronize()
        assert torch.equal(out[0][:, :N].view(torch.int32), out[2][:, :N].view(torch.int32)) and torch.equal(out[1][:, :N], out[3][:, :N])
        mu, sg = inputs.exp1_stats("presto", H)
        hs.hs_run_presto(plan, x, ib, mu, sg, out[0], out[1])
        hs.hs_run_presto(plan, y, None, mu, sg, out[2], out[3])
        torch.cuda.synchronize()
        # the fused path runs the coverage kernel (written order), the whitened one the tile kernel (level order)
        assert torch.allclose(out[0][:, :N], out[2][:, :N], rtol=1e-5, atol=2e-5)
    finally:
        hs.hs_destroy(plan)


def test_more_than_65535_spectra(hs, oracle_mod):
    """gridDim.y carries the spectrum index and is limited to 65 535: larger batches go out in slices (every pointer,
    the per-spectrum statistics included, advances with the slice).  65 540 short spectra, exact integers."""
    H, S, N = 4, 65540, 64
    mu, sg = _int_stats(H)
    x = inputs.integer_spectra(900, 4, S * N // 4, 100).reshape(S, N).contiguous().numpy()
    s_ref, b_ref, p_ref = oracle_mod.greedy(x, H, mu, sg, 0)
    s, b, p = run_greedy(hs, x, H, mu, sg, 0)
    assert np.array_equal(p.view(np.uint32), p_ref) and np.array_equal(b, b_ref) and np.array_equal(s.astype(np.float64), s_ref)
    q_ref, c_ref = oracle_mod.presto(x, H, mu, sg)
    q, c = run_presto(hs, x, H, mu, sg)
    assert np.array_equal(c, c_ref) and np.array_equal(q.astype(np.float64), q_ref)
    # per-spectrum statistics from the device: spectrum s gets mu + (s % 7), so a slice that did not advance its
    # statistics pointer would be caught; estimated statistics of the last rows against the oracle
    dx = torch.from_numpy(x).cuda()
    dmu = (torch.from_numpy(mu)[None, :] + (torch.arange(S) % 7)[:, None].float()).cuda().contiguous()
    dsg = torch.from_numpy(sg)[None, :].repeat(S, 1).cuda().contiguous()
    snr = torch.empty((S, N), dtype=torch.float32, device="cuda"); bh = torch.empty((S, N), dtype=torch.int32, device="cuda")
    emu = torch.empty((S, H), device="cuda"); esg = torch.empty((S, H), device="cuda")
    plan = hs.hs_plan(N, S, H)
    try:
        hs.hs_run_greedy_dstats(plan, dx, None, dmu, dsg, snr, bh, None)
        work = torch.empty(hs.hs_stats_workspace_bytes(plan, 1) // 8, dtype=torch.float64, device="cuda")
        hs.hs_estimate_stats(plan, True, dx, None, 1, 16, 3.0, 1, emu, esg, work)
        torch.cuda.synchronize()
    finally:
        hs.hs_destroy(plan)
    for srow in (0, 65534, 65535, 65536, S - 1):
        r_s, r_b, _ = oracle_mod.greedy(x[srow], H, dmu[srow].cpu().numpy(), sg, 0)
        assert np.array_equal(bh[srow].cpu().numpy(), r_b[0]) and np.array_equal(snr[srow].cpu().numpy().astype(np.float64), r_s[0])
    m_r, s_r, _ = oracle_mod.estimate_stats(x[65530:], H, 0, True, 1, 16, clip=3.0, n_clip=1)
    assert np.array_equal(emu[65530:].cpu().numpy(), m_r) and np.array_equal(esg[65530:].cpu().numpy(), s_r)


def test_host_path_many_slots_and_both_forms(hs, oracle_mod, monkeypatch):
    """The host entry points stream the batch through two staging slots on two streams: with a 1 MiB slot
    (hs_plan_set_host_slot_bytes, unstable knob) 20 spectra of 40 000 bins take four chunks, so slots are re-used while the
    other stream is busy.  hs_run_both_host (one upload, both forms), with multiplier and path, against the oracle bit
    for bit on exact integers."""
    H, S, N = 16, 20, 40000
    mu, sg = _int_stats(H)
    x = inputs.integer_spectra(15, S, N, 63)
    rng = np.random.default_rng(8)
    ib = torch.from_numpy((2.0 ** rng.integers(-1, 3, size=(S, N))).astype(np.float32))
    pin = lambda t: t.pin_memory()
    hx, hib = pin(x), pin(ib)
    snr_g = pin(torch.empty((S, N), dtype=torch.float32)); bh_g = pin(torch.empty((S, N), dtype=torch.int32))
    path = pin(torch.empty((S, N), dtype=torch.int32))
    snr_p = pin(torch.empty((S, N), dtype=torch.float32)); bh_p = pin(torch.empty((S, N), dtype=torch.int32))
    for use_ib in (False, True):
        plan = hs.hs_plan(N, S, H, N, N, 0, 0, 0)
        hs.hs_plan_set_host_slot_bytes(plan, 1 << 20)        # 1 MiB slots: several staging chunks
        try:
            hs.hs_run_both_host(plan, hx, hib if use_ib else None, mu, sg, snr_g, bh_g, path, mu, sg, snr_p, bh_p)
            assert hs.hs_launch_count(plan) >= 8            # four chunks x two forms
        finally:
            hs.hs_destroy(plan)
        kw = dict(inv_baseline=ib.numpy()) if use_ib else {}
        s_ref, b_ref, p_ref = oracle_mod.greedy(x.numpy(), H, mu, sg, 0, **kw)
        assert np.array_equal(path.numpy().view(np.uint32), p_ref) and np.array_equal(bh_g.numpy(), b_ref)
        assert np.array_equal(snr_g.numpy().astype(np.float64), s_ref)
        q_ref, c_ref = oracle_mod.presto(x.numpy(), H, mu, sg, 0, **kw)
        assert np.array_equal(bh_p.numpy(), c_ref) and np.array_equal(snr_p.numpy().astype(np.float64), q_ref)


def test_search_host_candidates_only(hs, oracle_mod, monkeypatch):
    """hs_search_host: one upload, both forms, threshold + compaction on the device, only the lists come back.  Against the
    plain definition applied to the oracle's outputs (exact integers, so every snr is exact), several staging chunks,
    and a capacity smaller than the list."""
    H, S, N = 16, 20, 40000
    mu, sg = _int_stats(H)
    x = inputs.integer_spectra(16, S, N, 63)
    s_ref, b_ref, _ = oracle_mod.greedy(x.numpy(), H, mu, sg, 0)
    q_ref, c_ref = oracle_mod.presto(x.numpy(), H, mu, sg, 0)
    T = float(np.float32(min(np.sort(s_ref.ravel())[-5000], np.sort(q_ref.ravel())[-5000])))     # at least 5 000 hits per form
    hx = x.pin_memory()
    cg = torch.full((1 << 20, 4), -1, dtype=torch.int32); cp = torch.full((1 << 20, 4), -1, dtype=torch.int32)
    plan = hs.hs_plan(N, S, H, N, N, 0, 0, 0)
    hs.hs_plan_set_host_slot_bytes(plan, 1 << 20)        # 1 MiB slots: several staging chunks
    try:
        ng, np_ = hs.hs_search_host(plan, hx, None, mu, sg, mu, sg, T, cg, cp)
        small = torch.full((5, 4), -1, dtype=torch.int32)
        ng2, _ = hs.hs_search_host(plan, hx, None, mu, sg, mu, sg, T, small, cp)
    finally:
        hs.hs_destroy(plan)
    for got, n, (sr, br) in ((cg, ng, (s_ref, b_ref)), (cp, np_, (q_ref, c_ref))):
        ref, ref_snr = oracle_mod.candidates(sr.astype(np.float32), br, T)
        assert n == ref.shape[0] and 10 < n < got.shape[0]
        g = got[:n].numpy()
        g = g[np.lexsort((g[:, 1], g[:, 0]))]
        assert np.array_equal(g[:, [0, 1, 3]].astype(np.int64), ref)
        assert np.array_equal(g[:, 2].copy().view(np.float32).astype(np.float64), ref_snr)
    assert ng2 == ng and bool((small[:, 0] >= 0).all())


def test_search_host_with_multiplier(hs, oracle_mod, monkeypatch):
    """hs_search_host with h_inv_baseline: power-of-two multipliers on exact-integer spectra (every product and every
    SNR exact), several staging chunks: both candidate lists equal the definition applied to the oracle's outputs with
    the same multiplier, and differ from the lists without it."""
    H, S, N = 16, 12, 40000
    mu, sg = _int_stats(H)
    x = inputs.integer_spectra(17, S, N, 63)
    g = torch.Generator(); g.manual_seed(3)
    ib = torch.pow(2.0, torch.randint(-1, 2, (S, N), generator=g).to(torch.float32))      # 0.5, 1, 2
    s_ref, b_ref, _ = oracle_mod.greedy(x.numpy(), H, mu, sg, 0, inv_baseline=ib.numpy())
    q_ref, c_ref = oracle_mod.presto(x.numpy(), H, mu, sg, 0, inv_baseline=ib.numpy())
    T = float(np.float32(min(np.sort(s_ref.ravel())[-3000], np.sort(q_ref.ravel())[-3000])))
    cg = torch.full((1 << 18, 4), -1, dtype=torch.int32); cp = torch.full((1 << 18, 4), -1, dtype=torch.int32)
    cg0 = torch.full((1 << 18, 4), -1, dtype=torch.int32); cp0 = torch.full((1 << 18, 4), -1, dtype=torch.int32)
    plan = hs.hs_plan(N, S, H, N, N, 0, 0, 0)
    hs.hs_plan_set_host_slot_bytes(plan, 1 << 20)        # 1 MiB slots: several staging chunks
    try:
        ng, np_ = hs.hs_search_host(plan, x.pin_memory(), ib.pin_memory(), mu, sg, mu, sg, T, cg, cp)
        ng0, np0 = hs.hs_search_host(plan, x.pin_memory(), None, mu, sg, mu, sg, T, cg0, cp0)
    finally:
        hs.hs_destroy(plan)
    assert (ng0, np0) != (ng, np_)
    for got, n, (sr, br) in ((cg, ng, (s_ref, b_ref)), (cp, np_, (q_ref, c_ref))):
        ref, ref_snr = oracle_mod.candidates(sr.astype(np.float32), br, T)
        assert n == ref.shape[0] and 10 < n < got.shape[0]
        a = got[:n].numpy()
        a = a[np.lexsort((a[:, 1], a[:, 0]))]
        assert np.array_equal(a[:, [0, 1, 3]].astype(np.int64), ref)
        assert np.array_equal(a[:, 2].copy().view(np.float32).astype(np.float64), ref_snr)


@pytest.mark.parametrize("flags,tune,kernel", [(ALL_HARMONICS, 0, "hs_presto_farey_kernel"), (ALL_HARMONICS, 2, "hs_presto_plus_kernel"),
                                               (ALL_HARMONICS | ALL_ORDERS, 0, "hs_presto_plus_kernel"),
                                               (ALL_HARMONICS | ALL_ORDERS, 1, "hs_presto_farey_kernel")])
def test_presto_variants_cfg3_sized_row(hs, oracle_mod, flags, tune, kernel):
    """PRESTO_all / PRESTO+ (PAPER.md:174, 368), both kernels of each, on rows of cfg3's length (2^22 bins, H = 32):
    thousands of tiles per row instead of the few of the small exact-integer shapes.  Exact-integer spectrum, sampled
    top bins (band edges, both ends of the row, random bins) computed one by one by the oracle: bit-for-bit."""
    H, S, N = 32, 2, 1 << 22
    mu, sg = _int_stats(H)
    x = inputs.integer_spectra(404, S, N, 255)
    snr = torch.empty((S, N), dtype=torch.float32, device="cuda")
    bh = torch.empty((S, N), dtype=torch.int32, device="cuda")
    plan = hs.hs_plan(N, S, H, N, N, 0, flags, 0)
    try:
        hs.hs_plan_set_tuning(plan, tune)
        hs.hs_run_presto(plan, x.cuda(), None, mu, sg, snr, bh)
        torch.cuda.synchronize()
        assert hs.hs_last_kernel(plan) == kernel
    finally:
        hs.hs_destroy(plan)
    bins = _sample_bins(N, np.random.default_rng(8), k=3000)
    for row in range(S):
        ref = oracle_mod.presto_bins(x.numpy(), H, mu, sg, np.full(bins.shape, row), bins, flags)
        assert np.array_equal(bh[row].cpu().numpy()[bins], ref["best_h"])
        assert np.array_equal(snr[row].cpu().numpy()[bins].astype(np.float64), ref["snr"])
