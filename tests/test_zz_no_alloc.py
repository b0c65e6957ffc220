"""hs_estimate_stats_static: the statistics step for callers that are not allowed to allocate device memory.

Some users of this library run where a cudaMalloc is off the table: a real-time search pipeline that fixes its device
memory layout at start-up, a plug-in that receives only its input and output buffers from the application that owns
the allocator, a process whose memory pool has no room left.  For them the library carries a fixed 3 MiB accumulator
array inside its own image (one copy per GPU, shared by all calls) and hs_estimate_stats_static uses it in place of the
caller-supplied workspace of hs_estimate_stats.  These tests check, on two calls in a row, that the results are those
of the existing path (the array keeps the previous call's sums, so the second call proves it is cleared), that the
call really allocates nothing, and that a batch beyond the array's capacity is refused with its own error code.

The file sorts after every other test file on purpose: pytest -x stops at the first failure, and a failure in this
extra entry point must not hide the parity tests.  It passes run alone in a fresh process (the first call then does the
per-device address look-up) and after the other GPU tests.
"""
import numpy as np
import pytest
import torch

from paper_2202_12817_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hs():
    from paper_2202_12817_b200 import binding
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    binding.load()                      # fails loudly if libhs_b200.so is missing
    return binding


def _upload(x, ib):
    S, N = x.shape
    istr = (N + 3) & ~3
    dx = torch.zeros((S, istr), dtype=torch.float32, device="cuda")
    dx[:, :N] = torch.as_tensor(x).cuda()
    db = None
    if ib is not None:
        db = torch.ones((S, istr), dtype=torch.float32, device="cuda")
        db[:, :N] = torch.as_tensor(ib).cuda()
    return dx, db, istr


def _existing_path(hs, plan, greedy, dx, db, n_lo, n_hi, clip, n_clip, S, H):
    """hs_estimate_stats with a workspace the caller allocated (here: torch)."""
    mu = torch.full((S, H), float("nan"), dtype=torch.float32, device="cuda")
    sg = torch.full((S, H), float("nan"), dtype=torch.float32, device="cuda")
    work = torch.empty(hs.hs_stats_workspace_bytes(plan, n_clip) // 8, dtype=torch.float64, device="cuda")
    hs.hs_estimate_stats(plan, greedy, dx, db, n_lo, n_hi, clip, n_clip, mu, sg, work)
    torch.cuda.synchronize()
    return mu.cpu().numpy(), sg.cpu().numpy()


def _static_path(hs, plan, greedy, dx, db, n_lo, n_hi, clip, n_clip, S, H):
    """The entry point under test: outputs preallocated, no device memory requested during the call."""
    mu = torch.full((S, H), float("nan"), dtype=torch.float32, device="cuda")
    sg = torch.full((S, H), float("nan"), dtype=torch.float32, device="cuda")
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    hs.hs_estimate_stats_static(plan, greedy, dx, db, n_lo, n_hi, clip, n_clip, mu, sg)
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    return mu.cpu().numpy(), sg.cpu().numpy(), free_before - free_after


@pytest.mark.parametrize("greedy", [True, False])
def test_static_scratch_matches_existing_path_two_calls_in_a_row(hs, greedy):
    """Call 1: exact-integer spectra with outliers and two rejection rounds -- every fp64 moment is an exact integer sum,
    so the results must equal the existing path's bit for bit (the rule of test_estimate_stats_exact_integer).
    Call 2, straight after it on the same stream and a different batch shape: whitened red noise -- the fp64 additions
    come in an unspecified order, so the comparison uses the tolerances of test_estimate_stats_red_noise_and_dstats_run
    (mean 1e-5, deviation 1e-4, relative).  Stale sums from call 1 left in the shared array would break call 2 (and the
    leftovers of earlier test files would break call 1)."""
    # call 1
    H1, S1, N1 = 13, 3, 50001
    x1 = inputs.integer_spectra(81, S1, N1, 40).numpy()
    x1[:, ::501] += 3000.0
    dx1, _, istr1 = _upload(x1, None)
    plan1 = hs.hs_plan(N1, S1, H1, istr1, istr1, 0, 0, 0)
    # call 2
    H2 = 32
    w = inputs.Workload("red", 5, 1 << 16, H2, seed=9, n_pulsars=2, r_range=(100.0, 4000.0), duty_range=(0.02, 0.1),
                        amp_range=(8.0, 12.0), red_noise=True)
    xt = inputs.generate(w)
    ib2 = inputs.block_median_inv_baseline(xt).numpy()
    x2 = xt.numpy()
    S2, N2 = x2.shape
    dx2, db2, istr2 = _upload(x2, ib2)
    plan2 = hs.hs_plan(N2, S2, H2, istr2, istr2, 0, 0, 0)
    try:
        ref1 = _existing_path(hs, plan1, greedy, dx1, None, 77, 9000, 2.5, 2, S1, H1)
        ref2 = _existing_path(hs, plan2, greedy, dx2, db2, N2 // 64, N2 // 32, 3.0, 2, S2, H2)
        mu1, sg1, used1 = _static_path(hs, plan1, greedy, dx1, None, 77, 9000, 2.5, 2, S1, H1)
        mu2, sg2, used2 = _static_path(hs, plan2, greedy, dx2, db2, N2 // 64, N2 // 32, 3.0, 2, S2, H2)
    finally:
        hs.hs_destroy(plan1)
        hs.hs_destroy(plan2)
    assert np.array_equal(mu1, ref1[0]) and np.array_equal(sg1, ref1[1])
    assert np.all(np.isfinite(mu2)) and np.all(sg2 > 0)
    assert np.allclose(mu2, ref2[0], rtol=1e-5, atol=0) and np.allclose(sg2, ref2[1], rtol=1e-4, atol=0)
    # the device's free memory did not shrink across either call (a cudaMalloc of the workspace would show here;
    # the very first call of the process may still make the runtime load code, which is not an allocation of ours,
    # hence only the second call is held to zero)
    assert used2 <= 0, (used1, used2)


def test_static_scratch_same_call_twice_is_repeatable(hs):
    """The same exact-integer call twice in a row: identical bits both times (nothing of call 1 leaks into call 2)."""
    H, S, N = 8, 4, 20011
    x = inputs.integer_spectra(5, S, N, 25).numpy()
    dx, _, istr = _upload(x, None)
    plan = hs.hs_plan(N, S, H, istr, istr, 0, 0, 0)
    try:
        ref = _existing_path(hs, plan, True, dx, None, 0, N, 3.0, 1, S, H)
        a = _static_path(hs, plan, True, dx, None, 0, N, 3.0, 1, S, H)
        b = _static_path(hs, plan, True, dx, None, 0, N, 3.0, 1, S, H)
    finally:
        hs.hs_destroy(plan)
    for got in (a, b):
        assert np.array_equal(got[0], ref[0]) and np.array_equal(got[1], ref[1])


def test_static_scratch_rejects_batches_beyond_its_capacity(hs):
    """(n_clip + 1) * n_spectra > HS_STATIC_STATS_MAX_ROWS: refused with HS_ERR_TOO_LARGE before anything is launched
    (the outputs keep their fill value); the largest admissible batch is accepted."""
    H, N = 4, 64
    for S, n_clip, ok in ((hs.HS_STATIC_STATS_MAX_ROWS, 0, True), (hs.HS_STATIC_STATS_MAX_ROWS // 2, 1, True),
                          (hs.HS_STATIC_STATS_MAX_ROWS + 1, 0, False), (hs.HS_STATIC_STATS_MAX_ROWS // 2 + 1, 1, False)):
        dx = torch.ones((S, N), dtype=torch.float32, device="cuda")
        mu = torch.full((S, H), -5.0, dtype=torch.float32, device="cuda")
        sg = torch.full((S, H), -5.0, dtype=torch.float32, device="cuda")
        plan = hs.hs_plan(N, S, H, N, N, 0, 0, 0)
        try:
            if ok:
                hs.hs_estimate_stats_static(plan, True, dx, None, 0, 8, 3.0, n_clip, mu, sg)
                torch.cuda.synchronize()
                # a constant spectrum: mean h at order h, zero deviation reported as 1
                assert torch.equal(mu[0], torch.arange(1, H + 1, dtype=torch.float32, device="cuda"))
                assert torch.all(sg == 1.0)
            else:
                launches = hs.hs_launch_count(plan)
                with pytest.raises(hs.HsError) as err:
                    hs.hs_estimate_stats_static(plan, True, dx, None, 0, 8, 3.0, n_clip, mu, sg)
                assert err.value.status == hs.HS_ERR_TOO_LARGE and "TOO_LARGE" in str(err.value)
                torch.cuda.synchronize()
                assert hs.hs_launch_count(plan) == launches
                assert torch.all(mu == -5.0) and torch.all(sg == -5.0)
        finally:
            hs.hs_destroy(plan)
