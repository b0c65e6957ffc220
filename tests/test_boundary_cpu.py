"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol include/hs.h
declares; argument validation that needs no device; the N>1 host logic under gloo (world_size 2)."""
import ctypes
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2202_12817_b200 import _build, binding
    _build.build()
    return binding.load()


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "hs.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hs_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_exported(lib):
    from paper_2202_12817_b200 import binding
    names = _declared_symbols()
    assert set(names) == set(binding.EXPORTS)
    for n in names:
        assert getattr(lib, n) is not None


def test_no_torch_types_in_header():
    src = open(os.path.join(ROOT, "include", "hs.h")).read()
    assert "torch" not in src.lower().replace("pytorch", "") and "at::" not in src and 'extern "C"' in src


def test_status_strings(lib):
    for code, word in ((0, "HS_OK"), (1, "INVALID_ARG"), (2, "UNSUPPORTED"), (3, "ALLOC"), (4, "CUDA"), (5, "TOO_LARGE")):
        assert word in lib.hs_status_string(code).decode()


def test_plan_validation_needs_no_device(lib):
    """Invalid arguments are rejected before any CUDA call."""
    plan = ctypes.c_void_p()
    bad = [
        dict(n_bins=1), dict(H=0), dict(H=33), dict(n_spectra=0), dict(n_fund=2000), dict(in_stride=1001),
        dict(in_stride=500), dict(out_stride=10), dict(flags=8),        # ALL_ORDERS without ALL_HARMONICS
        dict(flags=1 << 5), dict(device=-1), dict(n_bins=(1 << 31)),
    ]
    for kw in bad:
        a = dict(n_bins=1000, n_spectra=2, H=8, in_stride=0, out_stride=0, n_fund=0, flags=0, device=0)
        a.update(kw)
        rc = lib.hs_plan(ctypes.byref(plan), a["n_bins"], a["n_spectra"], a["H"], a["in_stride"], a["out_stride"],
                         a["n_fund"], a["flags"], a["device"])
        assert rc == 1, kw
        assert plan.value is None
    assert lib.hs_plan(None, 1000, 1, 8, 0, 0, 0, 0, 0) == 1
    assert lib.hs_destroy(None) == 0
    assert lib.hs_launch_count(None) == -1


def test_product_path_does_not_import_oracle():
    """The product package never references oracle/ (no CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2202_12817_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "hs_oracle" not in txt, f


def test_shard_rows_partition():
    from paper_2202_12817_b200.sharding import shard_rows
    for S in (1, 7, 256, 1000):
        for world in (1, 2, 3, 8):
            spans = [shard_rows(S, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == S
            for a, b in zip(spans, spans[1:]):
                assert a[1] == b[0]
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1


def _gloo_worker(rank, world, port, q):
    import torch.distributed as dist
    from paper_2202_12817_b200.sharding import gather_candidates, max_over_ranks, shard_rows, sum_over_ranks
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    lo, hi = shard_rows(5, rank, world)
    t = max_over_ranks(1.0 + rank)
    tot = sum_over_ranks(float(hi - lo))
    local = torch.tensor([[0, 10 + rank, 2], [hi - lo - 1, 99, 4]], dtype=torch.int64)
    cands = gather_candidates(local, lo)
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, lo, hi, t, tot, cands))


def test_gloo_world2_host_logic():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_gloo_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, lo0, hi0, t0, tot0, c0), (r1, lo1, hi1, t1, tot1, c1) = res
    assert (lo0, hi0, lo1, hi1) == (0, 3, 3, 5)
    assert t0 == t1 == 2.0 and tot0 == tot1 == 5.0
    assert c0 == c1 == [(0, 10, 2), (2, 99, 4), (3, 11, 2), (4, 99, 4)]
