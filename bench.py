#!/usr/bin/env python
"""bench.py -- throughput of the harmonic-sum hot path (arXiv 2202.12817) on B200.

One STEP = one pass of the whole hot path over one batch of synthetic
power spectra: hs_run_greedy (Alg. 2) followed by hs_run_presto (Alg. 1,
PAPER.md:144-162) on the same batch, i.e. every spectrum bin receives both outputs.
Workload at N=1: BASELINE.json configs[2] ("cfg3": 256 DM trials x 2^22 fp32 bins, H = 32), the
configuration the metric is quoted on.  N>1: every rank owns its own 256 spectra (weak scaling,
no data-path collective: spectra are independent).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

Prints ONE JSON line (rank 0).  `value` = spectrum bins per second with the inputs resident in HBM
(paper eq. 12, counted once per bin although both forms are computed);
`e2e` = the same through hs_run_*_host with pinned HOST buffers (H2D + D2H inside the timed region).
`--impl reference` times the CPU oracle (oracle/, test infrastructure) on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "harmonic-sum spectrum bins/s at H=32 (greedy + PRESTO-like forms per bin)"
UNIT = "bins/s"
BYTES_PER_BIN = 12.0          # compulsory HBM bytes per bin and per form: 4 read + 4 + 4 written
FALLBACK_HBM_GBS = 6650.0     # /opt/skills/guides/B200_PROFILING.md, used only if MEASURED_PEAKS.json is absent
# Committed ncu evidence: profiles/ncu_kernels.json maps the name hs_last_kernel() reports to the per-launch
# counters of the `ncu --set full` capture of that kernel on cfg3 (dram bytes, L2 -> SM sectors);
# profiles/machine_model.json holds the measured L2 -> SM ceiling.  A kernel that is not in the file gets
# traffic = null (no stale numbers).
NCU_KERNELS_JSON = os.path.join(ROOT, "profiles", "ncu_kernels.json")
MACHINE_MODEL_JSON = os.path.join(ROOT, "profiles", "machine_model.json")


def _load_json(path):
    try:
        with open(path) as f:
            return json.load(f)
    except Exception:
        return {}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="cfg3", help="inputs.workload name (cfg3 = headline)")
    ap.add_argument("--spectra", type=int, default=0, help="override the number of spectra per rank (0 = workload's)")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--cpu-spectra", type=int, default=64, help="spectra in the oracle's bounded sample")
    ap.add_argument("--H", type=int, default=0, help="override the workload's maximum harmonic order (paper Table 2: 4, 8, 16, 32)")
    ap.add_argument("--forms", default="both", choices=["both", "greedy", "presto"],
                    help="which forms a step runs (cfg4 is quoted on the greedy form only)")
    ap.add_argument("--greedy-flags", type=int, default=0, help="HS_GREEDY_* plan flags (NEXT-1 variants)")
    ap.add_argument("--presto-flags", type=int, default=0, help="HS_PRESTO_* plan flags (NEXT-1 variants)")
    ap.add_argument("--stats", default="auto", choices=["auto", "given", "estimated"],
                    help="given: closed-form Exp(1) statistics passed by value; estimated: hs_estimate_stats (reading R14 of "
                         "GetMeanStdev) inside the step, then hs_run_*_dstats; auto = estimated for the red-noise workload (cfg4)")
    ap.add_argument("--whiten", default="pass", choices=["pass", "fused"],
                    help="red-noise workload (cfg4): pass = hs_whiten writes x * inv_baseline once and the sums read that array; "
                         "fused = every gather multiplies (two arrays read by the gather)")
    ap.add_argument("--no-extra", action="store_true",
                    help="skip the `extra` object of the default run (H sweep, NEXT-1 variants, streaming rate, cfg4 and cfg5 lines)")
    ap.add_argument("--n-fund-div", type=int, default=1,
                    help="diagnostic: outputs only for n < N / D (hs_plan's n_fund), e.g. 8 = the greedy gather band without "
                         "the streaming top band, for ncu captures; bins/s then counts S * N / D bins")
    ap.add_argument("--tune-greedy", type=int, default=0)
    ap.add_argument("--tune-presto", type=int, default=0)
    return ap.parse_args()


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy burst)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, reasons, smax, pw = [], set(), None, []
        try:
            for line in open(self.path):
                f = [t.strip() for t in line.split(",")]
                if len(f) < 9:
                    continue
                try:
                    sm.append(float(f[1])); smax = float(f[2]); pw.append(float(f[3]))
                except ValueError:
                    continue
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            s = sorted(sm)
            out.update(sm_mhz=s[len(s) // 2], sm_max_mhz=smax, reasons=sorted(reasons), samples=len(sm),
                       power_w_max=max(pw) if pw else None)
        return out


def respawn_under_torchrun(args) -> int:
    """`python bench.py --gpus N` (N > 1) outside torchrun: start the N ranks ourselves, one per GPU."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")                # the communicator lines (ranks, NVLS) of a scaling run
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd, env=env)


def dist_setup(n_gpus: int):
    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world != max(1, n_gpus):
        raise SystemExit(f"bench.py: --gpus {n_gpus} but WORLD_SIZE={world}: launch with torchrun --nproc-per-node {n_gpus} "
                         f"(or run `python bench.py --gpus {n_gpus}` outside torchrun: it starts the ranks itself)")
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        os.environ.setdefault("NCCL_DEBUG", "INFO")         # communicator lines of a scaling run (only the timing all-reduce uses NCCL)
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    return rank, local, world


def barrier(world):
    import torch
    import torch.distributed as dist
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()


def _variants(args):
    """(greedy stats variant, fund_select, PRESTO stats variant) for the plan flags of this run."""
    gv = "simple" if args.greedy_flags & 2 else "greedy"
    pv = "presto_plus" if (args.presto_flags & 12) == 12 else "presto_all" if args.presto_flags & 4 else "presto"
    return gv, not (args.greedy_flags & 1), pv


def run_cpu_sample(x_host, H, n_threads=None, args=None, ib_host=None):
    """Time the oracle, as it stands, on a [rows, N] float32 numpy sample: greedy then PRESTO."""
    import oracle
    from paper_2202_12817_b200 import inputs
    oracle.build()
    cores = n_threads or oracle.host_threads()
    gv, fs, pv = _variants(args) if args is not None else ("greedy", True, "presto")
    gflags = args.greedy_flags if args is not None else 0
    pflags = args.presto_flags if args is not None else 0
    forms = args.forms if args is not None else "both"
    mu_g, sg_g = inputs.exp1_stats(gv, H, fs)
    mu_p, sg_p = inputs.exp1_stats(pv, H)
    t0 = time.perf_counter()
    if forms != "presto":
        oracle.greedy(x_host, H, mu_g.numpy(), sg_g.numpy(), gflags, inv_baseline=ib_host, n_threads=cores, want_path=False)
    t1 = time.perf_counter()
    if forms != "greedy":
        oracle.presto(x_host, H, mu_p.numpy(), sg_p.numpy(), pflags, inv_baseline=ib_host, n_threads=cores)
    t2 = time.perf_counter()
    bins = x_host.shape[0] * x_host.shape[1]
    return {"bins": bins, "seconds": t2 - t0, "greedy_s": t1 - t0, "presto_s": t2 - t1, "cores": cores}


def run_reference(args):
    """--impl reference: the CPU oracle timed on the host cores, rank 0 only, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import torch
    from paper_2202_12817_b200 import inputs
    w = inputs.workload(args.workload)
    rows = min(args.cpu_spectra, w.n_spectra)
    dev = "cuda" if torch.cuda.is_available() else "cpu"   # generator only (no method arithmetic)
    x = inputs.generate(w, device=dev, n_spectra=rows).cpu().numpy()
    for _ in range(args.warmup):
        run_cpu_sample(x[:max(1, rows // 8)], w.H)
    tot, bins, cores = 0.0, 0, 0
    for _ in range(args.steps):
        r = run_cpu_sample(x, w.H)
        tot += r["seconds"]; bins += r["bins"]; cores = r["cores"]
    value = bins / tot
    sample = f"first {rows} of {w.n_spectra} spectra of {w.name} ({rows}x{w.n_bins} bins), greedy + PRESTO, fp64"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{w.name}: {w.n_spectra} spectra x {w.n_bins} fp32 bins, H={w.H}, greedy + PRESTO (Alg. 1)",
                       "step": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def child_line(argv, keys, timeout=600):
    """Run this script once more for another workload (its own process: its own buffers) and keep `keys` of its JSON line."""
    try:
        out = subprocess.run([sys.executable, os.path.abspath(__file__), "--no-e2e", "--no-cpu", "--no-extra"] + argv,
                             capture_output=True, text=True, timeout=timeout)
        for ln in reversed(out.stdout.splitlines()):
            if ln.startswith("{"):
                rec = json.loads(ln)
                return {k: rec.get(k) for k in keys}
        return {"error": f"no JSON line (rc {out.returncode}): {out.stderr[-300:]}"}
    except Exception as e:          # the headline line must not depend on an extra
        return {"error": repr(e)}


def run_cuda(args):
    import torch
    from paper_2202_12817_b200 import binding as hs
    from paper_2202_12817_b200 import inputs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    hs.load()
    rank, local, world = dist_setup(args.gpus)
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    w = inputs.workload(args.workload)
    S = args.spectra or w.n_spectra
    N, H = w.n_bins, (args.H or w.H)
    # rank r owns global rows [r*S, (r+1)*S): weak scaling, no exchange
    x = torch.empty((S, N), dtype=torch.float32, device=dev)
    for s in range(S):
        x[s].copy_(inputs.generate_row(w, rank * S + s, dev))
    do_g, do_p = args.forms != "presto", args.forms != "greedy"
    # cfg4: the caller's whitening estimate, a per-bin reciprocal block-median baseline (NEXT-2)
    ib = None
    if w.red_noise:
        ib = torch.empty((S, N), dtype=torch.float32, device=dev)
        for s in range(S):
            ib[s:s + 1].copy_(inputs.block_median_inv_baseline(x[s:s + 1]))
    snr_g = torch.empty((S, N), dtype=torch.float32, device=dev)
    bh_g = torch.empty((S, N), dtype=torch.int32, device=dev)
    snr_p = torch.empty_like(snr_g) if do_p and do_g else snr_g
    bh_p = torch.empty_like(bh_g) if do_p and do_g else bh_g
    gv, fs, pv = _variants(args)
    mu_g, sg_g = inputs.exp1_stats(gv, H, fs)
    mu_p, sg_p = inputs.exp1_stats(pv, H)
    n_out = N // max(1, args.n_fund_div)                 # outputs per spectrum (hs_plan's n_fund; N in every quoted run)
    plan_g = hs.hs_plan(N, S, H, N, N, n_out, flags=args.greedy_flags, device=local)
    plan_p = hs.hs_plan(N, S, H, N, N, n_out, flags=args.presto_flags, device=local)
    hs.hs_plan_set_tuning(plan_g, args.tune_greedy)     # 0 = the library's choice (diagnostic knob)
    hs.hs_plan_set_tuning(plan_p, args.tune_presto)
    stream = torch.cuda.current_stream(dev)
    # NEXT-2: the statistics estimated on the device inside the step (two rejection rounds at 3 sigma over the
    # fundamentals / top bins [N/64, N/32), where every order exists), then per-spectrum statistics from device memory
    est = args.stats == "estimated" or (args.stats == "auto" and w.red_noise)
    n_clip, clip = 2, 3.0
    if est:
        dmu_g = torch.empty((S, H), dtype=torch.float32, device=dev); dsg_g = torch.empty_like(dmu_g)
        dmu_p = torch.empty_like(dmu_g); dsg_p = torch.empty_like(dmu_g)
        # the large workspace: the first gather pass stores its sums, the rejection rounds stream them (include/hs.h)
        work = torch.empty((hs.hs_stats_workspace_bytes_cached(plan_g, n_clip, N // 64, N // 32) + 7) // 8, dtype=torch.float64, device=dev)

    # the whitening pass writes y = x * inv_baseline once; the sums then read y alone (same bits, reading R13)
    wpass = ib is not None and args.whiten == "pass"
    y = torch.empty_like(x) if wpass else None

    def step(ev=None):
        if ev is not None:
            ev[0].record(stream)
        xin, bin_ = x, ib
        if wpass:
            hs.hs_whiten(plan_g, x, ib, y, stream.cuda_stream)
            xin, bin_ = y, None
        if ev is not None:
            ev[4].record(stream)
        if est:
            if do_g:
                hs.hs_estimate_stats(plan_g, True, xin, bin_, N // 64, N // 32, clip, n_clip, dmu_g, dsg_g, work, stream.cuda_stream)
            if do_p:
                hs.hs_estimate_stats(plan_p, False, xin, bin_, N // 64, N // 32, clip, n_clip, dmu_p, dsg_p, work, stream.cuda_stream)
        if ev is not None:
            ev[3].record(stream)
        if do_g:
            if est:
                hs.hs_run_greedy_dstats(plan_g, xin, bin_, dmu_g, dsg_g, snr_g, bh_g, None, stream.cuda_stream)
            else:
                hs.hs_run_greedy(plan_g, xin, bin_, mu_g, sg_g, snr_g, bh_g, None, stream.cuda_stream)
        if ev is not None:
            ev[1].record(stream)
        if do_p:
            if est:
                hs.hs_run_presto_dstats(plan_p, xin, bin_, dmu_p, dsg_p, snr_p, bh_p, stream.cuda_stream)
            else:
                hs.hs_run_presto(plan_p, xin, bin_, mu_p, sg_p, snr_p, bh_p, stream.cuda_stream)
        if ev is not None:
            ev[2].record(stream)

    for _ in range(args.warmup):
        step()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(args.steps)]
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    l0 = hs.hs_launch_count(plan_g) + hs.hs_launch_count(plan_p)
    barrier(world)
    for k in range(args.steps):
        step(evs[k])
    barrier(world)
    launches = hs.hs_launch_count(plan_g) + hs.hs_launch_count(plan_p) - l0
    kname = {"greedy": hs.hs_last_kernel(plan_g) if do_g else None, "presto": hs.hs_last_kernel(plan_p) if do_p else None}
    total_ms = evs[0][0].elapsed_time(evs[-1][2])          # device time of exactly K steps
    w_ms = sum(e[0].elapsed_time(e[4]) for e in evs) / args.steps
    s_ms = sum(e[4].elapsed_time(e[3]) for e in evs) / args.steps
    g_ms = sum(e[3].elapsed_time(e[1]) for e in evs) / args.steps
    p_ms = sum(e[1].elapsed_time(e[2]) for e in evs) / args.steps
    # clocks: keep the sampler running through a few more device-only steps so short runs still get samples
    if rank == 0:
        t_end = time.time() + 1.0
        while time.time() < t_end:
            step()
            torch.cuda.synchronize()
    clocks = sampler.stop() if rank == 0 else None

    from paper_2202_12817_b200.sharding import max_over_ranks
    total_ms = max_over_ranks(total_ms, dev)
    g_ms = max_over_ranks(g_ms, dev)
    p_ms = max_over_ranks(p_ms, dev)
    s_ms = max_over_ranks(s_ms, dev)
    w_ms = max_over_ranks(w_ms, dev)
    if wpass:                       # the whitening pass belongs to each form's 16 B/bin (x and the multiplier read once)
        g_ms += w_ms if do_g else 0.0
        p_ms += w_ms if (do_p and not do_g) else 0.0
    bins_step = float(S) * n_out * world
    n_forms = int(do_g) + int(do_p)
    default_run = (args.n_fund_div == 1 and args.forms == "both" and not args.greedy_flags and not args.presto_flags and ib is None
                   and not args.tune_greedy and not args.tune_presto and w.name == "cfg3" and S == w.n_spectra)
    value = bins_step * args.steps / (total_ms * 1e-3)

    # ---- end to end through the host-buffer entry points (pinned host memory, H2D + D2H timed) ----
    e2e = None
    if not args.no_e2e:
        hx = torch.empty((S, N), dtype=torch.float32, pin_memory=True)
        hx.copy_(x)
        hsnr = torch.empty((S, N), dtype=torch.float32, pin_memory=True)
        hbh = torch.empty((S, N), dtype=torch.int32, pin_memory=True)
        both = do_g and do_p and args.greedy_flags == 0 and args.presto_flags == 0
        hsnr2 = torch.empty((S, N), dtype=torch.float32, pin_memory=True) if both else None
        hbh2 = torch.empty((S, N), dtype=torch.int32, pin_memory=True) if both else None
        e_steps = max(1, min(args.steps, 5))

        hib = None
        if ib is not None:
            hib = torch.empty((S, N), dtype=torch.float32, pin_memory=True)
            hib.copy_(ib)

        def e2e_step():
            if both:            # one upload of the spectra, both forms computed from it
                hs.hs_run_both_host(plan_g, hx, hib, mu_g, sg_g, hsnr, hbh, None, mu_p, sg_p, hsnr2, hbh2)
                return
            if do_g:
                hs.hs_run_greedy_host(plan_g, hx, hib, mu_g, sg_g, hsnr, hbh, None)
            if do_p:
                hs.hs_run_presto_host(plan_p, hx, hib, mu_p, sg_p, hsnr, hbh)

        e2e_step()
        barrier(world)
        t0 = time.perf_counter()
        for _ in range(e_steps):
            e2e_step()
        barrier(world)
        dt = max_over_ranks(time.perf_counter() - t0, dev)
        e2e = {"value": bins_step * e_steps / dt, "unit": UNIT, "steps": e_steps,
               "h2d_bytes_per_step": (1 if both else n_forms) * S * N * 4 * (2 if ib is not None else 1),
               "d2h_bytes_per_step": n_forms * S * N * 8,
               "ms_per_step": 1e3 * dt / e_steps,
               "note": ("hs_run_both_host (one upload, both forms)" if both else "hs_run_greedy_host / hs_run_presto_host") +
                       ", pinned host buffers, per rank; PCIe-bound"}
        # the search as one call: one upload, both forms, the candidate lists compacted on the device, only they come back
        if both:
            cgh = torch.empty((1 << 20, 4), dtype=torch.int32, pin_memory=True)
            cph = torch.empty((1 << 20, 4), dtype=torch.int32, pin_memory=True)
            ncand = hs.hs_search_host(plan_g, hx, hib, mu_g, sg_g, mu_p, sg_p, 10.0, cgh, cph)
            barrier(world)
            t0 = time.perf_counter()
            for _ in range(e_steps):
                ncand = hs.hs_search_host(plan_g, hx, hib, mu_g, sg_g, mu_p, sg_p, 10.0, cgh, cph)
            barrier(world)
            dt = max_over_ranks(time.perf_counter() - t0, dev)
            e2e["candidates_only"] = {"value": bins_step * e_steps / dt, "unit": UNIT, "ms_per_step": 1e3 * dt / e_steps,
                                      "h2d_bytes_per_step": S * N * 4 * (2 if ib is not None else 1),
                                      "d2h_bytes_per_step": 16 * (min(ncand[0], 1 << 20) + min(ncand[1], 1 << 20)) + 16,
                                      "candidates": {"greedy": ncand[0], "presto": ncand[1], "threshold": 10.0},
                                      "note": "hs_search_host: the per-bin outputs stay on the device, the two candidate lists are the result read back"}
            del cgh, cph
        del hx, hsnr, hbh, hib, hsnr2, hbh2

    # ---- NEXT-3: candidate list of the greedy outputs (one streaming pass; outside the step) ----
    cand = None
    if do_g:
        T = 10.0
        cbuf = torch.empty((1 << 20, 4), dtype=torch.int32, device=dev)
        ccnt = torch.zeros((1,), dtype=torch.int64, device=dev)
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        hs.hs_find_candidates(plan_g, snr_g, bh_g, T, cbuf, ccnt, stream.cuda_stream)
        c0.record(stream)
        for _ in range(5):
            hs.hs_find_candidates(plan_g, snr_g, bh_g, T, cbuf, ccnt, stream.cuda_stream)
        c1.record(stream)
        torch.cuda.synchronize()
        c_ms = c0.elapsed_time(c1) / 5
        from paper_2202_12817_b200.sharding import sum_over_ranks
        cand = {"threshold": T, "count": int(ccnt.item()), "ms": c_ms, "read_gbs": S * N * 4 / (c_ms * 1e-3) / 1e9}
        # N > 1: the candidate lists are the only result that crosses ranks; here their total size
        cand["count_all_ranks"] = int(sum_over_ranks(cand["count"], dev))
        del cbuf

    # ---- roofline of the dominant kernel (HBM-bound: 12 algorithmic bytes per bin and launch) ----
    peak, peak_src = measured_peak()
    dom, dom_ms = ("greedy", g_ms) if (g_ms >= p_ms or not do_p) and do_g else ("presto", p_ms)
    alg_bytes = (BYTES_PER_BIN + (4.0 if ib is not None else 0.0)) * S * n_out

    def roof(ms):
        a = alg_bytes / (ms * 1e-3) / 1e9
        return a, a / peak

    ncu = _load_json(NCU_KERNELS_JSON)
    mm = _load_json(MACHINE_MODEL_JSON)
    full_cfg3 = (w.name == "cfg3" and S == w.n_spectra and H == w.H and ib is None and args.n_fund_div == 1
                 and not args.greedy_flags and not args.presto_flags)

    def evidence(form):
        """Committed ncu counters of the kernel that actually ran (cfg3 captures only); None when there are none."""
        rec = ncu.get(kname[form] or "", None) if full_cfg3 else None
        return rec if isinstance(rec, dict) else None

    def second(form, ms):
        """The on-chip ceiling beside the HBM one: L2 -> SM sector bytes of the launch over the measured L2 -> SM rate."""
        rec = evidence(form)
        l2 = mm.get("l2_to_sm_gbs")
        if rec is None or not l2 or not rec.get("l2_to_sm_sector_bytes"):
            return None
        floor_ms = rec["l2_to_sm_sector_bytes"] / (l2 * 1e9) * 1e3
        out = {"l2_to_sm_gbs": l2, "sector_bytes_per_launch": rec["l2_to_sm_sector_bytes"],
               "ceiling_ms": floor_ms, "frac_of_ceiling": floor_ms / ms, "source": mm.get("source"), "capture": rec.get("capture"),
               "reproducible_from_repository": mm.get("reproducible_from_repository", False)}
        if rec.get("access_form_ceiling_ms"):      # the measured rate of the kernel's own access form (L1 line requests included)
            out.update(access_form_ceiling_ms=rec["access_form_ceiling_ms"], frac_of_access_form_ceiling=rec["access_form_ceiling_ms"] / ms,
                       access_form_note=rec.get("access_form_note"))
        return out

    def per_kernel(form, ms):
        rec = evidence(form)
        return {"kernel": kname[form], "launch_ms": ms, "achieved": roof(ms)[0], "frac": roof(ms)[1],
                "gbins_per_s": S * N / ms / 1e6,
                "traffic": (rec["dram_bytes_read"] + rec["dram_bytes_write"]) if rec else None,
                "secondary_ceiling": second(form, ms)}

    a, fr = roof(dom_ms)
    dom_rec = evidence(dom)
    roofline = {"bound": "hbm", "kernel": dom, "kernel_name": kname[dom], "achieved": a, "peak": peak, "unit": "GB/s", "frac": fr,
                "traffic": (dom_rec["dram_bytes_read"] + dom_rec["dram_bytes_write"]) if dom_rec else None,
                "traffic_source": dom_rec.get("capture") if dom_rec else None, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": alg_bytes, "launch_ms": dom_ms,
                "secondary_ceiling": second(dom, dom_ms), "per_kernel": {}}
    if do_g:
        roofline["per_kernel"]["greedy"] = per_kernel("greedy", g_ms)
    if do_p:
        roofline["per_kernel"]["presto"] = per_kernel("presto", p_ms)

    # ---- extra (default run only, after the headline region): the other configurations of BASELINE.json / BASELINE.md,
    # measured in THIS run so that every fraction quoted there has a counterpart in the driver's record ----
    extra = None
    if default_run and world == 1 and not args.no_extra:
        def timed(fn, reps=3):
            fn()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(reps):
                fn()
            e1.record(stream)
            torch.cuda.synchronize()
            return e0.elapsed_time(e1) / reps

        def entry(plan, ms, bytes_per_bin=BYTES_PER_BIN):
            gbs = bytes_per_bin * S * N / (ms * 1e-3) / 1e9
            return {"kernel": hs.hs_last_kernel(plan), "launch_ms": ms, "achieved": gbs, "frac": gbs / peak, "gbins_per_s": S * N / ms / 1e6}

        extra = {"note": "same batch (cfg3 spectra), CUDA events, 1 warm-up + 3 launches each; frac = 12 B/bin over the same peak as the headline"}
        # sustained streaming rate of a product kernel (hs_whiten: two 4 GiB arrays read, one written, 12 B per element, 16-byte
        # accesses): a live second denominator beside the copy-burst peak of MEASURED_PEAKS.json, which these kernels can exceed
        wh_ms = timed(lambda: hs.hs_whiten(plan_g, x, snr_g, snr_p, stream.cuda_stream))
        stream_gbs = 12.0 * S * N / (wh_ms * 1e-3) / 1e9
        extra["stream"] = {"kernel": "hs_whiten_kernel", "launch_ms": wh_ms, "gbs": stream_gbs, "bytes_per_element": 12,
                           "note": "measured in this run (16-byte loads and stores)"}
        sweep = {}
        for Hs in (4, 8, 16):                       # paper Table 2's H values on the cfg3 shape
            pg, pp = hs.hs_plan(N, S, Hs, device=local), hs.hs_plan(N, S, Hs, device=local)
            mg, sgg = inputs.exp1_stats("greedy", Hs, True)
            mp, sgp = inputs.exp1_stats("presto", Hs)
            t_g = timed(lambda: hs.hs_run_greedy(pg, x, None, mg, sgg, snr_g, bh_g, None, stream.cuda_stream))
            t_p = timed(lambda: hs.hs_run_presto(pp, x, None, mp, sgp, snr_p, bh_p, stream.cuda_stream))
            sweep[f"H{Hs}"] = {"greedy": entry(pg, t_g), "presto": entry(pp, t_p)}
            hs.hs_destroy(pg); hs.hs_destroy(pp)
        extra["h_sweep"] = sweep
        for name, gflags, pflags in (("simple", 2, None), ("presto_all", None, 4), ("presto_plus", None, 12)):   # NEXT-1 variants, H = 32
            pl = hs.hs_plan(N, S, H, flags=(gflags if gflags is not None else pflags), device=local)
            if gflags is not None:
                m_, s_ = inputs.exp1_stats("simple", H, True)
                t = timed(lambda: hs.hs_run_greedy(pl, x, None, m_, s_, snr_g, bh_g, None, stream.cuda_stream))
            else:
                m_, s_ = inputs.exp1_stats(name, H)
                t = timed(lambda: hs.hs_run_presto(pl, x, None, m_, s_, snr_p, bh_p, stream.cuda_stream), reps=2)
            extra[name] = entry(pl, t)
            hs.hs_destroy(pl)
        # The copy-burst peak under-measures what HBM sustains on this pool: the H = 4 / 8 PRESTO launches above move
        # their 12 B/bin faster than it (frac > 1).  A fraction above 1 says the denominator is low, not that a kernel
        # beat the memory; so every fraction is also given against the highest rate any launch of THIS run sustained.
        best = max([stream_gbs] + [v[f]["achieved"] for v in sweep.values() for f in v])
        extra["stream"]["best_observed_gbs"] = best
        extra["stream"]["best_observed_note"] = "max over hs_whiten and the H sweep of algorithmic bytes / time in this run"
        for form in roofline["per_kernel"].values():
            form["frac_vs_best_observed"] = form["achieved"] / best
        roofline["frac_vs_best_observed"] = roofline["achieved"] / best

    cpu = None
    if rank == 0 and not args.no_cpu:
        rows = min(args.cpu_spectra, S)
        r = run_cpu_sample(x[:rows].cpu().numpy(), H, args=args, ib_host=None if ib is None else ib[:rows].cpu().numpy())
        cpu = {"value": r["bins"] / r["seconds"], "unit": UNIT, "cores": r["cores"], "kind": "oracle",
               "sample": f"first {rows} of {S} spectra of {w.name} ({rows}x{N} bins), greedy {r['greedy_s']:.2f} s + "
                         f"PRESTO {r['presto_s']:.2f} s, fp64"}
    hs.hs_destroy(plan_g)
    hs.hs_destroy(plan_p)
    if extra is not None:
        del x, snr_g, bh_g, snr_p, bh_p
        torch.cuda.empty_cache()
        # the paper's Table 2 shape (1024 spectra x 131 072 bins, pure noise), H = 32 / 16 / 8 / 4: context for
        # BASELINE.md's comparison table; 512 MiB of spectra, so partly L2-warm between launches (said in the entry)
        wp = inputs.workload("cfgP")
        Sp, Np = wp.n_spectra, wp.n_bins
        xp = torch.empty((Sp, Np), dtype=torch.float32, device=dev)
        for srow in range(Sp):
            xp[srow].copy_(inputs.generate_row(wp, srow, dev))
        o_s = torch.empty((Sp, Np), dtype=torch.float32, device=dev); o_b = torch.empty((Sp, Np), dtype=torch.int32, device=dev)
        cfgp = {"note": f"{Sp} x {Np} fp32 bins (paper's Table 2 shape), 1 warm-up + 3 launches, partly L2-warm; frac = 12 B/bin over the measured peak"}
        for Hs in (32, 16, 8, 4):
            pg, pp = hs.hs_plan(Np, Sp, Hs, device=local), hs.hs_plan(Np, Sp, Hs, device=local)
            mg, sgg = inputs.exp1_stats("greedy", Hs, True)
            mp, sgp = inputs.exp1_stats("presto", Hs)
            t_g = timed(lambda: hs.hs_run_greedy(pg, xp, None, mg, sgg, o_s, o_b, None, stream.cuda_stream))
            t_p = timed(lambda: hs.hs_run_presto(pp, xp, None, mp, sgp, o_s, o_b, stream.cuda_stream))
            cfgp[f"H{Hs}"] = {f: {"launch_ms": t, "gbins_per_s": Sp * Np / t / 1e6, "frac": 12.0 * Sp * Np / (t * 1e-3) / 1e9 / peak}
                              for f, t in (("greedy", t_g), ("presto", t_p))}
            hs.hs_destroy(pg); hs.hs_destroy(pp)
        extra["cfgP"] = cfgp
        del xp, o_s, o_b
        torch.cuda.empty_cache()
        extra["cfg4"] = child_line(["--workload", "cfg4", "--forms", "greedy", "--steps", "3", "--warmup", "1"],
                                   ("config", "ms_per_step", "value", "whiten", "stats", "roofline", "gpu_launches"))
        extra["cfg5"] = child_line(["--workload", "cfg5", "--steps", "3", "--warmup", "1"],
                                   ("config", "ms_per_step", "value", "roofline", "gpu_launches"))
    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": f"{w.name}: {S} spectra x {N} fp32 bins per GPU, H={H}, " +
                                       {"both": "greedy (Alg. 2) + PRESTO (Alg. 1) per step", "greedy": "greedy (Alg. 2) only",
                                        "presto": "PRESTO (Alg. 1) only"}[args.forms] +
                                       (f", stats/flags {gv}/{pv} ({args.greedy_flags}/{args.presto_flags})" if args.greedy_flags or args.presto_flags else "") +
                                       (", per-bin inverse baseline" if ib is not None else "") +
                                       (f", DIAGNOSTIC: outputs for n < N/{args.n_fund_div} only" if args.n_fund_div != 1 else ""),
                           "seed": w.seed, "n_pulsars": len(w.pulsars), "l2": f"inputs ({S * N * 4 / 2**30:.2f} GiB) exceed L2; no flush needed" if S * N * 4 > 256 * 2**20 else "inputs fit in L2: warm-L2 numbers",
                           "parallelism": f"spectra sharded over {world} GPU(s), no collective"},
                "whiten": ({"source": "hs_whiten pass inside the step; its time is counted in the form's launch_ms (16 B/bin)", "ms": w_ms} if wpass else None),
                "stats": ({"source": "hs_estimate_stats inside the step (reading R14): bins [N/64, N/32), 2 rejection rounds at 3 sigma "
                                     "(one gather pass, the rounds stream the stored sums), then hs_run_*_dstats", "ms": s_ms} if est else
                          {"source": "closed-form Exp(1) statistics passed by value", "ms": 0.0}),
                "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "candidates": cand,
                "cpu_baseline": cpu, "extra": extra}
        print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()
    return 0


def run_cuda_2d(args):
    """--workload cfg5 (BASELINE.json configs[4], NEXT-4): one f-fdot plane, 201 x 2^21 bins, H = 16; a step =
    hs_run_greedy_2d (the 2-D greedy rule of reading R15) + hs_run_presto_2d on the same plane.  1 GPU."""
    import torch
    from paper_2202_12817_b200 import binding as hs
    from paper_2202_12817_b200 import inputs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    hs.load()
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    w = inputs.plane_workload(args.workload)
    nz, N, H = w.n_z, w.n_bins, (args.H or w.H)
    P = inputs.generate_plane(w, dev)
    snr_g = torch.empty((nz, N), dtype=torch.float32, device=dev); bh_g = torch.empty((nz, N), dtype=torch.int32, device=dev)
    snr_p = torch.empty_like(snr_g); bh_p = torch.empty_like(bh_g)
    gv, fs, pv = _variants(args)
    mu_g, sg_g = inputs.exp1_stats("simple", H)
    mu_p, sg_p = inputs.exp1_stats(pv, H)
    plan_g = hs.hs_plan_2d(N, nz, H, flags=args.greedy_flags, device=0)
    plan_p = hs.hs_plan_2d(N, nz, H, flags=args.presto_flags, device=0)
    stream = torch.cuda.current_stream(dev)
    do_g, do_p = args.forms != "presto", args.forms != "greedy"

    def step(ev=None):
        if ev is not None:
            ev[0].record(stream)
        if do_g:
            hs.hs_run_greedy_2d(plan_g, P, mu_g, sg_g, snr_g, bh_g, None, stream.cuda_stream)
        if ev is not None:
            ev[1].record(stream)
        if do_p:
            hs.hs_run_presto_2d(plan_p, P, mu_p, sg_p, snr_p, bh_p, stream.cuda_stream)
        if ev is not None:
            ev[2].record(stream)

    for _ in range(args.warmup):
        step()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    sampler = ClockSampler(0)
    sampler.start()
    time.sleep(0.3)
    l0 = hs.hs_launch_count(plan_g) + hs.hs_launch_count(plan_p)
    torch.cuda.synchronize()
    for k in range(args.steps):
        step(evs[k])
    torch.cuda.synchronize()
    launches = hs.hs_launch_count(plan_g) + hs.hs_launch_count(plan_p) - l0
    total_ms = evs[0][0].elapsed_time(evs[-1][2])
    g_ms = sum(e[0].elapsed_time(e[1]) for e in evs) / args.steps
    p_ms = sum(e[1].elapsed_time(e[2]) for e in evs) / args.steps
    t_end = time.time() + 1.0
    while time.time() < t_end:
        step()
        torch.cuda.synchronize()
    clocks = sampler.stop()
    peak, peak_src = measured_peak()
    bins = float(nz) * N
    alg_bytes = BYTES_PER_BIN * bins

    def per_kernel(name, ms):
        a = alg_bytes / (ms * 1e-3) / 1e9
        return {"kernel": name, "launch_ms": ms, "achieved": a, "frac": a / peak, "gbins_per_s": bins / ms / 1e6, "traffic": None}

    pk = {}
    if do_g:
        pk["greedy_2d"] = per_kernel(hs.hs_last_kernel(plan_g), g_ms)
    if do_p:
        pk["presto_2d"] = per_kernel(hs.hs_last_kernel(plan_p), p_ms)
    dom = max(pk, key=lambda k: pk[k]["launch_ms"])
    cpu = None
    if not args.no_cpu:
        import oracle
        oracle.build()
        rows = (98, 102)                                   # z = -2 .. 1: rows where all 16 orders exist
        Ph = P.cpu().numpy()
        t0 = time.perf_counter()
        if do_g:
            oracle.greedy_2d(Ph, H, mu_g.numpy(), sg_g.numpy(), args.greedy_flags, rows=rows)
        if do_p:
            oracle.presto_2d(Ph, H, mu_p.numpy(), sg_p.numpy(), args.presto_flags, rows=rows)
        dt = time.perf_counter() - t0
        cpu = {"value": (rows[1] - rows[0]) * N / dt, "unit": UNIT, "cores": oracle.host_threads(), "kind": "oracle",
               "sample": f"rows z = -2 .. 1 of the plane (4 x {N} bins, all 16 orders evaluated), fp64"}
    hs.hs_destroy(plan_g); hs.hs_destroy(plan_p)
    line = {"metric": "2-D harmonic-sum plane bins/s at H=16 (greedy-2D + PRESTO-like-2D forms per bin)", "value": bins * args.steps / (total_ms * 1e-3),
            "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": total_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"{w.name}: one f-fdot plane, {nz} rows (z = -{(nz - 1) // 2}..{(nz - 1) // 2}) x {N} fp32 bins, H={H}, "
                                   f"{len(w.signals)} drifting signals; reading R15 (the 2-D greedy rule is this repository's, not the paper's)",
                       "seed": w.seed, "l2": f"plane ({nz * N * 4 / 2**30:.2f} GiB) exceeds L2; no flush needed"},
            "clocks": clocks, "e2e": None, "gpu_launches": int(launches),
            "roofline": {"bound": "hbm", "kernel": dom, "kernel_name": pk[dom]["kernel"], "achieved": pk[dom]["achieved"], "peak": peak,
                         "unit": "GB/s", "frac": pk[dom]["frac"], "traffic": None, "peak_source": peak_src,
                         "algorithmic_bytes_per_launch": alg_bytes, "launch_ms": pk[dom]["launch_ms"], "per_kernel": pk},
            "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)
    return 0


def main():
    args = parse_args()
    if args.workload == "cfg5":
        if args.impl == "reference" or args.gpus > 1:
            raise SystemExit("bench.py: --workload cfg5 (NEXT-4) is a 1-GPU, CUDA-arm workload")
        return run_cuda_2d(args)
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return respawn_under_torchrun(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
