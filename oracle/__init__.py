"""CPU oracle for the harmonic sum of arXiv 2202.12817 -- TEST INFRASTRUCTURE ONLY.

Thin ctypes loader around ``oracle/hs_oracle.cpp`` (double precision, written from the
paper; see the header of that file for citations, readings and pins).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs
may import this package.  It imports nothing from ``paper_2202_12817_b200`` and the CUDA
path imports nothing from here.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hs_oracle.cpp")
_LIB = os.path.join(_HERE, "libhs_oracle.so")

# Flag values as documented for the boundary (restated, not imported).
NO_FUND_SELECT = 1 << 0
NO_DRIFT = 1 << 1
ALL_HARMONICS = 1 << 2
ALL_ORDERS = 1 << 3

_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with g++ -O2 (no fast-math: plain IEEE double)."""
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-pthread", "-ffp-contract=off",
               "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        c_f = ctypes.POINTER(ctypes.c_float)
        c_d = ctypes.POINTER(ctypes.c_double)
        c_i32 = ctypes.POINTER(ctypes.c_int32)
        c_u32 = ctypes.POINTER(ctypes.c_uint32)
        c_i64 = ctypes.POINTER(ctypes.c_int64)
        i64, i32, u32 = ctypes.c_int64, ctypes.c_int32, ctypes.c_uint32
        lib.hs_oracle_greedy.argtypes = [c_f, c_f, i64, i32, i64, i32, c_f, c_f, u32, i64,
                                         c_d, c_i32, c_u32, i64, i32]
        lib.hs_oracle_presto.argtypes = [c_f, c_f, i64, i32, i64, i32, c_f, c_f, u32, i64,
                                         c_d, c_i32, i64, i32]
        lib.hs_oracle_greedy_bins.argtypes = [c_f, c_f, i64, i64, i32, c_f, c_f, u32, c_i64, c_i64, i64,
                                              c_d, c_i32, c_u32, c_d, c_i64]
        lib.hs_oracle_presto_bins.argtypes = [c_f, c_f, i64, i64, i32, c_f, c_f, u32, c_i64, c_i64, i64,
                                              c_d, c_i32, c_d]
        lib.hs_oracle_estimate_stats.argtypes = [c_f, c_f, i64, i32, i64, i32, u32, i32, i64, i64,
                                                 ctypes.c_double, i32, c_f, c_f, c_i64]
        lib.hs_oracle_greedy_2d.argtypes = [c_f, i64, i32, i64, i32, c_f, c_f, u32, c_d, c_i32, c_u32, i64, i32, i32, i32]
        lib.hs_oracle_presto_2d.argtypes = [c_f, i64, i32, i64, i32, c_f, c_f, u32, c_d, c_i32, i64, i32, i32, i32]
        lib.hs_oracle_2d_bins.argtypes = [c_f, i64, i32, i64, i32, c_f, c_f, u32, i32, c_i64, c_i64, i64, c_d, c_i32, c_d]
        lib.hs_oracle_round_half_up.argtypes = [i64, i64]
        lib.hs_oracle_round_half_up.restype = i64
        lib.hs_oracle_presto_index.argtypes = [i32, i32, i64]
        lib.hs_oracle_presto_index.restype = i64
        lib.hs_oracle_presto_order_in_set.argtypes = [i32, u32]
        lib.hs_oracle_presto_order_in_set.restype = i32
        lib.hs_oracle_hardware_threads.restype = i32
        _lib = lib
    return _lib


def _ptr(a: Optional[np.ndarray], ctype):
    if a is None:
        return ctypes.cast(None, ctypes.POINTER(ctype))
    return a.ctypes.data_as(ctypes.POINTER(ctype))


def _as_f32_2d(x) -> np.ndarray:
    a = np.asarray(x)
    if a.dtype != np.float32:
        raise TypeError("spectra must be float32 (the method's input precision)")
    if a.ndim == 1:
        a = a[None, :]
    if not a.flags.c_contiguous:
        a = np.ascontiguousarray(a)
    return a


def _stats(mu, sigma, H) -> Tuple[np.ndarray, np.ndarray]:
    mu = np.ascontiguousarray(np.asarray(mu, dtype=np.float32))
    sigma = np.ascontiguousarray(np.asarray(sigma, dtype=np.float32))
    if mu.shape != (H,) or sigma.shape != (H,):
        raise ValueError("mu and sigma must have length H")
    return mu, sigma


def host_threads() -> int:
    """Threads the oracle will use by default = cores this process may run on."""
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:  # pragma: no cover
        return int(_load().hs_oracle_hardware_threads())


def greedy(x, H: int, mu, sigma, flags: int = 0, inv_baseline=None, n_fund: Optional[int] = None,
           n_threads: Optional[int] = None, want_path: bool = True):
    """Alg. 2 over a batch.  Returns (snr float64 [S,n_fund], best_h int32, path uint32 or None)."""
    lib = _load()
    a = _as_f32_2d(x)
    S, N = a.shape
    nf = N if n_fund is None else int(n_fund)
    mu, sigma = _stats(mu, sigma, H)
    ib = None if inv_baseline is None else _as_f32_2d(inv_baseline)
    snr = np.empty((S, nf), dtype=np.float64)
    bh = np.empty((S, nf), dtype=np.int32)
    path = np.empty((S, nf), dtype=np.uint32) if want_path else None
    rc = lib.hs_oracle_greedy(_ptr(a, ctypes.c_float), _ptr(ib, ctypes.c_float), N, S, N, H,
                              _ptr(mu, ctypes.c_float), _ptr(sigma, ctypes.c_float), flags, nf,
                              _ptr(snr, ctypes.c_double), _ptr(bh, ctypes.c_int32), _ptr(path, ctypes.c_uint32),
                              nf, n_threads or host_threads())
    if rc != 0:
        raise ValueError("hs_oracle_greedy: invalid arguments")
    return snr, bh, path


def presto(x, H: int, mu, sigma, flags: int = 0, inv_baseline=None, n_fund: Optional[int] = None,
           n_threads: Optional[int] = None):
    """Alg. 1 family over a batch.  Returns (snr float64 [S,n_fund], best_h int32)."""
    lib = _load()
    a = _as_f32_2d(x)
    S, N = a.shape
    nf = N if n_fund is None else int(n_fund)
    mu, sigma = _stats(mu, sigma, H)
    ib = None if inv_baseline is None else _as_f32_2d(inv_baseline)
    snr = np.empty((S, nf), dtype=np.float64)
    bh = np.empty((S, nf), dtype=np.int32)
    rc = lib.hs_oracle_presto(_ptr(a, ctypes.c_float), _ptr(ib, ctypes.c_float), N, S, N, H,
                              _ptr(mu, ctypes.c_float), _ptr(sigma, ctypes.c_float), flags, nf,
                              _ptr(snr, ctypes.c_double), _ptr(bh, ctypes.c_int32), nf,
                              n_threads or host_threads())
    if rc != 0:
        raise ValueError("hs_oracle_presto: invalid arguments")
    return snr, bh


def greedy_bins(x, H: int, mu, sigma, rows, bins, flags: int = 0, inv_baseline=None):
    """Alg. 2 for selected (row, bin) pairs, with per-order detail.

    Returns dict(snr, best_h, path, snr_h [count,H] (NaN = order not evaluated), bin_h [count,H])."""
    lib = _load()
    a = _as_f32_2d(x)
    S, N = a.shape
    mu, sigma = _stats(mu, sigma, H)
    ib = None if inv_baseline is None else _as_f32_2d(inv_baseline)
    rows = np.ascontiguousarray(np.asarray(rows, dtype=np.int64))
    bins = np.ascontiguousarray(np.asarray(bins, dtype=np.int64))
    if rows.shape != bins.shape or (rows.size and (rows.min() < 0 or rows.max() >= S)):
        raise ValueError("rows/bins")
    c = rows.size
    snr = np.empty(c, np.float64); bh = np.empty(c, np.int32); path = np.empty(c, np.uint32)
    snr_h = np.empty((c, H), np.float64); bin_h = np.empty((c, H), np.int64)
    rc = lib.hs_oracle_greedy_bins(_ptr(a, ctypes.c_float), _ptr(ib, ctypes.c_float), N, N, H,
                                   _ptr(mu, ctypes.c_float), _ptr(sigma, ctypes.c_float), flags,
                                   _ptr(rows, ctypes.c_int64), _ptr(bins, ctypes.c_int64), c,
                                   _ptr(snr, ctypes.c_double), _ptr(bh, ctypes.c_int32), _ptr(path, ctypes.c_uint32),
                                   _ptr(snr_h, ctypes.c_double), _ptr(bin_h, ctypes.c_int64))
    if rc != 0:
        raise ValueError("hs_oracle_greedy_bins: invalid arguments")
    return dict(snr=snr, best_h=bh, path=path, snr_h=snr_h, bin_h=bin_h)


def presto_bins(x, H: int, mu, sigma, rows, bins, flags: int = 0, inv_baseline=None):
    """Alg. 1 family for selected (row, top bin) pairs.  Returns dict(snr, best_h, snr_h [count,H])."""
    lib = _load()
    a = _as_f32_2d(x)
    S, N = a.shape
    mu, sigma = _stats(mu, sigma, H)
    ib = None if inv_baseline is None else _as_f32_2d(inv_baseline)
    rows = np.ascontiguousarray(np.asarray(rows, dtype=np.int64))
    bins = np.ascontiguousarray(np.asarray(bins, dtype=np.int64))
    if rows.shape != bins.shape or (rows.size and (rows.min() < 0 or rows.max() >= S)):
        raise ValueError("rows/bins")
    c = rows.size
    snr = np.empty(c, np.float64); bh = np.empty(c, np.int32)
    snr_h = np.empty((c, H), np.float64)
    rc = lib.hs_oracle_presto_bins(_ptr(a, ctypes.c_float), _ptr(ib, ctypes.c_float), N, N, H,
                                   _ptr(mu, ctypes.c_float), _ptr(sigma, ctypes.c_float), flags,
                                   _ptr(rows, ctypes.c_int64), _ptr(bins, ctypes.c_int64), c,
                                   _ptr(snr, ctypes.c_double), _ptr(bh, ctypes.c_int32), _ptr(snr_h, ctypes.c_double))
    if rc != 0:
        raise ValueError("hs_oracle_presto_bins: invalid arguments")
    return dict(snr=snr, best_h=bh, snr_h=snr_h)


def estimate_stats(x, H: int, flags: int = 0, greedy: bool = True, n_lo: int = 0, n_hi: Optional[int] = None,
                   clip: float = 3.0, n_clip: int = 0, inv_baseline=None):
    """Reading R14 of GetMeanStdev(): per spectrum and order h, mean and standard deviation
    over n in [n_lo, n_hi) of the variant's partial sum S_h(n), with n_clip rounds of outlier rejection at
    mean +/- clip * std.  Returns (mu [S,H] float32, sigma [S,H] float32, count [S,H] int64)."""
    lib = _load()
    a = _as_f32_2d(x)
    S, N = a.shape
    ib = None if inv_baseline is None else _as_f32_2d(inv_baseline)
    n_hi = N if n_hi is None else n_hi
    mu = np.empty((S, H), np.float32); sg = np.empty((S, H), np.float32); cnt = np.empty((S, H), np.int64)
    rc = lib.hs_oracle_estimate_stats(_ptr(a, ctypes.c_float), _ptr(ib, ctypes.c_float), N, S, N, H, flags,
                                      1 if greedy else 0, n_lo, n_hi, float(clip), n_clip,
                                      _ptr(mu, ctypes.c_float), _ptr(sg, ctypes.c_float), _ptr(cnt, ctypes.c_int64))
    if rc != 0:
        raise ValueError("hs_oracle_estimate_stats: invalid arguments")
    return mu, sg, cnt


def greedy_2d(plane, H: int, mu, sigma, flags: int = 0, n_threads: Optional[int] = None, rows: Optional[Tuple[int, int]] = None):
    """R15: 2-D greedy (ours) / simple (NO_DRIFT) harmonic sum over a plane [n_z, N], n_z = 2 Z + 1.
    Returns (snr float64, best_h int32, path uint32: bits 0-15 r-shifts, bits 16-31 z-shifts), each [n_z, N];
    with rows = (lo, hi) only the rows lo <= z + Z < hi are computed (the others are left as NaN / 0)."""
    lib = _load()
    a = _as_f32_2d(plane)
    nz, N = a.shape
    mu, sigma = _stats(mu, sigma, H)
    lo, hi = rows if rows is not None else (0, nz)
    snr = np.full((nz, N), np.nan, np.float64); bh = np.zeros((nz, N), np.int32); path = np.zeros((nz, N), np.uint32)
    rc = lib.hs_oracle_greedy_2d(_ptr(a, ctypes.c_float), N, nz, N, H, _ptr(mu, ctypes.c_float), _ptr(sigma, ctypes.c_float), flags,
                                 _ptr(snr, ctypes.c_double), _ptr(bh, ctypes.c_int32), _ptr(path, ctypes.c_uint32), N,
                                 n_threads or host_threads(), lo, hi)
    if rc != 0:
        raise ValueError("hs_oracle_greedy_2d: invalid arguments")
    return snr, bh, path


def bins_2d(plane, H: int, mu, sigma, zi, r, flags: int = 0, greedy: bool = True):
    """R15 for selected (row zi = z + Z, column r) pairs.  Returns dict(snr, best_h, snr_h [count, H]); snr_h is NaN for
    the orders that were not evaluated."""
    lib = _load()
    a = _as_f32_2d(plane)
    nz, N = a.shape
    mu, sigma = _stats(mu, sigma, H)
    zi = np.ascontiguousarray(np.asarray(zi, dtype=np.int64)); r = np.ascontiguousarray(np.asarray(r, dtype=np.int64))
    if zi.shape != r.shape:
        raise ValueError("zi/r")
    c = zi.size
    snr = np.empty(c, np.float64); bh = np.empty(c, np.int32); snr_h = np.empty((c, H), np.float64)
    rc = lib.hs_oracle_2d_bins(_ptr(a, ctypes.c_float), N, nz, N, H, _ptr(mu, ctypes.c_float), _ptr(sigma, ctypes.c_float), flags,
                               1 if greedy else 0, _ptr(zi, ctypes.c_int64), _ptr(r, ctypes.c_int64), c,
                               _ptr(snr, ctypes.c_double), _ptr(bh, ctypes.c_int32), _ptr(snr_h, ctypes.c_double))
    if rc != 0:
        raise ValueError("hs_oracle_2d_bins: invalid arguments")
    return dict(snr=snr, best_h=bh, snr_h=snr_h)


def presto_2d(plane, H: int, mu, sigma, flags: int = 0, n_threads: Optional[int] = None, rows: Optional[Tuple[int, int]] = None):
    """R15: PRESTO-like 2-D harmonic sum, output indexed by the top harmonic (r, z).  Returns (snr, best_h)."""
    lib = _load()
    a = _as_f32_2d(plane)
    nz, N = a.shape
    mu, sigma = _stats(mu, sigma, H)
    lo, hi = rows if rows is not None else (0, nz)
    snr = np.full((nz, N), np.nan, np.float64); bh = np.zeros((nz, N), np.int32)
    rc = lib.hs_oracle_presto_2d(_ptr(a, ctypes.c_float), N, nz, N, H, _ptr(mu, ctypes.c_float), _ptr(sigma, ctypes.c_float), flags,
                                 _ptr(snr, ctypes.c_double), _ptr(bh, ctypes.c_int32), N, n_threads or host_threads(), lo, hi)
    if rc != 0:
        raise ValueError("hs_oracle_presto_2d: invalid arguments")
    return snr, bh


def round_half_up(a: int, b: int) -> int:
    """Round(a / b), b > 0, as the 2-D oracle computes it (half up, also for negative a)."""
    return int(_load().hs_oracle_round_half_up(a, b))


def presto_index(h: int, Hp: int, n: int) -> int:
    """Round(h/H' * n) as the oracle computes it (R3)."""
    return int(_load().hs_oracle_presto_index(h, Hp, n))


def presto_orders(H: int, flags: int = 0):
    """ORDERS(H): the H' values Alg. 1's outer loop visits."""
    lib = _load()
    return [Hp for Hp in range(1, H + 1) if lib.hs_oracle_presto_order_in_set(Hp, flags)]


def candidates(snr, best_h, threshold: float):
    """Reading R11: every (spectrum, bin) with snr >= threshold, with its best_h, sorted by
    (spectrum, bin).  Returns an int64 array [k, 3] (spectrum, bin, best_h) and the float64 snr values [k]."""
    snr = np.asarray(snr)
    rows, bins = np.nonzero(snr >= threshold)          # row-major order = sorted by (spectrum, bin); NaN never qualifies
    return np.stack([rows, bins, np.asarray(best_h)[rows, bins]], axis=1).astype(np.int64), snr[rows, bins].astype(np.float64)
