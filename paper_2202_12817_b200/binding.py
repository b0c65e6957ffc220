"""Thin Python binding of the C-ABI library declared in ``include/hs.h``.

Same names as the C entry points; argument marshalling only (tensor -> pointer, sequence ->
``float[H]``).  Every step of the method runs inside ``libhs_b200.so``; PyTorch supplies device
memory and streams.  There is NO fallback: if the library is missing or a call fails, an
exception is raised.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import torch

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libhs_b200.so")

HS_OK, HS_ERR_INVALID_ARG, HS_ERR_UNSUPPORTED, HS_ERR_ALLOC, HS_ERR_CUDA, HS_ERR_TOO_LARGE = range(6)
HS_STATIC_STATS_MAX_ROWS = 4096      # hs_estimate_stats_static: (n_clip + 1) * n_spectra may not exceed this

HS_GREEDY_NO_FUND_SELECT = 1 << 0
HS_GREEDY_NO_DRIFT = 1 << 1
HS_PRESTO_ALL_HARMONICS = 1 << 2
HS_PRESTO_ALL_ORDERS = 1 << 3
HS_TUNE_GENERIC = 255        # hs_plan_set_tuning: the coverage kernels

EXPORTS = ["hs_plan", "hs_run_greedy", "hs_run_presto", "hs_run_greedy_host", "hs_run_presto_host", "hs_run_both_host",
           "hs_find_candidates", "hs_plan_set_tuning", "hs_plan_set_host_slot_bytes",
           "hs_plan_2d", "hs_run_greedy_2d", "hs_run_presto_2d", "hs_run_greedy_dstats", "hs_run_presto_dstats", "hs_estimate_stats", "hs_estimate_stats_static", "hs_stats_workspace_bytes", "hs_stats_workspace_bytes_cached", "hs_whiten", "hs_search_host",
           "hs_launch_count", "hs_last_kernel", "hs_destroy", "hs_status_string", "hs_last_cuda_error"]


class HsError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = _lib.hs_status_string(status).decode() if _lib is not None else str(status)
        if status == HS_ERR_CUDA and _lib is not None:
            msg += f" [cudaError {_lib.hs_last_cuda_error()}]"
        super().__init__(f"{where}: {msg}")


_lib = None


def load() -> ctypes.CDLL:
    """Load libhs_b200.so (built by ``__graft_entry__.build()`` / ``_build.build()``)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2202_12817_b200._build` "
                           "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i64, i32, u32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_uint32
    fp = ctypes.POINTER(ctypes.c_float)
    lib.hs_plan.argtypes = [ctypes.POINTER(vp), i64, i32, i32, i64, i64, i64, u32, i32]
    lib.hs_plan.restype = ctypes.c_int
    lib.hs_run_greedy.argtypes = [vp, vp, vp, fp, fp, vp, vp, vp, vp]
    lib.hs_run_greedy.restype = ctypes.c_int
    lib.hs_run_presto.argtypes = [vp, vp, vp, fp, fp, vp, vp, vp]
    lib.hs_run_presto.restype = ctypes.c_int
    lib.hs_run_greedy_host.argtypes = [vp, vp, vp, fp, fp, vp, vp, vp]
    lib.hs_run_greedy_host.restype = ctypes.c_int
    lib.hs_run_presto_host.argtypes = [vp, vp, vp, fp, fp, vp, vp]
    lib.hs_run_presto_host.restype = ctypes.c_int
    lib.hs_run_both_host.argtypes = [vp, vp, vp, fp, fp, vp, vp, vp, fp, fp, vp, vp]
    lib.hs_run_both_host.restype = ctypes.c_int
    lib.hs_plan_set_tuning.argtypes = [vp, u32]
    lib.hs_plan_set_tuning.restype = ctypes.c_int
    lib.hs_plan_set_host_slot_bytes.argtypes = [vp, i64]
    lib.hs_plan_set_host_slot_bytes.restype = ctypes.c_int
    lib.hs_find_candidates.argtypes = [vp, vp, vp, ctypes.c_float, vp, i64, vp, vp]
    lib.hs_find_candidates.restype = ctypes.c_int
    lib.hs_plan_2d.argtypes = [ctypes.POINTER(vp), i64, i32, i32, i64, i64, u32, i32]
    lib.hs_plan_2d.restype = ctypes.c_int
    lib.hs_run_greedy_2d.argtypes = [vp, vp, fp, fp, vp, vp, vp, vp]
    lib.hs_run_greedy_2d.restype = ctypes.c_int
    lib.hs_run_presto_2d.argtypes = [vp, vp, fp, fp, vp, vp, vp]
    lib.hs_run_presto_2d.restype = ctypes.c_int
    lib.hs_run_greedy_dstats.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.hs_run_greedy_dstats.restype = ctypes.c_int
    lib.hs_run_presto_dstats.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp]
    lib.hs_run_presto_dstats.restype = ctypes.c_int
    lib.hs_estimate_stats.argtypes = [vp, i32, vp, vp, i64, i64, ctypes.c_float, i32, vp, vp, vp, i64, vp]
    lib.hs_estimate_stats.restype = ctypes.c_int
    lib.hs_estimate_stats_static.argtypes = [vp, i32, vp, vp, i64, i64, ctypes.c_float, i32, vp, vp, vp]
    lib.hs_estimate_stats_static.restype = ctypes.c_int
    lib.hs_search_host.argtypes = [vp, vp, vp, fp, fp, fp, fp, ctypes.c_float, vp, i64, vp, vp, i64, vp]
    lib.hs_search_host.restype = ctypes.c_int
    lib.hs_whiten.argtypes = [vp, vp, vp, vp, vp]
    lib.hs_whiten.restype = ctypes.c_int
    lib.hs_stats_workspace_bytes.argtypes = [vp, i32]
    lib.hs_stats_workspace_bytes.restype = i64
    lib.hs_stats_workspace_bytes_cached.argtypes = [vp, i32, i64, i64]
    lib.hs_stats_workspace_bytes_cached.restype = i64
    lib.hs_launch_count.argtypes = [vp]
    lib.hs_launch_count.restype = i64
    lib.hs_last_kernel.argtypes = [vp]
    lib.hs_last_kernel.restype = ctypes.c_char_p
    lib.hs_destroy.argtypes = [vp]
    lib.hs_destroy.restype = ctypes.c_int
    lib.hs_status_string.argtypes = [ctypes.c_int]
    lib.hs_status_string.restype = ctypes.c_char_p
    lib.hs_last_cuda_error.argtypes = []
    lib.hs_last_cuda_error.restype = i32
    _lib = lib
    return lib


def _check(rc: int, where: str) -> None:
    if rc != HS_OK:
        raise HsError(rc, where)


def _farr(v: Sequence[float]):
    vals = [float(t) for t in (v.tolist() if hasattr(v, "tolist") else v)]
    return (ctypes.c_float * len(vals))(*vals)


def _dptr(t: Optional[torch.Tensor], dtype, name: str) -> Optional[int]:
    if t is None:
        return None
    if not t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous CUDA tensor of {dtype}")
    return t.data_ptr()


def _hptr(t, dtype, name: str) -> Optional[int]:
    if t is None:
        return None
    if isinstance(t, torch.Tensor):
        if t.is_cuda or t.dtype != dtype or not t.is_contiguous():
            raise TypeError(f"{name}: expected a contiguous CPU tensor of {dtype}")
        return t.data_ptr()
    raise TypeError(f"{name}: expected a CPU torch tensor")


def hs_plan(n_bins: int, n_spectra: int, H: int, in_stride: int = 0, out_stride: int = 0, n_fund: int = 0,
            flags: int = 0, device: int = 0) -> ctypes.c_void_p:
    lib = load()
    plan = ctypes.c_void_p()
    _check(lib.hs_plan(ctypes.byref(plan), n_bins, n_spectra, H, in_stride, out_stride, n_fund, flags, device), "hs_plan")
    return plan


def hs_run_greedy(plan, d_spectra: torch.Tensor, d_inv_baseline: Optional[torch.Tensor], mu, sigma,
                  d_snr: torch.Tensor, d_best_h: torch.Tensor, d_path: Optional[torch.Tensor] = None,
                  stream: Optional[int] = None) -> None:
    lib = load()
    if stream is None:
        stream = torch.cuda.current_stream(d_spectra.device).cuda_stream
    _check(lib.hs_run_greedy(plan, _dptr(d_spectra, torch.float32, "d_spectra"),
                             _dptr(d_inv_baseline, torch.float32, "d_inv_baseline"), _farr(mu), _farr(sigma),
                             _dptr(d_snr, torch.float32, "d_snr"), _dptr(d_best_h, torch.int32, "d_best_h"),
                             _dptr(d_path, torch.int32, "d_path"),   # uint32 bit masks held in an int32 tensor
                             stream), "hs_run_greedy")


def hs_run_presto(plan, d_spectra: torch.Tensor, d_inv_baseline: Optional[torch.Tensor], mu, sigma,
                  d_snr: torch.Tensor, d_best_h: torch.Tensor, stream: Optional[int] = None) -> None:
    lib = load()
    if stream is None:
        stream = torch.cuda.current_stream(d_spectra.device).cuda_stream
    _check(lib.hs_run_presto(plan, _dptr(d_spectra, torch.float32, "d_spectra"),
                             _dptr(d_inv_baseline, torch.float32, "d_inv_baseline"), _farr(mu), _farr(sigma),
                             _dptr(d_snr, torch.float32, "d_snr"), _dptr(d_best_h, torch.int32, "d_best_h"),
                             stream), "hs_run_presto")


def hs_plan_2d(n_bins: int, n_z: int, H: int, in_stride: int = 0, out_stride: int = 0, flags: int = 0, device: int = 0) -> ctypes.c_void_p:
    lib = load()
    plan = ctypes.c_void_p()
    _check(lib.hs_plan_2d(ctypes.byref(plan), n_bins, n_z, H, in_stride, out_stride, flags, device), "hs_plan_2d")
    return plan


def hs_run_greedy_2d(plan, d_plane: torch.Tensor, mu, sigma, d_snr: torch.Tensor, d_best_h: torch.Tensor,
                     d_path: Optional[torch.Tensor] = None, stream: Optional[int] = None) -> None:
    lib = load()
    if stream is None:
        stream = torch.cuda.current_stream(d_plane.device).cuda_stream
    _check(lib.hs_run_greedy_2d(plan, _dptr(d_plane, torch.float32, "d_plane"), _farr(mu), _farr(sigma),
                                _dptr(d_snr, torch.float32, "d_snr"), _dptr(d_best_h, torch.int32, "d_best_h"),
                                _dptr(d_path, torch.int32, "d_path"), stream), "hs_run_greedy_2d")


def hs_run_presto_2d(plan, d_plane: torch.Tensor, mu, sigma, d_snr: torch.Tensor, d_best_h: torch.Tensor,
                     stream: Optional[int] = None) -> None:
    lib = load()
    if stream is None:
        stream = torch.cuda.current_stream(d_plane.device).cuda_stream
    _check(lib.hs_run_presto_2d(plan, _dptr(d_plane, torch.float32, "d_plane"), _farr(mu), _farr(sigma),
                                _dptr(d_snr, torch.float32, "d_snr"), _dptr(d_best_h, torch.int32, "d_best_h"), stream),
           "hs_run_presto_2d")


def hs_run_greedy_dstats(plan, d_spectra: torch.Tensor, d_inv_baseline: Optional[torch.Tensor], d_mu: torch.Tensor,
                         d_sigma: torch.Tensor, d_snr: torch.Tensor, d_best_h: torch.Tensor,
                         d_path: Optional[torch.Tensor] = None, stream: Optional[int] = None) -> None:
    lib = load()
    if stream is None:
        stream = torch.cuda.current_stream(d_spectra.device).cuda_stream
    _check(lib.hs_run_greedy_dstats(plan, _dptr(d_spectra, torch.float32, "d_spectra"),
                                    _dptr(d_inv_baseline, torch.float32, "d_inv_baseline"),
                                    _dptr(d_mu, torch.float32, "d_mu"), _dptr(d_sigma, torch.float32, "d_sigma"),
                                    _dptr(d_snr, torch.float32, "d_snr"), _dptr(d_best_h, torch.int32, "d_best_h"),
                                    _dptr(d_path, torch.int32, "d_path"), stream), "hs_run_greedy_dstats")


def hs_run_presto_dstats(plan, d_spectra: torch.Tensor, d_inv_baseline: Optional[torch.Tensor], d_mu: torch.Tensor,
                         d_sigma: torch.Tensor, d_snr: torch.Tensor, d_best_h: torch.Tensor,
                         stream: Optional[int] = None) -> None:
    lib = load()
    if stream is None:
        stream = torch.cuda.current_stream(d_spectra.device).cuda_stream
    _check(lib.hs_run_presto_dstats(plan, _dptr(d_spectra, torch.float32, "d_spectra"),
                                    _dptr(d_inv_baseline, torch.float32, "d_inv_baseline"),
                                    _dptr(d_mu, torch.float32, "d_mu"), _dptr(d_sigma, torch.float32, "d_sigma"),
                                    _dptr(d_snr, torch.float32, "d_snr"), _dptr(d_best_h, torch.int32, "d_best_h"),
                                    stream), "hs_run_presto_dstats")


def hs_whiten(plan, d_spectra: torch.Tensor, d_inv_baseline: torch.Tensor, d_whitened: torch.Tensor, stream: Optional[int] = None) -> None:
    lib = load()
    if stream is None:
        stream = torch.cuda.current_stream(d_spectra.device).cuda_stream
    _check(lib.hs_whiten(plan, _dptr(d_spectra, torch.float32, "d_spectra"), _dptr(d_inv_baseline, torch.float32, "d_inv_baseline"),
                         _dptr(d_whitened, torch.float32, "d_whitened"), stream), "hs_whiten")


def hs_search_host(plan, h_spectra, h_inv_baseline, mu_greedy, sigma_greedy, mu_presto, sigma_presto, threshold: float,
                   h_cand_greedy: torch.Tensor, h_cand_presto: torch.Tensor):
    """h_cand_*: CPU int32 tensors [capacity, 4] (spectrum, bin, snr bits, best_h).  Returns (count_greedy, count_presto)."""
    lib = load()
    cg, cp = ctypes.c_uint64(0), ctypes.c_uint64(0)
    _check(lib.hs_search_host(plan, _hptr(h_spectra, torch.float32, "h_spectra"), _hptr(h_inv_baseline, torch.float32, "h_inv_baseline"),
                              _farr(mu_greedy), _farr(sigma_greedy), _farr(mu_presto), _farr(sigma_presto), threshold,
                              _hptr(h_cand_greedy, torch.int32, "h_cand_greedy"), h_cand_greedy.shape[0], ctypes.byref(cg),
                              _hptr(h_cand_presto, torch.int32, "h_cand_presto"), h_cand_presto.shape[0], ctypes.byref(cp)),
           "hs_search_host")
    return int(cg.value), int(cp.value)


def hs_stats_workspace_bytes(plan, n_clip: int) -> int:
    return int(load().hs_stats_workspace_bytes(plan, n_clip))


def hs_stats_workspace_bytes_cached(plan, n_clip: int, n_lo: int, n_hi: int) -> int:
    return int(load().hs_stats_workspace_bytes_cached(plan, n_clip, n_lo, n_hi))


def hs_estimate_stats(plan, greedy: bool, d_spectra: torch.Tensor, d_inv_baseline: Optional[torch.Tensor],
                      n_lo: int, n_hi: int, clip_sigma: float, n_clip: int, d_mu: torch.Tensor, d_sigma: torch.Tensor,
                      d_work: torch.Tensor, stream: Optional[int] = None) -> None:
    lib = load()
    if stream is None:
        stream = torch.cuda.current_stream(d_spectra.device).cuda_stream
    if not d_work.is_cuda or not d_work.is_contiguous():
        raise TypeError("d_work: expected a contiguous CUDA tensor")
    _check(lib.hs_estimate_stats(plan, 1 if greedy else 0, _dptr(d_spectra, torch.float32, "d_spectra"),
                                 _dptr(d_inv_baseline, torch.float32, "d_inv_baseline"), n_lo, n_hi, clip_sigma, n_clip,
                                 _dptr(d_mu, torch.float32, "d_mu"), _dptr(d_sigma, torch.float32, "d_sigma"),
                                 d_work.data_ptr(), d_work.numel() * d_work.element_size(), stream), "hs_estimate_stats")


def hs_estimate_stats_static(plan, greedy: bool, d_spectra: torch.Tensor, d_inv_baseline: Optional[torch.Tensor],
                             n_lo: int, n_hi: int, clip_sigma: float, n_clip: int, d_mu: torch.Tensor, d_sigma: torch.Tensor,
                             stream: Optional[int] = None) -> None:
    """hs_estimate_stats without a workspace argument, for callers that must not allocate device memory (a pipeline
    with a frozen memory layout, a plug-in that is handed only its inputs and outputs): the accumulators sit in a
    3 MiB array inside the library.  (n_clip + 1) * n_spectra <= HS_STATIC_STATS_MAX_ROWS, else HsError with status
    HS_ERR_TOO_LARGE.  One array per device: calls that overlap on the GPU race; make the first call on a device
    before any stream capture (include/hs.h)."""
    lib = load()
    if stream is None:
        stream = torch.cuda.current_stream(d_spectra.device).cuda_stream
    _check(lib.hs_estimate_stats_static(plan, 1 if greedy else 0, _dptr(d_spectra, torch.float32, "d_spectra"),
                                        _dptr(d_inv_baseline, torch.float32, "d_inv_baseline"), n_lo, n_hi, clip_sigma, n_clip,
                                        _dptr(d_mu, torch.float32, "d_mu"), _dptr(d_sigma, torch.float32, "d_sigma"), stream),
           "hs_estimate_stats_static")


def hs_run_greedy_host(plan, h_spectra, h_inv_baseline, mu, sigma, h_snr, h_best_h, h_path=None) -> None:
    lib = load()
    _check(lib.hs_run_greedy_host(plan, _hptr(h_spectra, torch.float32, "h_spectra"),
                                  _hptr(h_inv_baseline, torch.float32, "h_inv_baseline"), _farr(mu), _farr(sigma),
                                  _hptr(h_snr, torch.float32, "h_snr"), _hptr(h_best_h, torch.int32, "h_best_h"),
                                  _hptr(h_path, torch.int32, "h_path")), "hs_run_greedy_host")


def hs_run_presto_host(plan, h_spectra, h_inv_baseline, mu, sigma, h_snr, h_best_h) -> None:
    lib = load()
    _check(lib.hs_run_presto_host(plan, _hptr(h_spectra, torch.float32, "h_spectra"),
                                  _hptr(h_inv_baseline, torch.float32, "h_inv_baseline"), _farr(mu), _farr(sigma),
                                  _hptr(h_snr, torch.float32, "h_snr"), _hptr(h_best_h, torch.int32, "h_best_h")),
           "hs_run_presto_host")


def hs_run_both_host(plan, h_spectra, h_inv_baseline, mu_greedy, sigma_greedy, h_snr_greedy, h_best_h_greedy, h_path,
                     mu_presto, sigma_presto, h_snr_presto, h_best_h_presto) -> None:
    lib = load()
    _check(lib.hs_run_both_host(plan, _hptr(h_spectra, torch.float32, "h_spectra"),
                                _hptr(h_inv_baseline, torch.float32, "h_inv_baseline"),
                                _farr(mu_greedy), _farr(sigma_greedy),
                                _hptr(h_snr_greedy, torch.float32, "h_snr_greedy"),
                                _hptr(h_best_h_greedy, torch.int32, "h_best_h_greedy"), _hptr(h_path, torch.int32, "h_path"),
                                _farr(mu_presto), _farr(sigma_presto),
                                _hptr(h_snr_presto, torch.float32, "h_snr_presto"),
                                _hptr(h_best_h_presto, torch.int32, "h_best_h_presto")), "hs_run_both_host")


def hs_find_candidates(plan, d_snr: torch.Tensor, d_best_h: torch.Tensor, threshold: float,
                       d_out: Optional[torch.Tensor], d_count: torch.Tensor, stream: Optional[int] = None) -> None:
    """d_out: int32 CUDA tensor [capacity, 4] (rows = hs_candidate: spectrum, bin, snr bits, best_h) or None;
    d_count: int64 CUDA tensor with one element (uint64 count)."""
    lib = load()
    if stream is None:
        stream = torch.cuda.current_stream(d_snr.device).cuda_stream
    cap = 0 if d_out is None else int(d_out.shape[0])
    if d_out is not None and (d_out.ndim != 2 or d_out.shape[1] != 4):
        raise TypeError("d_out: expected an int32 tensor of shape [capacity, 4]")
    _check(lib.hs_find_candidates(plan, _dptr(d_snr, torch.float32, "d_snr"), _dptr(d_best_h, torch.int32, "d_best_h"),
                                  float(threshold), _dptr(d_out, torch.int32, "d_out"), cap,
                                  _dptr(d_count, torch.int64, "d_count"), stream), "hs_find_candidates")


def hs_plan_set_tuning(plan, variant: int) -> None:
    _check(load().hs_plan_set_tuning(plan, int(variant)), "hs_plan_set_tuning")


def hs_plan_set_host_slot_bytes(plan, nbytes: int) -> None:
    _check(load().hs_plan_set_host_slot_bytes(plan, int(nbytes)), "hs_plan_set_host_slot_bytes")


def hs_launch_count(plan) -> int:
    return int(load().hs_launch_count(plan))


def hs_last_kernel(plan) -> str:
    return load().hs_last_kernel(plan).decode()


def hs_destroy(plan) -> None:
    _check(load().hs_destroy(plan), "hs_destroy")
