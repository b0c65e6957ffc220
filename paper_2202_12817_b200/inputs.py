"""Seeded synthetic inputs for the harmonic-sum hot path (arXiv 2202.12817).

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
path (``paper_2202_12817_b200/csrc``).  It holds none of the method's arithmetic:
it produces power spectra, the normalisation statistics the caller of the method
has to supply ("GetMeanStdev()"), and small hand-made
spectra used as test fixtures.  Everything is a pure function of its seed.

Recipe (stands in for the paper's workloads):

* noise: per bin a complex Gaussian w ~ CN(0,1) drawn from a counter-based hash of
  (seed, spectrum, bin), so |w|^2 ~ Exp(1) (BASELINE.json "|complex Gaussian|^2");
* pulsar j: fractional fundamental bin r_j, duty cycle delta_j, amplitude A_j
  (in noise-sigma units), phase phi_j, living in one spectrum s_j.  Harmonic k
  sits at p = k r_j with amplitude A_j g(k)/g(1), g(k) = exp(-(pi delta k)^2/(4 ln 2))
  (Gaussian pulse of FWHM delta periods), and is spread over the bins |b-p| <= 8
  with the DFT response sinc(b-p) e^{-i pi (b-p)} (scalloping);
* power x[b] = |w_b + sum signal_b|^2, stored fp32.

The tensors are built with torch integer/float64 ops so the same code runs on the
CPU (tests) and on the GPU (bench, full-size parity).  CPU and GPU results may
differ in the last ulp of log/sin/cos; that never matters because oracle and CUDA
path always consume the *same* buffer.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Optional, Tuple

import torch

_MASK64 = (1 << 64) - 1
_C1 = 0x9E3779B97F4A7C15
_C2 = 0xBF58476D1CE4E5B9
_C3 = 0x94D049BB133111EB


def _s64(v: int) -> int:
    """Two's-complement view of a 64-bit pattern as a signed python int."""
    v &= _MASK64
    return v - (1 << 64) if v >= (1 << 63) else v


def _mix_py(z: int) -> int:
    z &= _MASK64
    z = ((z ^ (z >> 30)) * _C2) & _MASK64
    z = ((z ^ (z >> 27)) * _C3) & _MASK64
    return z ^ (z >> 31)


def hash_u01(seed: int, *keys: int) -> float:
    """Scalar uniform in (0,1) from a hash chain of integer keys (python ints)."""
    z = _mix_py(seed * _C1 + 0x1234567)
    for k in keys:
        z = _mix_py(z ^ ((k * _C1) & _MASK64))
    return ((z >> 11) + 0.5) / float(1 << 53)


def _lsr(z: torch.Tensor, k: int) -> torch.Tensor:
    """Logical shift right on int64 tensors (torch's >> is arithmetic)."""
    return (z >> k) & ((1 << (64 - k)) - 1)


def _mix_t(z: torch.Tensor) -> torch.Tensor:
    z = (z ^ _lsr(z, 30)) * _s64(_C2)
    z = (z ^ _lsr(z, 27)) * _s64(_C3)
    return z ^ _lsr(z, 31)


def _row_key(seed: int, s: int, stream: int) -> int:
    return _s64(_mix_py(_mix_py(seed * _C1 + 0x1234567) ^ ((s * _C1) & _MASK64)) ^ ((stream * _C3) & _MASK64))


def _uniform40(seed: int, s: int, stream: int, b: torch.Tensor) -> torch.Tensor:
    """float64 uniforms in (0,1) with 40 random bits, one per bin index in ``b`` (int64)."""
    z = _mix_t(b * _s64(_C1) + _row_key(seed, s, stream))
    return (_lsr(z, 24).to(torch.float64) + 0.5) * (1.0 / float(1 << 40))


def noise_row_complex(seed: int, s: int, n_bins: int, device="cpu") -> Tuple[torch.Tensor, torch.Tensor]:
    """Real and imaginary parts (float64) of w ~ CN(0,1) for spectrum ``s``: |w|^2 ~ Exp(1)."""
    b = torch.arange(n_bins, dtype=torch.int64, device=device)
    u1 = _uniform40(seed, s, 1, b)
    u2 = _uniform40(seed, s, 2, b)
    r = torch.sqrt(-torch.log(u1))
    th = (2.0 * math.pi) * u2
    return r * torch.cos(th), r * torch.sin(th)


@dataclass
class Pulsar:
    spectrum: int      # s_j
    r: float           # fractional fundamental bin
    duty: float        # duty cycle delta (FWHM / period)
    amp: float         # fundamental amplitude in noise-sigma units ("amplitude SNR")
    phase: float       # phi_j

    def n_harmonics(self, n_bins: int) -> int:
        """Harmonics "to the bin limit" (BASELINE.json), dropped once below 1e-6 of the fundamental."""
        k_band = int(math.floor((n_bins - 2) / self.r))
        k_amp = int(math.sqrt(4.0 * math.log(2.0) * math.log(1e6)) / (math.pi * self.duty)) + 1
        return max(0, min(k_band, k_amp, 1 << 16))


def _inject(re: torch.Tensor, im: torch.Tensor, p: Pulsar, half_width: int = 8) -> None:
    n_bins = re.numel()
    K = p.n_harmonics(n_bins)
    if K <= 0:
        return
    dev = re.device
    k = torch.arange(1, K + 1, dtype=torch.float64, device=dev)
    g = torch.exp(-((math.pi * p.duty) ** 2) * (k * k - 1.0) / (4.0 * math.log(2.0)))  # g(k)/g(1)
    pos = k * p.r
    centre = torch.round(pos).to(torch.int64)
    off = torch.arange(-half_width, half_width + 1, dtype=torch.int64, device=dev)
    bins = centre[:, None] + off[None, :]
    t = bins.to(torch.float64) - pos[:, None]
    # DFT response of an off-centre tone: sinc(t) e^{-i pi t}; harmonic phase k*phi
    resp = torch.sinc(t) * (p.amp * g)[:, None]
    ang = (k * p.phase)[:, None] - math.pi * t
    ok = (bins >= 0) & (bins < n_bins)
    idx = bins[ok]
    re.index_add_(0, idx, (resp * torch.cos(ang))[ok])
    im.index_add_(0, idx, (resp * torch.sin(ang))[ok])


@dataclass
class Workload:
    """One named configuration of BASELINE.json / SURVEY.md section 8(d)."""
    name: str
    n_spectra: int
    n_bins: int
    H: int
    seed: int
    n_pulsars: int = 0
    r_range: Tuple[float, float] = (100.0, 65536.0)
    duty_range: Tuple[float, float] = (0.05, 0.05)
    amp_range: Tuple[float, float] = (8.0, 8.0)
    fixed: Optional[List[Pulsar]] = None
    red_noise: bool = False
    pulsars: List[Pulsar] = field(default_factory=list)

    def __post_init__(self):
        if self.fixed is not None:
            self.pulsars = list(self.fixed)
        else:
            self.pulsars = []
            for j in range(self.n_pulsars):
                u = [hash_u01(self.seed, 0xABCD, j, q) for q in range(5)]
                self.pulsars.append(Pulsar(
                    spectrum=min(self.n_spectra - 1, int(u[0] * self.n_spectra)),
                    r=self.r_range[0] + u[1] * (self.r_range[1] - self.r_range[0]),
                    duty=self.duty_range[0] + u[2] * (self.duty_range[1] - self.duty_range[0]),
                    amp=self.amp_range[0] + u[3] * (self.amp_range[1] - self.amp_range[0]),
                    phase=2.0 * math.pi * u[4]))


def workload(name: str) -> Workload:
    """The configurations of BASELINE.json ("configs") and the paper-shaped case P."""
    if name == "cfg1":      # BASELINE.json configs[0]
        return Workload("cfg1", 1, 1 << 16, 8, seed=1,
                        fixed=[Pulsar(0, 1000.5, 0.05, 8.0, 0.7)])
    if name == "cfg2":      # configs[1]
        return Workload("cfg2", 64, 1 << 20, 16, seed=2, n_pulsars=16,
                        r_range=(100.0, float(1 << 16)), duty_range=(0.01, 0.2), amp_range=(5.0, 15.0))
    if name == "cfg3":      # configs[2] -- the headline throughput configuration
        n = 1 << 22
        return Workload("cfg3", 256, n, 32, seed=3, n_pulsars=64,
                        r_range=(100.0, n / 32.0), duty_range=(0.01, 0.3), amp_range=(4.0, 12.0))
    if name == "cfg4":      # configs[3] (NEXT-2): red noise + per-bin baseline
        n = 1 << 21
        return Workload("cfg4", 1024, n, 32, seed=4, n_pulsars=128,
                        r_range=(100.0, n / 32.0), duty_range=(0.01, 0.3), amp_range=(4.0, 12.0),
                        red_noise=True)
    if name == "cfgP":      # the paper's Table 2 shape: 1024 x "131 thousand", pure noise
        return Workload("cfgP", 1024, 1 << 17, 32, seed=6)
    raise KeyError(name)


def red_noise_trend(n_bins: int, device="cpu") -> torch.Tensor:
    """Per-bin mean 1 + 20/(1 + bin/500) (BASELINE.json configs[3])."""
    b = torch.arange(n_bins, dtype=torch.float64, device=device)
    return 1.0 + 20.0 / (1.0 + b / 500.0)


def generate_row(w: Workload, s: int, device="cpu", n_bins: Optional[int] = None) -> torch.Tensor:
    """fp32 power spectrum of DM trial ``s`` of workload ``w``."""
    n = w.n_bins if n_bins is None else n_bins
    re, im = noise_row_complex(w.seed, s, n, device)
    for p in w.pulsars:
        if p.spectrum == s:
            _inject(re, im, p)
    x = re * re + im * im
    if w.red_noise:
        x = x * red_noise_trend(n, device)
    return x.to(torch.float32)


def generate(w: Workload, device="cpu", n_spectra: Optional[int] = None,
             out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """[S, N] fp32 batch of power spectra (row-major, one row per DM trial)."""
    S = w.n_spectra if n_spectra is None else n_spectra
    if out is None:
        out = torch.empty((S, w.n_bins), dtype=torch.float32, device=device)
    for s in range(S):
        out[s].copy_(generate_row(w, s, device))
    return out


def block_median_inv_baseline(x: torch.Tensor, block: int = 1024) -> torch.Tensor:
    """Per-bin reciprocal running-median baseline (configs[3]): block medians / ln 2, expanded per bin.

    This is the *caller's* whitening estimate; the method only receives it."""
    S, N = x.shape
    nb = (N + block - 1) // block
    pad = nb * block - N
    xp = torch.nn.functional.pad(x, (0, pad), mode="replicate") if pad else x
    med = xp.view(S, nb, block).median(dim=2).values.to(torch.float64) / math.log(2.0)
    inv = (1.0 / med).to(torch.float32)
    return inv.repeat_interleave(block, dim=1)[:, :N].contiguous()


# ----------------------------------------------------------------------------------------------
# Normalisation statistics supplied by the caller for Exp(1) noise.
# These are INPUTS of the method (mu[h], sigma[h]); any values are accepted.
# ----------------------------------------------------------------------------------------------
def exp1_stats(variant: str, H: int, fund_select: bool = True) -> Tuple[torch.Tensor, torch.Tensor]:
    """(mu, sigma) float32 arrays of length H, entry h-1 for harmonic order h.

    greedy: every step adds the larger of two iid Exp(1) (mean 3/2, variance 5/4); without
    fundamental selection the first term is a plain Exp(1).  presto (Alg. 1): 1 term at H'=1,
    1 + H'/2 terms otherwise; presto_all/presto_plus/simple: H' terms of mean 1, variance 1."""
    mu, var = [], []
    for h in range(1, H + 1):
        if variant == "greedy":
            if fund_select:
                mu.append(1.5 * h); var.append(1.25 * h)
            else:
                mu.append(1.0 + 1.5 * (h - 1)); var.append(1.0 + 1.25 * (h - 1))
        elif variant == "presto":
            t = 1.0 if h == 1 else 1.0 + (h // 2)
            mu.append(t); var.append(t)
        elif variant in ("presto_all", "presto_plus", "simple"):
            mu.append(float(h)); var.append(float(h))
        else:
            raise ValueError(variant)
    return (torch.tensor(mu, dtype=torch.float32),
            torch.tensor([math.sqrt(v) for v in var], dtype=torch.float32))


# ----------------------------------------------------------------------------------------------
# Hand-made fixtures (tests only)
# ----------------------------------------------------------------------------------------------
def integer_spectra(seed: int, n_spectra: int, n_bins: int, max_val: int = 255) -> torch.Tensor:
    """Small non-negative integers as fp32: every partial sum is exact in fp32 and fp64 (pin P7)."""
    out = torch.empty((n_spectra, n_bins), dtype=torch.float32)
    b = torch.arange(n_bins, dtype=torch.int64)
    for s in range(n_spectra):
        z = _mix_t(b * _s64(_C1) + _row_key(seed, s, 7))
        out[s] = (_lsr(z, 33) % (max_val + 1)).to(torch.float32)
    return out


def delta_train(n_bins: int, f0: int, K: int, A: float) -> torch.Tensor:
    """x = 0 except x[k f0] = A for k = 1..K (pin P3)."""
    x = torch.zeros(n_bins, dtype=torch.float32)
    for k in range(1, K + 1):
        x[k * f0] = A
    return x


# ----------------------------------------------------------------------------------------------
# configs[4] (NEXT-4): an f-fdot plane -- n_z = 2 Z + 1 rows (z = -Z .. Z) of n_bins Exp(1) powers with drifting signals
# ----------------------------------------------------------------------------------------------
@dataclass
class Drifter:
    r: float          # fractional fundamental frequency bin
    z: float          # fractional fundamental drift (f-dot) row
    duty: float
    amp: float
    phase: float


@dataclass
class PlaneWorkload:
    name: str
    n_z: int
    n_bins: int
    H: int
    seed: int
    n_signals: int
    signals: List[Drifter] = field(default_factory=list)

    def __post_init__(self):
        Z = (self.n_z - 1) // 2
        zmax = max(0.0, Z / 16.0 - 0.25)                 # all 16 harmonics of every signal stay inside the plane
        self.signals = []
        for j in range(self.n_signals):
            u = [hash_u01(self.seed, 0xD51F, j, q) for q in range(5)]
            self.signals.append(Drifter(r=100.0 + u[0] * (self.n_bins / 16.0 - 100.0), z=(2.0 * u[1] - 1.0) * zmax,
                                        duty=0.02 + u[2] * 0.18, amp=6.0 + u[3] * 8.0, phase=2.0 * math.pi * u[4]))


def plane_workload(name: str) -> PlaneWorkload:
    if name == "cfg5":      # BASELINE.json configs[4]: 2^21 frequency bins x 201 fdot rows, 32 drifting signals, H = 16
        return PlaneWorkload("cfg5", 201, 1 << 21, 16, seed=5, n_signals=32)
    raise KeyError(name)


def generate_plane(w: PlaneWorkload, device="cpu", n_bins: Optional[int] = None) -> torch.Tensor:
    """[n_z, N] fp32 plane: |complex Gaussian noise + signals|^2.  Harmonic k of a signal sits at (k r, k z): the DFT
    response in r (as in the 1-D generator) is put into the row floor(k z) with weight cos^2 and the row above with
    weight sin^2 of the fractional part (a stand-in for the f-dot response; none of the method's arithmetic)."""
    n = w.n_bins if n_bins is None else n_bins
    Z = (w.n_z - 1) // 2
    out = torch.empty((w.n_z, n), dtype=torch.float32, device=device)
    for zi in range(w.n_z):
        re, im = noise_row_complex(w.seed, zi, n, device)
        for sg in w.signals:
            for k in range(1, 17):
                zz = k * sg.z
                row = math.floor(zz)
                frac = zz - row
                for rr, wgt in ((row, math.cos(0.5 * math.pi * frac) ** 2), (row + 1, math.sin(0.5 * math.pi * frac) ** 2)):
                    if rr + Z != zi or wgt < 1e-6 or k * sg.r >= n - 1:
                        continue
                    g = math.exp(-((math.pi * sg.duty * k) ** 2) / (4.0 * math.log(2.0)))
                    g1 = math.exp(-((math.pi * sg.duty) ** 2) / (4.0 * math.log(2.0)))
                    amp = sg.amp * g / g1 * math.sqrt(wgt)
                    pos = k * sg.r
                    b = torch.arange(max(0, math.floor(pos) - 8), min(n, math.floor(pos) + 10), device=device)
                    dlt = b.to(torch.float64) - pos
                    resp = amp * torch.sinc(dlt)
                    ang = sg.phase * k - math.pi * dlt
                    re[b] += (resp * torch.cos(ang)).to(re.dtype)
                    im[b] += (resp * torch.sin(ang)).to(im.dtype)
        out[zi].copy_((re * re + im * im).to(torch.float32))
    return out
