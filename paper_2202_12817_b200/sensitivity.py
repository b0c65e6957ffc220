"""Sensitivity-loss workload of the paper (section 4.1.1).

A noiseless artificial pulsar -- the modified von Mises pulse train of eq. 10 -- is
generated for a set of true frequencies that step from the centre of frequency bin ``n_c`` to the
centre of bin ``n_c + 1`` (T = 20 s, t_s = 64 us, bin width 0.05 Hz, 50 steps: PAPER.md:286), each
time series is Fourier transformed, and the power spectra form one batch for the harmonic-sum
library.  The sensitivity loss of an algorithm is l(f) = RSNR(f) / RSNR(f_0), eq. 11.

This module only builds the INPUTS (time series -> power spectra, with torch) and reduces the
library's OUTPUTS to l(f); it holds none of the method's arithmetic.  The figures of the paper
(Fig. 9-11) are not in PAPER.md, so tests only check what the text states.
"""
from __future__ import annotations

import math
from typing import Tuple

import torch

T_OBS = 20.0            # s
T_SAMP = 64e-6          # s
N_STEPS = 50            # steps across one bin width


def von_mises_spectra(n_c: int = 500, kappa: float = 50.0, phase: float = 0.3, device="cpu",
                      n_steps: int = N_STEPS, peak_power: float = 100.0) -> Tuple[torch.Tensor, float]:
    """[n_steps + 1, N] fp32 power spectra of eq. 10 with f_r = (n_c + k / n_steps) / T, k = 0..n_steps.

    Returns (spectra, bin width in Hz).  The spectra are scaled so that the bin-centred fundamental (k = 0)
    has power ``peak_power``; the DC bin is set to 0 (the pulse train has a non-zero mean)."""
    n_samp = int(round(T_OBS / T_SAMP))
    t = torch.arange(n_samp, dtype=torch.float64, device=device) * T_SAMP
    e2k = math.exp(-2.0 * kappa)
    norm = float(torch.special.i0e(torch.tensor(kappa, dtype=torch.float64))) - e2k     # (I0(k) - e^-k) e^-k
    rows = []
    for k in range(n_steps + 1):
        f_r = (n_c + k / n_steps) / T_OBS
        series = (torch.exp(kappa * (torch.cos(2.0 * math.pi * f_r * t + phase) - 1.0)) - e2k) / norm
        spec = torch.fft.rfft(series)
        rows.append(spec.real ** 2 + spec.imag ** 2)
    p = torch.stack(rows)
    p[:, 0] = 0.0
    p *= peak_power / float(p[0, n_c])
    return p.to(torch.float32).contiguous(), 1.0 / T_OBS


def loss_curve(snr: torch.Tensor, lo: int = 10) -> torch.Tensor:
    """l(f_k) = RSNR(f_k) / RSNR(f_0) (eq. 11) with RSNR = the largest SNR the algorithm returned for the
    spectrum (noiseless data: the maximum sits on the signal), bins below ``lo`` ignored."""
    rsnr = snr[:, lo:].max(dim=1).values.to(torch.float64)
    return rsnr / rsnr[0]
