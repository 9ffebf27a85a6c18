"""Seeded generators for the SPD workloads (inputs only - none of the method).

Input recipe:
  plane[d, n] = noise[d, n] + drift[d, n] + sum_p A_p * [t_p <= n < t_p + S_p] * [d == d_p]
  noise ~ i.i.d. N(0, 1) float32                         (sec. 4.4)
  A_p = SNR_T / sqrt(S_p)                                (eq. 6)
  drift = a * sin(2 pi n / (n_t / 8) + phi_d)            (config 5 only; reading A12)

Pulse parameters always come from ``numpy.random.default_rng(seed)`` so that the
CPU (numpy) and GPU (torch) plane builders inject the same pulses.  The noise
stream differs between the two builders (numpy PCG64 vs torch Philox); each
test or bench run builds the plane once and hands the same buffer to both the
oracle and the CUDA path.
"""
from __future__ import annotations

import math
from dataclasses import dataclass
from typing import List, Tuple

import numpy as np

from .configs import Workload


@dataclass(frozen=True)
class Pulse:
    dm: int          # DM-trial (row) index
    t0: int          # first sample of the pulse
    width: int       # S, samples
    snr_t: float     # true SNR: what a matched boxcar recovers on unit noise
    amplitude: float  # A = snr_t / sqrt(S)


def pulse_amplitude(snr_t: float, width: int) -> float:
    """A(S) = C / sqrt(S), eq. (6) with C = SNR_T."""
    return float(snr_t) / math.sqrt(float(width))


def pulse_profile(shape: str, width: int, snr_t: float) -> np.ndarray:
    """Samples of one pulse of ``width`` samples (float64), normalised as PAPER.md:553: "when all its
    samples are summed together, i.e. a boxcar of signal width is applied to it, it will produce
    RSNR = C" on unit noise, i.e. sum = snr_t * sqrt(width).

    shape "rect": eq. (6).  "gauss" / "double_gauss": eq. (20), sampled at
    the integers 0 .. width-1 with mean width/2 (reading A15: the printed variances S/(8 ln 2),
    (S/4)/(8 ln 2), (S/5)/(8 ln 2) are taken as FWHM^2/(8 ln 2) with FWHM = S/2, S/4, S/5 - the
    reading that reproduces the worked example of PAPER.md:577, a 20-sample Gaussian best matched by
    an 11-sample boxcar 4-5 samples late; the two components of the double Gaussian sit at S/3 and
    2S/3 with equal weight - the paper does not say where)."""
    n = np.arange(width, dtype=np.float64)
    k = 8.0 * math.log(2.0)
    if shape == "rect":
        prof = np.ones(width, dtype=np.float64)
    elif shape == "gauss":
        var = (width / 2.0) ** 2 / k
        prof = np.exp(-((n - width / 2.0) ** 2) / (2.0 * var))
    elif shape == "double_gauss":
        v1, v2 = (width / 4.0) ** 2 / k, (width / 5.0) ** 2 / k
        prof = (np.exp(-((n - width / 3.0) ** 2) / (2.0 * v1)) / math.sqrt(v1)
                + np.exp(-((n - 2.0 * width / 3.0) ** 2) / (2.0 * v2)) / math.sqrt(v2))
    else:
        raise ValueError(f"unknown pulse shape {shape!r}")
    return prof * (float(snr_t) * math.sqrt(float(width)) / prof.sum())


def make_shaped_pulse_plane_numpy(w: Workload, shape: str, noise: bool = False) -> Tuple[np.ndarray, List[Pulse]]:
    """The workload's pulses drawn with another profile (sec. 4.3) on a zero
    background ("The input time-series is zeroed") or on the workload's noise."""
    if noise:
        rng = np.random.default_rng(w.seed + 104729)
        plane = rng.standard_normal(size=(w.n_dm, w.n_t), dtype=np.float32)
    else:
        plane = np.zeros((w.n_dm, w.n_t), dtype=np.float32)
    pulses = draw_pulses(w)
    for p in pulses:
        plane[p.dm, p.t0:p.t0 + p.width] += pulse_profile(shape, p.width, p.snr_t).astype(np.float32)
    return plane, pulses


def draw_pulses(w: Workload) -> List[Pulse]:
    """Draw the injected-pulse population of a workload from its seed."""
    rng = np.random.default_rng(w.seed)
    pulses: List[Pulse] = []
    for i in range(w.n_pulses):
        dm = int(rng.integers(0, w.n_dm))
        if w.pulse_widths is not None:
            width = int(w.pulse_widths[i % len(w.pulse_widths)])
        else:
            lo, hi = w.pulse_width_range
            width = int(round(math.exp(rng.uniform(math.log(lo), math.log(hi)))))
            width = max(lo, min(hi, width))
        width = min(width, w.n_t)
        s_lo, s_hi = w.snr_range
        snr_t = float(s_lo if s_lo == s_hi else rng.uniform(s_lo, s_hi))
        # start uniform in [M, n_t - S - M] when that range exists, else anywhere it fits
        lo_t, hi_t = w.max_width, w.n_t - width - w.max_width
        if hi_t < lo_t:
            lo_t, hi_t = 0, w.n_t - width
        t0 = int(rng.integers(lo_t, hi_t + 1))
        pulses.append(Pulse(dm, t0, width, snr_t, pulse_amplitude(snr_t, width)))
    return pulses


def _drift_phases(w: Workload) -> np.ndarray:
    rng = np.random.default_rng(w.seed + 7919)
    return rng.uniform(0.0, 2.0 * math.pi, size=w.n_dm)


def make_pulse_only_plane_numpy(w: Workload) -> Tuple[np.ndarray, List[Pulse]]:
    """Noise-free twin: zero background plus the same pulses."""
    plane = np.zeros((w.n_dm, w.n_t), dtype=np.float32)
    pulses = draw_pulses(w)
    for p in pulses:
        plane[p.dm, p.t0:p.t0 + p.width] += np.float32(p.amplitude)
    return plane, pulses


def make_plane_numpy(w: Workload, noise: bool = True) -> Tuple[np.ndarray, List[Pulse]]:
    """Full workload plane on the host (use for planes that fit host RAM)."""
    if noise:
        rng = np.random.default_rng(w.seed + 104729)
        plane = rng.standard_normal(size=(w.n_dm, w.n_t), dtype=np.float32)
    else:
        plane = np.zeros((w.n_dm, w.n_t), dtype=np.float32)
    if w.drift_amplitude != 0.0:
        phases = _drift_phases(w)
        period = w.n_t / 8.0
        n = np.arange(w.n_t, dtype=np.float64)
        for d in range(w.n_dm):
            plane[d] += (w.drift_amplitude * np.sin(2.0 * math.pi * n / period + phases[d])).astype(np.float32)
    pulses = draw_pulses(w)
    for p in pulses:
        plane[p.dm, p.t0:p.t0 + p.width] += np.float32(p.amplitude)
    return plane, pulses


def make_plane_torch(w: Workload, device, noise: bool = True, rows_per_block: int = 64):
    """Full workload plane built directly in device memory (torch plumbing only).

    Returns (plane [n_dm, n_t] float32 on ``device``, pulses).  Generated in row
    blocks so that the 16 GiB planes never need a second full-size buffer.
    """
    import torch

    dev = torch.device(device)
    plane = torch.empty((w.n_dm, w.n_t), dtype=torch.float32, device=dev)
    if noise:
        gen = torch.Generator(device=dev)
        gen.manual_seed(w.seed + 104729)
        for r0 in range(0, w.n_dm, rows_per_block):
            r1 = min(w.n_dm, r0 + rows_per_block)
            plane[r0:r1].normal_(mean=0.0, std=1.0, generator=gen)
    else:
        plane.zero_()
    if w.drift_amplitude != 0.0:
        phases = _drift_phases(w)
        period = w.n_t / 8.0
        chunk = 1 << 24
        for c0 in range(0, w.n_t, chunk):
            c1 = min(w.n_t, c0 + chunk)
            n = torch.arange(c0, c1, dtype=torch.float64, device=dev) * (2.0 * math.pi / period)
            for d in range(w.n_dm):
                plane[d, c0:c1] += (w.drift_amplitude * torch.sin(n + float(phases[d]))).to(torch.float32)
    pulses = draw_pulses(w)
    for p in pulses:
        plane[p.dm, p.t0:p.t0 + p.width] += p.amplitude
    return plane, pulses
