"""Seeded synthetic inputs for the single-pulse-detection (SPD) hot path.

This package is the ONLY code shared by the CPU oracle (``oracle/``) and the
CUDA product (``paper_1910_08324_b200/``).  It holds none of the method's
arithmetic: no boxcar sums, no SNR, no width-set generation, no max-reduce.
It only describes the five workloads of ``BASELINE.json`` (shape, pulse
population, noise, drift, sampling time) and draws them from a seed.

The recipe follows the paper's idealised signal model (sec. 2.1,
eq. 6: rectangular pulse of width S and amplitude A = C / sqrt(S)) with N(0,1)
white noise added (sec. 4.4).  See DESIGN.md "Input recipe".
"""
from .configs import CONFIGS, Workload, get_workload
from .generate import (
    Pulse,
    draw_pulses,
    make_plane_numpy,
    make_plane_torch,
    make_pulse_only_plane_numpy,
    make_shaped_pulse_plane_numpy,
    pulse_amplitude,
    pulse_profile,
)

__all__ = [
    "CONFIGS",
    "Workload",
    "get_workload",
    "Pulse",
    "draw_pulses",
    "make_plane_numpy",
    "make_plane_torch",
    "make_pulse_only_plane_numpy",
    "make_shaped_pulse_plane_numpy",
    "pulse_amplitude",
    "pulse_profile",
]
