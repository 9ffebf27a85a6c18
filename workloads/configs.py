"""The five workloads of BASELINE.json ``configs`` as plain data.

Width sets are named by (kind, param, max_width) only; the actual widths come
from the width-set generator of whichever side consumes the workload
(``oracle.formulas.width_set`` or the product's ``spd_width_set_generate``),
so this module carries none of the method.

Readings of the config text:
  * "lossy width set" = the decimation-in-time set {2^i <= max_width}
    (Alg. 3) evaluated at every sample; 14 widths at 8192 give
    8.10 % cumulative mean loss by eq. (19) and 7.36 % on log-uniform widths,
    the sparsest natural set meeting the config's "about 7 %".
  * pulse amplitude A = SNR_T / sqrt(S) on top of the noise (eq. 6,
    PAPER.md:97); SNR_T ~ U[6, 20] where the config gives no value.
  * config 5 drift: 0.1 * sin(2 pi n / (n_t / 8) + phi_d), phi_d seeded.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional, Tuple

BASE_SEED = 191008324


@dataclass(frozen=True)
class Workload:
    name: str
    index: int                      # 1-based, BASELINE.json configs order
    n_dm: int
    n_t: int
    width_kind: str                 # "ALL" | "POW2" | "BOXDIT" | "IGRID" | "GEOMETRIC"
    width_param: int
    max_width: int
    n_pulses: int
    pulse_widths: Optional[Tuple[int, ...]]   # cycle through these, or
    pulse_width_range: Optional[Tuple[int, int]]  # round(log-uniform[lo, hi])
    snr_range: Tuple[float, float]  # SNR_T uniform in [lo, hi] (lo == hi: fixed)
    stats: str                      # "unit" (mu=0, sigma=1 supplied) | "measured" (A6)
    sampling_time_s: float
    drift_amplitude: float = 0.0
    candidate_threshold: Optional[float] = None
    seed: int = field(default=0)

    @property
    def n_samples(self) -> int:
        return self.n_dm * self.n_t

    def scaled(self, n_dm: int, n_t: int, n_pulses: Optional[int] = None) -> "Workload":
        """Same recipe on a smaller plane (tests, CPU-baseline samples)."""
        from dataclasses import replace
        return replace(self, n_dm=n_dm, n_t=n_t,
                       n_pulses=self.n_pulses if n_pulses is None else n_pulses)


CONFIGS = (
    Workload("tiny_lossless", 1, 64, 16384, "ALL", 0, 64, 8,
             (1, 3, 7, 20, 45), None, (10.0, 10.0), "unit", 64e-6, seed=BASE_SEED + 1),
    Workload("small_lossy", 2, 1024, 131072, "POW2", 0, 256, 64,
             None, (1, 256), (6.0, 20.0), "measured", 64e-6, seed=BASE_SEED + 2),
    Workload("ska_mid_like", 3, 4096, 1048576, "POW2", 0, 8192, 256,
             None, (1, 8192), (6.0, 20.0), "unit", 64e-6, seed=BASE_SEED + 3),
    Workload("wide_pulse_stress", 4, 512, 4194304, "POW2", 0, 32768, 128,
             None, (512, 32768), (6.0, 20.0), "unit", 64e-6, seed=BASE_SEED + 4),
    Workload("high_time_res", 5, 64, 67108864, "POW2", 0, 16384, 512,
             None, (1, 16384), (6.0, 20.0), "unit", 256e-9,
             drift_amplitude=0.1, candidate_threshold=6.0, seed=BASE_SEED + 5),
)


def get_workload(key) -> Workload:
    """Look a workload up by 1-based index or by name."""
    for w in CONFIGS:
        if key == w.index or key == w.name:
            return w
    raise KeyError(f"unknown workload {key!r}")
