"""ORACLE (test infrastructure only) - the paper's sensitivity formulae and width sets.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s CPU-baseline /
``--impl reference`` legs may import this.  The CUDA product never does; it has
its own width-set generator in C++ (``spd_width_set_generate``).

Everything follows /root/reference/PAPER.md (Adamek & Armour 2020) in the
paper's notation, C = 1 (responses are fractions of the true SNR):

  rsnr(S, L, d_s)            eq. (22)
  rsnr_max_single(S, L)      eq. (23)
  rsnr_max(S, widths)        eq. (24)
  coverage_lt / coverage_gt  eq. (27), (29)
  rsnr_min_single(S, L, Ls)  eq. (30)
  rsnr_min(S, widths, Ls)    eq. (31)
  loss                       eq. (7)-(9) PAPER.md:105-128
  cumulative_mean_loss       eq. (19)
  width sets                 ideal, DIT,
                             BoxDIT eq. (14), IGRID eq. (18)/Table 1
                             PAPER.md:364-387

Pinned by tests/test_formulas.py against the numbers the paper prints and
against a brute-force scan over pulse shifts (which shares no code with the
closed forms).  Readings of garbled passages: DESIGN.md "Readings" G3 (the
case list at PAPER.md:947-950 lost its minus signs; eq. 27/29/30 as typeset
are used).
"""
from __future__ import annotations

import math
from typing import Callable, Dict, Iterable, List, Sequence, Union

import numpy as np

# ----------------------------------------------------------------------------
# Responses (fractions of SNR_T, i.e. C = 1)
# ----------------------------------------------------------------------------


def rsnr(S: int, L: int, d_s: int) -> float:
    """eq. (22): RSNR = d_s * C / (sqrt(L) * sqrt(S)), C = 1."""
    return d_s / (math.sqrt(L) * math.sqrt(S))


def rsnr_max_single(S: int, L: int) -> float:
    """eq. (23): best-case response of one boxcar of width L to a pulse of width S."""
    if S < L:
        return math.sqrt(S) / math.sqrt(L)
    return math.sqrt(L) / math.sqrt(S)


def rsnr_max(S: int, widths: Iterable[int]) -> float:
    """eq. (24): best-case response of the whole width set."""
    return max(rsnr_max_single(S, L) for L in widths)


def coverage_lt(S: int, L: int, Ls: int) -> int:
    """eq. (27): d_s^< = S - floor((S - L + Ls) / 2), for L - Ls < S < L."""
    return S - (S - L + Ls) // 2


def coverage_gt(S: int, L: int, Ls: int) -> int:
    """eq. (29): d_s^> = L - floor((L + Ls - S) / 2), for L <= S < L + Ls."""
    return L - (L + Ls - S) // 2


def rsnr_min_single(S: int, L: int, Ls: int) -> float:
    """eq. (30): worst-case response of boxcars of width L placed every Ls samples."""
    if S <= L - Ls:
        return math.sqrt(S) / math.sqrt(L)
    if S < L:
        return coverage_lt(S, L, Ls) / math.sqrt(L * S)
    if S < L + Ls:
        return coverage_gt(S, L, Ls) / math.sqrt(L * S)
    return math.sqrt(L) / math.sqrt(S)


SeparationSpec = Union[int, Dict[int, int], Callable[[int], int]]


def _separation(Ls: SeparationSpec, L: int) -> int:
    if callable(Ls):
        return int(Ls(L))
    if isinstance(Ls, dict):
        return int(Ls[L])
    return int(Ls)


def rsnr_min(S: int, widths: Iterable[int], Ls: SeparationSpec) -> float:
    """eq. (31): worst-case response of the whole algorithm; Ls may depend on L."""
    return max(rsnr_min_single(S, L, _separation(Ls, L)) for L in widths)


def systematic_loss(S: int, widths: Iterable[int]) -> float:
    """eq. (9): Psi_l(S) = 1 - RSNR_max(S) / SNR_T."""
    return 1.0 - rsnr_max(S, widths)


def worst_loss(S: int, widths: Iterable[int], Ls: SeparationSpec) -> float:
    """eq. (8): Psi_w(S) = 1 - RSNR_min(S) / SNR_T."""
    return 1.0 - rsnr_min(S, widths, Ls)


def cumulative_mean_loss(psi: Callable[[int], float], S0: int) -> float:
    """eq. (19) exactly as printed: sum_{s=1}^{S0} Psi(s) / (S0 - 1)."""
    return sum(psi(s) for s in range(1, S0 + 1)) / (S0 - 1)


def mean_loss_over_widths(pulse_widths: Iterable[int], widths: Sequence[int]) -> float:
    """Mean of eq. (9) over a given pulse-width population (north_star's
    'mean SNR loss measured on injected rectangular pulses')."""
    pw = list(pulse_widths)
    return sum(systematic_loss(S, widths) for S in pw) / len(pw)


# ----------------------------------------------------------------------------
# Brute force over pulse shifts - shares nothing with eq. (27)-(31); used to pin them
# ----------------------------------------------------------------------------


def brute_force_response(S: int, widths: Sequence[int], Ls: SeparationSpec):
    """Slide a width-S pulse over every integer shift, measure the best response
    of boxcars of each width L placed at multiples of Ls(L) (the paper's method,
    PAPER.md:492-494).  Returns (min over shifts, max over shifts, mean over shifts)
    of the per-shift best response."""
    seps = [_separation(Ls, L) for L in widths]
    period = 1
    for s in seps:
        period = period * s // math.gcd(period, s)
    best_per_shift: List[float] = []
    for shift in range(period):
        t0 = shift
        t1 = shift + S
        best = 0.0
        for L, sep in zip(widths, seps):
            # boxcars start at k*sep; those intersecting [t0, t1)
            k_lo = (t0 - L) // sep
            k_hi = t1 // sep + 1
            for k in range(k_lo, k_hi + 1):
                b0 = k * sep
                ov = min(t1, b0 + L) - max(t0, b0)
                if ov > 0:
                    r = ov / math.sqrt(L * S)
                    if r > best:
                        best = r
        best_per_shift.append(best)
    return min(best_per_shift), max(best_per_shift), sum(best_per_shift) / len(best_per_shift)


# ----------------------------------------------------------------------------
# Width sets
# ----------------------------------------------------------------------------


def widths_all(max_width: int) -> List[int]:
    """Ideal SPD algorithm: every width 1..L_max."""
    return list(range(1, max_width + 1))


def widths_pow2(max_width: int) -> List[int]:
    """Decimation-in-time set B = {1, 2, 4, ..., 2^I}."""
    out, L = [], 1
    while L <= max_width:
        out.append(L)
        L *= 2
    return out


def widths_boxdit(l_max: int, max_width: int, D: int = 2) -> List[int]:
    """BoxDIT widths by eq. (14): L = sum_{k<i} D^k L_max + D^i m, m = 1..L_max,
    for iterations i = 0, 1, ... until max_width (example
    L_max = 4: 1,2,3,4 then 6,8,10,12)."""
    out: List[int] = []
    base, step = 0, 1
    while True:
        added = False
        for m in range(1, l_max + 1):
            L = base + step * m
            if L <= max_width:
                out.append(L)
                added = True
        base += step * l_max
        step *= D
        if not added or base >= max_width:
            break
    return sorted(set(out))


def widths_igrid(depth: int, max_width: int) -> List[int]:
    """IGRID widths: each step 2^i contributes L = sum_k a_k 2^(i-k), a_0 = a_1 = 1,
    a_k = +-1, k <= depth (eq. 18), i.e. 2^i + j * 2^(i-depth),
    j = 0 .. 2^depth - 1 (Table 1: 16 -> 16,24 | 16,20,24,28 |
    16,18,...,30).  For 2^i < 2^depth the step is one sample."""
    out: List[int] = []
    base = 1
    while base <= max_width:
        step = max(1, base >> depth)
        L = base
        while L < 2 * base:
            if L <= max_width:
                out.append(L)
            L += step
        base *= 2
    return sorted(set(out))


def widths_geometric(ratio: float, max_width: int) -> List[int]:
    """Rounded geometric progression 1, r, r^2, ... capped at max_width."""
    out, x = [], 1.0
    while round(x) <= max_width:
        out.append(int(round(x)))
        x *= ratio
    return sorted(set(out))


def width_set(kind: str, param: int, max_width: int) -> List[int]:
    """Width set named by a workload (workloads.configs.Workload.width_kind)."""
    kind = kind.upper()
    if kind == "ALL":
        return widths_all(max_width)
    if kind == "POW2":
        return widths_pow2(max_width)
    if kind == "BOXDIT":
        return widths_boxdit(param, max_width)
    if kind == "IGRID":
        return widths_igrid(param, max_width)
    if kind == "GEOMETRIC":
        return widths_geometric(param / 1000.0, max_width)
    raise ValueError(f"unknown width-set kind {kind!r}")


def boxdit_separation(l_max: int, D: int = 2) -> Callable[[int], int]:
    """Boxcar separation of a BoxDIT width: L_s = D^i in iteration i (Alg. 1)."""
    def sep(L: int) -> int:
        base, step = 0, 1
        while L > base + step * l_max:
            base += step * l_max
            step *= D
        return step
    return sep


def igrid_separation(layers: int) -> Callable[[int], int]:
    """Boxcar separation of an IGRID width in step i with P layers: L_s = 2^i / P
    (PAPER.md:356), at least one sample."""
    def sep(L: int) -> int:
        base = 1 << (int(L).bit_length() - 1)
        return max(1, base // layers)
    return sep


def as_array(widths: Iterable[int]) -> np.ndarray:
    return np.asarray(sorted(set(int(w) for w in widths)), dtype=np.int32)
