"""Comparison rule of the parity tests (north_star / SURVEY.md sec. 8(c) "Comparison rule").

  * best SNR:   |dSNR| <= 1e-4 * max(1, |SNR_oracle|) at every sample;
  * best width: exact wherever the oracle's best and runner-up SNR differ by more than
                that tolerance; elsewhere the width the CUDA path chose must itself have an
                oracle SNR within the tolerance of the oracle's best (any near-tie is valid);
  * samples where no width fits (reading A3): SNR = -inf and width index = -1 on both sides.

Only the oracle is called here; the CUDA outputs arrive as numpy arrays.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

SNR_RTOL = 1e-4  # north_star: |dSNR| <= 1e-4 * max(1, |SNR|)


@dataclass
class ParityStats:
    n: int
    max_err_over_tol: float
    n_width_mismatch: int
    n_near_tie_checked: int


def snr_tolerance(ref: np.ndarray) -> np.ndarray:
    return SNR_RTOL * np.maximum(1.0, np.abs(ref))


def assert_parity(oracle, plane_rows: np.ndarray, mu, sg, widths, got_snr: np.ndarray, got_idx: np.ndarray,
                  ref_snr: np.ndarray, ref_idx: np.ndarray, ref_second: np.ndarray, t0: int = 0,
                  what: str = "", stride: int = 1) -> ParityStats:
    """plane_rows [r, n_t] float32 are the rows the outputs belong to; outputs cover samples
    [t0, t0 + span) of those rows - or, for the decimated plane of one iteration (eq. 12), column c is
    sample (t0 + c) * stride.  mu, sg: per-row float64 arrays (or scalars)."""
    got_snr = np.asarray(got_snr)
    got_idx = np.asarray(got_idx)
    assert got_snr.shape == ref_snr.shape == got_idx.shape == ref_idx.shape, what
    r, span = ref_snr.shape
    mu = np.broadcast_to(np.asarray(mu, dtype=np.float64), (r,))
    sg = np.broadcast_to(np.asarray(sg, dtype=np.float64), (r,))
    widths = np.asarray(sorted(set(int(w) for w in widths)), dtype=np.int64)

    # no-fit samples
    nofit = ref_idx < 0
    if nofit.any():
        assert np.all(np.isneginf(got_snr[nofit])), f"{what}: expected -inf where no width fits"
        assert np.all(got_idx[nofit] == -1), f"{what}: expected width index -1 where no width fits"
    ok = ~nofit
    assert np.all(np.isfinite(got_snr[ok])), f"{what}: non-finite SNR from the CUDA path"

    tol = snr_tolerance(np.where(ok, ref_snr, 0.0))
    err = np.where(ok, np.abs(got_snr.astype(np.float64) - np.where(ok, ref_snr, 0.0)), 0.0)
    ratio = err / tol
    worst = float(ratio.max()) if ratio.size else 0.0
    if worst > 1.0:
        i = np.unravel_index(int(np.argmax(ratio)), ratio.shape)
        raise AssertionError(
            f"{what}: SNR mismatch at row {i[0]} sample {t0 + i[1]}: cuda {got_snr[i]!r} oracle {ref_snr[i]!r} "
            f"(err/tol = {worst:.3g}; {int((ratio > 1).sum())} of {ratio.size} samples out of tolerance)")

    assert np.all((got_idx[ok] >= 0) & (got_idx[ok] < widths.size)), f"{what}: width index out of range"
    diff = ok & (got_idx != ref_idx)
    n_diff = int(diff.sum())
    n_checked = 0
    if n_diff:
        with np.errstate(invalid="ignore"):   # -inf - -inf where no width fits: those samples are not in `diff`
            gap = ref_snr - ref_second
        decisive = diff & (gap > tol)
        if decisive.any():
            i = np.argwhere(decisive)[0]
            raise AssertionError(
                f"{what}: width index mismatch at row {i[0]} sample {t0 + i[1]} where the oracle's top two "
                f"differ by {gap[tuple(i)]:.3g} > tol: cuda {got_idx[tuple(i)]} oracle {ref_idx[tuple(i)]} "
                f"({int(decisive.sum())} decisive mismatches)")
        # near ties: the chosen width must be within tolerance of the best
        rows, cols = np.nonzero(diff)
        for row in np.unique(rows):
            sel = rows == row
            c = cols[sel]
            chosen = widths[got_idx[row, c]]
            for L in np.unique(chosen):
                m = chosen == L
                s = oracle.snr_of_width(plane_rows[row], float(mu[row]), float(sg[row]), int(L),
                                        ((c[m] + t0) * stride).astype(np.int64))
                bad = ~(np.abs(s - ref_snr[row, c[m]]) <= tol[row, c[m]])
                assert not bad.any(), (
                    f"{what}: near-tie width {L} at row {row} sample {t0 + c[m][bad][0]} has oracle SNR "
                    f"{s[bad][0]!r}, best {ref_snr[row, c[m]][bad][0]!r}")
                n_checked += int(m.sum())
    return ParityStats(int(ref_snr.size), worst, n_diff, n_checked)


def assert_parity_table(oracle, plane_rows: np.ndarray, mu, sigma_w, widths, seps, got_snr, got_idx,
                        ref_snr, ref_idx, ref_second, what: str = "") -> ParityStats:
    """The same rule for runs with a standard deviation per (row, width) (sigma_w [r, n_w], row f1) and,
    optionally, a boxcar separation per width (seps, row f2): references from oracle.spd_direct_sw /
    oracle.spd_grid_sw over whole rows.  A near-tie is settled by the oracle's SNR of the chosen width
    alone (one-width run of the same oracle function)."""
    got_snr = np.asarray(got_snr)
    got_idx = np.asarray(got_idx)
    assert got_snr.shape == ref_snr.shape == got_idx.shape == ref_idx.shape, what
    r, n_t = ref_snr.shape
    widths = [int(w) for w in widths]
    seps = [1] * len(widths) if seps is None else [int(v) for v in seps]
    mu = np.broadcast_to(np.asarray(mu, dtype=np.float64), (r,))
    sigma_w = np.asarray(sigma_w, dtype=np.float64).reshape(r, len(widths))
    nofit = ref_idx < 0
    if nofit.any():
        assert np.all(np.isneginf(got_snr[nofit])), f"{what}: expected -inf where no width applies"
        assert np.all(got_idx[nofit] == -1), f"{what}: expected width index -1 where no width applies"
    ok = ~nofit
    assert np.all(np.isfinite(got_snr[ok])), f"{what}: non-finite SNR from the CUDA path"
    tol = snr_tolerance(np.where(ok, ref_snr, 0.0))
    err = np.where(ok, np.abs(got_snr.astype(np.float64) - np.where(ok, ref_snr, 0.0)), 0.0)
    ratio = err / tol
    worst = float(ratio.max()) if ratio.size else 0.0
    if worst > 1.0:
        i = np.unravel_index(int(np.argmax(ratio)), ratio.shape)
        raise AssertionError(f"{what}: SNR mismatch at row {i[0]} sample {i[1]}: cuda {got_snr[i]!r} oracle "
                             f"{ref_snr[i]!r} (err/tol = {worst:.3g}; {int((ratio > 1).sum())} samples out)")
    assert np.all((got_idx[ok] >= 0) & (got_idx[ok] < len(widths))), f"{what}: width index out of range"
    diff = ok & (got_idx != ref_idx)
    n_diff = int(diff.sum())
    n_checked = 0
    if n_diff:
        with np.errstate(invalid="ignore"):   # -inf - -inf where no width fits: those samples are not in `diff`
            gap = ref_snr - ref_second
        decisive = diff & (gap > tol)
        if decisive.any():
            i = tuple(np.argwhere(decisive)[0])
            raise AssertionError(f"{what}: width index mismatch at row {i[0]} sample {i[1]} where the oracle's top "
                                 f"two differ by {gap[i]:.3g} > tol: cuda {got_idx[i]} oracle {ref_idx[i]}")
        for k in np.unique(got_idx[diff]):
            one = oracle.spd_grid_sw(plane_rows, mu, sigma_w[:, k:k + 1], [widths[k]], [seps[k]])[0]
            m = diff & (got_idx == k)
            bad = m & ~(np.abs(one - ref_snr) <= tol)
            assert not bad.any(), (f"{what}: near-tie width {widths[k]} at {tuple(np.argwhere(bad)[0])} is not within "
                                   f"tolerance of the best (or not on its grid)")
            n_checked += int(m.sum())
    return ParityStats(int(ref_snr.size), worst, n_diff, n_checked)
