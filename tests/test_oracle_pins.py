"""Pins for the CPU oracle (oracle/spd_oracle.c): each test checks it against
something other than itself - a closed form from the paper, a library routine
on a special case, an invariant, or brute force written out in this file."""
import math

import numpy as np
import pytest

from oracle import formulas as F
from workloads import get_workload, make_plane_numpy, make_pulse_only_plane_numpy


def _single_pulse_row(n_t, t0, S, snr_t):
    x = np.zeros(n_t, dtype=np.float32)
    x[t0:t0 + S] = np.float32(snr_t / math.sqrt(S))
    return x


def _closed_form_single_pulse(n_t, t0, S, amp, widths):
    """eq. (22): SNR_L[n] = d_s A / sqrt(L) with d_s the overlap of
    [n, n+L) and [t0, t0+S); no summation anywhere."""
    n = np.arange(n_t)[:, None].astype(np.int64)
    L = np.asarray(widths, dtype=np.int64)[None, :]
    ov = np.minimum(n + L, t0 + S) - np.maximum(n, t0)
    ov = np.clip(ov, 0, None).astype(np.float64)
    snr = ov * amp / np.sqrt(L.astype(np.float64))
    snr[(n + L) > n_t] = -np.inf                      # valid windows only (A3)
    return snr                                        # [n_t, n_w]


# --- P6: whole-plane closed form ------------------------------------------------------

@pytest.mark.parametrize("S,t0", [(1, 40), (3, 17), (7, 100), (20, 100), (45, 60), (64, 0), (33, 190)])
@pytest.mark.parametrize("kind", ["POW2", "ALL", "IGRID1", "RANDOM"])
def test_single_pulse_plane_matches_eq22(oracle_lib, S, t0, kind):
    n_t = 256
    rng = np.random.default_rng(S * 1000 + t0)
    widths = {"POW2": F.widths_pow2(64), "ALL": F.widths_all(64), "IGRID1": F.widths_igrid(1, 64),
              "RANDOM": sorted(set(int(v) for v in rng.integers(1, 90, size=9)))}[kind]
    x = _single_pulse_row(n_t, t0, S, 10.0)
    amp = float(x[t0])
    want = _closed_form_single_pulse(n_t, t0, S, amp, widths)
    snr, idx, sec = oracle_lib.spd_direct(x, 0.0, 1.0, widths)
    assert np.allclose(snr[0], want.max(axis=1), rtol=1e-12, atol=1e-12)
    # arg-max: first (smallest-width) maximum of the closed form, where it is unique to 1e-9
    srt = np.sort(want, axis=1)
    with np.errstate(invalid="ignore"):
        unique = (srt[:, -1] - srt[:, -2]) > 1e-9 if want.shape[1] > 1 else np.ones(n_t, bool)
    assert np.array_equal(idx[0][unique], want.argmax(axis=1)[unique])
    if want.shape[1] > 1:
        assert np.allclose(sec[0][unique], srt[:, -2][unique], rtol=1e-12, atol=1e-12)
    # outside any window touching the pulse everything is exactly zero -> smallest width wins the tie (A4)
    far = np.arange(n_t) > t0 + S
    far &= np.arange(n_t) + widths[0] <= n_t
    assert np.all(snr[0][far] == 0.0) and np.all(idx[0][far] == 0)
    # prefix-difference oracle agrees
    snr_b, idx_b, _ = oracle_lib.spd_prefix(x, 0.0, 1.0, widths)
    assert np.allclose(snr_b, snr, rtol=0, atol=1e-9)


# --- P7: the paper's worked example (Fig. 17) ----------------------------------------

def test_fig17_worked_example(oracle_lib, paper_pins):
    p = paper_pins["fig17_example"]
    widths = F.widths_all(64)
    for snr_t in p["snr"]:
        x = _single_pulse_row(512, p["pulse_start"], p["pulse_width"], float(snr_t))
        snr, idx, _ = oracle_lib.spd_direct(x, 0.0, 1.0, widths)
        n_best = int(np.argmax(snr[0]))
        L_best = widths[int(idx[0][n_best])]
        assert L_best == p["detected_width"]
        assert n_best == p["pulse_start"]                              # start-aligned (A2) ...
        assert n_best + L_best // 2 == p["detected_centre"]            # ... whose centre is sample 110
        assert snr[0][n_best] == pytest.approx(float(snr_t), rel=1e-6)  # eq. (6): matched boxcar returns C


# --- P8: special cases that reduce to a library routine ------------------------------

def test_width_one_is_eq3(oracle_lib):
    rng = np.random.default_rng(3)
    x = rng.standard_normal((4, 300)).astype(np.float32)
    mu = np.array([0.1, -0.2, 0.0, 1.5])
    sg = np.array([1.0, 2.0, 0.5, 3.0])
    snr, idx, sec = oracle_lib.spd_direct(x, mu, sg, [1])
    assert np.allclose(snr, (x.astype(np.float64) - mu[:, None]) / sg[:, None], rtol=1e-14, atol=1e-14)
    assert np.all(idx == 0) and np.all(np.isneginf(sec))


@pytest.mark.parametrize("L", [2, 5, 16, 37])
def test_single_width_is_numpy_convolve(oracle_lib, L):
    rng = np.random.default_rng(L)
    x = rng.standard_normal(400).astype(np.float32)
    mu, sg = 0.25, 1.7
    snr, idx, _ = oracle_lib.spd_direct(x, mu, sg, [L])
    box = np.convolve(x.astype(np.float64), np.ones(L), mode="valid")     # X_L[n], n = 0..n_t-L
    want = (box - L * mu) / (math.sqrt(L) * sg)
    assert np.allclose(snr[0][:400 - L + 1], want, rtol=1e-12, atol=1e-12)
    assert np.all(np.isneginf(snr[0][400 - L + 1:])) and np.all(idx[0][400 - L + 1:] == -1)   # A3
    s2 = oracle_lib.snr_of_width(x, mu, sg, L, np.arange(400 - L + 1))
    assert np.allclose(s2, want, rtol=1e-12, atol=1e-12)


def test_row_stats_is_numpy_mean_std(oracle_lib):
    rng = np.random.default_rng(11)
    x = (rng.standard_normal((5, 1000)) * 2.0 + 3.0).astype(np.float32)
    mu, sg = oracle_lib.row_stats(x)
    x64 = x.astype(np.float64)
    assert np.allclose(mu, x64.mean(axis=1), rtol=1e-13)
    assert np.allclose(sg, x64.std(axis=1, ddof=0), rtol=1e-12)


# --- reading A14: mean / sigma with point-wise outlier rejection -----

def test_clipped_stats_zero_passes_is_plain_stats(oracle_lib):
    rng = np.random.default_rng(12)
    x = (rng.standard_normal((4, 5000)) * 1.7 - 0.4).astype(np.float32)
    mu0, sg0 = oracle_lib.row_stats(x)
    mu, sg = oracle_lib.row_stats_clipped(x, 2.0, 0)
    assert np.array_equal(mu, mu0) and np.array_equal(sg, sg0)


def test_clipped_stats_two_valued_row_with_outliers_exact(oracle_lib):
    """A row of +-1 (mean 0, sigma 1 exactly) plus k outliers of height V: the plain estimate is
    (kV/n, sqrt(...)) in closed form; one 3-sigma rejection removes exactly the outliers and gives
    (0, 1); further passes change nothing."""
    n, k, V = 4000, 8, 50.0
    row = np.tile(np.array([1.0, -1.0], dtype=np.float32), n // 2)
    pos = np.arange(k) * 401 + 7
    row_out = row.copy()
    base_sum = float(row.sum()) - float(row[pos].sum())
    row_out[pos] = V
    x = np.stack([row, row_out])
    mu, sg = oracle_lib.row_stats_clipped(x, 3.0, 0)
    m1 = (base_sum + k * V) / n
    v1 = ((n - k) * 1.0 + k * V * V) / n - m1 * m1
    assert mu[0] == 0.0 and sg[0] == 1.0
    assert abs(mu[1] - m1) < 1e-6 and abs(sg[1] - math.sqrt(v1)) < 1e-5
    assert abs(m1) + 3.0 * math.sqrt(v1) < V  # the outliers are beyond 3 sigma of the plain estimate
    for passes in (1, 2, 5):
        mu, sg = oracle_lib.row_stats_clipped(x, 3.0, passes)
        kept_mean = base_sum / (n - k)
        kept_sigma = math.sqrt(1.0 - kept_mean * kept_mean)
        assert mu[0] == 0.0 and sg[0] == 1.0
        assert abs(mu[1] - kept_mean) < 1e-7 and abs(sg[1] - kept_sigma) < 1e-7


def test_clipped_stats_truncated_normal_variance(oracle_lib):
    """One rejection pass at c sigma on N(0,1) data leaves a normal truncated at +-c:
    variance 1 - 2 c phi(c) / (2 Phi(c) - 1) (textbook)."""
    rng = np.random.default_rng(13)
    x = rng.standard_normal((2, 1 << 20)).astype(np.float32)
    for c in (2.0, 3.0):
        mu, sg = oracle_lib.row_stats_clipped(x, c, 1)
        phi = math.exp(-0.5 * c * c) / math.sqrt(2.0 * math.pi)
        Phi = 0.5 * (1.0 + math.erf(c / math.sqrt(2.0)))
        want = math.sqrt(1.0 - 2.0 * c * phi / (2.0 * Phi - 1.0))
        assert np.all(np.abs(sg - want) < 4e-3) and np.all(np.abs(mu) < 4e-3)


def test_clipped_stats_rejection_is_monotone_and_affine(oracle_lib):
    rng = np.random.default_rng(14)
    x = rng.standard_normal((3, 20000)).astype(np.float32)
    x[1, 5000:5200] += 30.0   # a strong pulse
    sgs = [oracle_lib.row_stats_clipped(x, 2.5, p)[1] for p in range(4)]
    for a, b in zip(sgs, sgs[1:]):
        assert np.all(b <= a + 1e-12)              # rejecting outliers never raises sigma
    assert sgs[0][1] > 2.0 and abs(sgs[3][1] - sgs[3][0]) < 0.05  # the pulse is gone after a few passes
    # scaling by a power of two is exact in float32 and in double: the kept sets are the same
    mu, sg = oracle_lib.row_stats_clipped(x, 2.5, 2)
    mu2, sg2 = oracle_lib.row_stats_clipped((x * np.float32(4.0)), 2.5, 2)
    assert np.array_equal(mu2, 4.0 * mu) and np.array_equal(sg2, 4.0 * sg)


def test_clipped_stats_everything_rejected_keeps_estimate(oracle_lib):
    x = np.array([[0.0, 0.0, 10.0, 10.0]], dtype=np.float32)  # mean 5, sigma 5: clip 0.5 rejects all
    mu, sg = oracle_lib.row_stats_clipped(x, 0.5, 3)
    assert mu[0] == 5.0 and sg[0] == 5.0


def test_clipped_stats_until_convergence(oracle_lib):
    """PAPER.md:726 "This is repeated until convergence".  (a) The two-valued row with outliers: pass 1
    removes exactly the outliers, pass 2 changes nothing, so the iteration stops after 2 rejection passes
    whatever the pass limit; a row without outliers stops after 1.  (b) On N(0,1) data the fixed point of
    sigma -> sigma_trunc(clip * sigma) is the root of s^2 = 1 - 2 t phi(t) / (2 Phi(t) - 1), t = clip * s
    (variance of a normal truncated at +-t, textbook), found here by iterating the formula."""
    n, k, V = 4000, 8, 50.0
    row = np.tile(np.array([1.0, -1.0], dtype=np.float32), n // 2)
    row_out = row.copy()
    row_out[np.arange(k) * 401 + 7] = V
    x = np.stack([row, row_out])
    mu, sg, n_pass, _ = oracle_lib.row_stats_clipped(x, 3.0, 50, rel_tol=0.0, details=True)
    assert list(n_pass) == [1, 2] and sg[0] == 1.0 and abs(sg[1] - 1.0) < 1e-5
    mu5, sg5 = oracle_lib.row_stats_clipped(x, 3.0, 2)                 # the same two passes, counted by the caller
    assert np.array_equal(mu, mu5) and np.array_equal(sg, sg5)
    rng = np.random.default_rng(15)
    y = rng.standard_normal((2, 1 << 20)).astype(np.float32)
    clip = 2.0
    mu, sg, n_pass, _ = oracle_lib.row_stats_clipped(y, clip, 200, rel_tol=1e-7, details=True)
    s = 1.0
    for _ in range(500):
        t = clip * s
        phi = math.exp(-0.5 * t * t) / math.sqrt(2.0 * math.pi)
        Phi = 0.5 * (1.0 + math.erf(t / math.sqrt(2.0)))
        s = math.sqrt(1.0 - 2.0 * t * phi / (2.0 * Phi - 1.0))
    assert np.all(np.abs(sg - s) < 6e-3) and np.all(n_pass < 200) and np.all(n_pass > 5)
    # a looser tolerance stops earlier and lands between the first pass and the fixed point
    _, sg_loose, n_loose, _ = oracle_lib.row_stats_clipped(y, clip, 200, rel_tol=1e-2, details=True)
    _, sg_one = oracle_lib.row_stats_clipped(y, clip, 1)
    assert np.all(n_loose < n_pass) and np.all(sg_loose <= sg_one + 1e-12) and np.all(sg_loose >= sg - 1e-12)


def test_clipped_stats_border_count(oracle_lib):
    """n_border counts the samples within border_eps * sigma of the rejection limit, per pass: the row
    (-1, +1) x 8 has mean 0, sigma 1; with clip 1 all sixteen samples sit exactly on the limit in every
    pass (and are kept: '<='); with clip 2 none is within 1e-3."""
    x = np.tile(np.array([-1.0, 1.0], dtype=np.float32), 8)[None, :]
    mu, sg, n_pass, n_border = oracle_lib.row_stats_clipped(x, 1.0, 3, border_eps=1e-3, details=True)
    assert mu[0] == 0.0 and sg[0] == 1.0 and n_pass[0] == 3 and n_border[0] == 3 * 16
    _, _, _, n_border = oracle_lib.row_stats_clipped(x, 2.0, 3, border_eps=1e-3, details=True)
    assert n_border[0] == 0


# --- sec. 4.3: other pulse shapes (reading A15) ---------------------

def test_gaussian_pulse_worked_example(oracle_lib, paper_pins):
    """The ideal algorithm (all widths) on a zero plane with one Gaussian pulse of 20 samples, C = 16:
    best boxcar 11 samples wide, 4 or 5 samples late, RSNR above C."""
    from workloads.generate import pulse_profile
    pin = paper_pins["gaussian_pulse_example"]
    S, C, t0 = pin["pulse_width"], pin["C"], 100
    x = np.zeros((1, 400), dtype=np.float32)
    x[0, t0:t0 + S] += pulse_profile("gauss", S, C).astype(np.float32)
    assert abs(float(x[0].sum()) / math.sqrt(S) - C) < 1e-4           # boxcar of the signal width gives C
    widths = list(range(1, 2 * S + 1))
    snr, idx, _ = oracle_lib.spd_direct(x, 0.0, 1.0, widths)
    n = int(np.argmax(snr[0]))
    assert widths[idx[0, n]] == pin["detected_width"]
    assert (n - t0) in pin["time_delay"]
    assert snr[0, n] > C


def test_gaussian_pulse_width_error_and_recovered_power(oracle_lib, paper_pins):
    """Wide Gaussian pulses: width under-estimated by about 40 %, about 85 % of the power summed."""
    from workloads.generate import pulse_profile
    pin = paper_pins["gaussian_pulse_example"]
    for S in (100, 200):
        x = np.zeros((1, 4 * S), dtype=np.float32)
        x[0, S:2 * S] += pulse_profile("gauss", S, pin["C"]).astype(np.float32)
        widths = list(range(1, S + 1))
        snr, idx, _ = oracle_lib.spd_direct(x, 0.0, 1.0, widths)
        n = int(np.argmax(snr[0]))
        L = widths[idx[0, n]]
        assert abs((L - S) / S - pin["width_error"]) < 0.02
        assert abs(float(x[0, n:n + L].sum() / x[0].sum()) - pin["recovered_power"]) < 0.01


# --- P9: brute force written out here, tiny planes ------------------------------------

def _brute(x, mu, sg, widths):
    n_dm, n_t = x.shape
    snr = np.full((n_dm, n_t), -np.inf)
    idx = np.full((n_dm, n_t), -1, dtype=np.int32)
    for d in range(n_dm):
        for n in range(n_t):
            for k, L in enumerate(widths):
                if n + L > n_t:
                    continue
                X = 0.0
                for j in range(L):
                    X += float(x[d, n + j])
                s = (X - L * mu[d]) / (math.sqrt(L) * sg[d])
                if s > snr[d, n]:
                    snr[d, n] = s
                    idx[d, n] = k
    return snr, idx


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_brute_force_tiny_planes(oracle_lib, seed):
    rng = np.random.default_rng(seed)
    x = rng.standard_normal((3, 50)).astype(np.float32)
    x[1, 20:27] += 2.0
    mu = rng.normal(0, 0.1, 3)
    sg = rng.uniform(0.5, 2.0, 3)
    widths = sorted(set(int(v) for v in rng.integers(1, 30, size=6)))
    want_snr, want_idx = _brute(x, mu, sg, widths)
    for fn in (oracle_lib.spd_direct, oracle_lib.spd_prefix):
        snr, idx, _ = fn(x, mu, sg, widths)
        assert np.allclose(snr, want_snr, rtol=1e-12, atol=1e-12)
        assert np.array_equal(idx, want_idx)


# --- P10/P11: closed forms that catch index, tail and scaling mistakes ----------------

def test_constant_offset_closed_form(oracle_lib):
    n_t, mu, sg, a = 200, 1.25, 0.5, 0.75
    widths = [1, 2, 4, 7, 16, 50]
    x = np.full(n_t, mu + a, dtype=np.float32)
    snr, idx, _ = oracle_lib.spd_direct(x, mu, sg, widths)
    for n in range(n_t):
        fit = [k for k, L in enumerate(widths) if n + L <= n_t]
        k = fit[-1]                                       # SNR_L = a sqrt(L)/sigma grows with L
        assert idx[0][n] == k
        assert snr[0][n] == pytest.approx(a * math.sqrt(widths[k]) / sg, rel=1e-12)
    snr_neg, idx_neg, _ = oracle_lib.spd_direct(np.full(n_t, mu - a, dtype=np.float32), mu, sg, widths)
    assert np.all(idx_neg == 0) and np.allclose(snr_neg, -a / sg)


def test_tail_rule_without_width_one(oracle_lib):
    x = np.ones(40, dtype=np.float32)
    snr, idx, sec = oracle_lib.spd_direct(x, 0.0, 1.0, [4, 8])
    assert np.all(np.isneginf(snr[0][37:])) and np.all(idx[0][37:] == -1)
    assert np.all(idx[0][33:37] == 0) and np.all(np.isneginf(sec[0][33:37]))
    assert np.all(idx[0][:33] == 1)


def test_ramp_closed_form(oracle_lib):
    n_t = 120
    widths = [1, 3, 8, 20]
    x = np.arange(n_t, dtype=np.float32)
    snr, idx, _ = oracle_lib.spd_direct(x, 0.0, 1.0, widths)
    for n in range(n_t):
        vals = [(L * n + L * (L - 1) / 2) / math.sqrt(L) if n + L <= n_t else -math.inf for L in widths]
        assert snr[0][n] == pytest.approx(max(vals), rel=1e-13)
        assert idx[0][n] == int(np.argmax(vals))


def test_unit_impulse_closed_form(oracle_lib):
    n_t, t0, A = 128, 70, 5.0
    widths = [1, 2, 4, 8, 16, 32]
    x = np.zeros(n_t, dtype=np.float32)
    x[t0] = A
    snr, idx, _ = oracle_lib.spd_direct(x, 0.0, 1.0, widths)
    for n in range(n_t):
        if n > t0 or t0 - n + 1 > widths[-1]:
            assert snr[0][n] == 0.0 and idx[0][n] == 0
        else:
            k = next(k for k, L in enumerate(widths) if L >= t0 - n + 1)
            assert idx[0][n] == k and snr[0][n] == pytest.approx(A / math.sqrt(widths[k]))


# --- P12: invariants ---------------------------------------------------------------------

def test_affine_invariance_and_superset_monotonicity(oracle_lib):
    rng = np.random.default_rng(5)
    x = np.round(rng.standard_normal((2, 600)) * 1024.0) / 1024.0     # exact in float32, and so is 4x + 8
    widths = F.widths_pow2(64)
    snr, idx, _ = oracle_lib.spd_direct(x.astype(np.float32), 0.0, 1.0, widths)
    alpha, beta = 4.0, 8.0                       # powers of two: exact in float32
    snr2, idx2, _ = oracle_lib.spd_direct((alpha * x.astype(np.float32) + beta).astype(np.float32), beta, alpha, widths)
    assert np.allclose(snr2, snr, rtol=1e-12, atol=1e-12) and np.array_equal(idx2, idx)
    full, idx_full, _ = oracle_lib.spd_direct(x.astype(np.float32), 0.0, 1.0, F.widths_all(64))
    assert np.all(full >= snr - 1e-12)
    all_w = F.widths_all(64)
    chosen = np.array(all_w)[idx_full]
    in_set = np.isin(chosen, widths)
    assert np.allclose(full[in_set], snr[in_set], rtol=1e-12)


def test_time_shift_equivariance(oracle_lib):
    rng = np.random.default_rng(6)
    x = rng.standard_normal(700).astype(np.float32)
    widths = [1, 3, 8, 21]
    a, ia, _ = oracle_lib.spd_direct(x, 0.0, 1.0, widths)
    b, ib, _ = oracle_lib.spd_direct(x[50:], 0.0, 1.0, widths)
    assert np.array_equal(a[0][50:], b[0]) and np.array_equal(ia[0][50:], ib[0])
    # windowed evaluation equals the slice of the full evaluation
    c, ic, _ = oracle_lib.spd_direct(x, 0.0, 1.0, widths, t0=123, t1=456)
    assert np.array_equal(c[0], a[0][123:456]) and np.array_equal(ic[0], ia[0][123:456])


# --- P13: white-noise statistics (eq. 5) --------------------------------------------------

def test_white_noise_per_width_statistics(oracle_lib):
    rng = np.random.default_rng(13)
    n_t = 1 << 18
    x = rng.standard_normal(n_t).astype(np.float32)
    for L in (1, 4, 32, 256):
        s = oracle_lib.snr_of_width(x, 0.0, 1.0, L, np.arange(0, n_t - L, L))   # non-overlapping windows
        n_ind = s.size
        assert abs(s.mean()) < 5.0 / math.sqrt(n_ind)
        assert abs(s.var() - 1.0) < 5.0 * math.sqrt(2.0 / n_ind)


# --- P14: eq. (24) on the noise-free twin of a workload ----------------------------------

@pytest.mark.parametrize("cfg,n_dm,n_t,n_pulses", [(1, 8, 4096, 8), (2, 8, 8192, 16)])
def test_noise_free_twin_recovers_eq24(oracle_lib, cfg, n_dm, n_t, n_pulses):
    w = get_workload(cfg).scaled(n_dm, n_t, n_pulses)
    plane, pulses = make_pulse_only_plane_numpy(w)
    widths = F.width_set(w.width_kind, w.width_param, w.max_width)
    snr, idx, _ = oracle_lib.spd_prefix(plane, 0.0, 1.0, widths)
    ratios = []
    for p in pulses:
        others = [q for q in pulses if q is not p and q.dm == p.dm
                  and q.t0 < p.t0 + p.width + w.max_width and p.t0 < q.t0 + q.width + w.max_width]
        if others:
            continue                                     # overlapping neighbourhoods: not an isolated pulse
        lo, hi = max(0, p.t0 - w.max_width), min(n_t, p.t0 + p.width)
        r = snr[p.dm, lo:hi].max() / p.snr_t
        assert r == pytest.approx(F.rsnr_max(p.width, widths), rel=1e-6)
        ratios.append((p.width, r))
    assert len(ratios) >= n_pulses // 2
    mean_loss = 1.0 - sum(r for _, r in ratios) / len(ratios)
    assert mean_loss == pytest.approx(F.mean_loss_over_widths([s for s, _ in ratios], widths), abs=1e-6)


# --- A vs B on a config-1-shaped plane ----------------------------------------------------

def test_direct_and_prefix_agree_on_config1_shape(oracle_lib):
    w = get_workload(1).scaled(4, 2048, 4)
    plane, _ = make_plane_numpy(w)
    widths = F.width_set(w.width_kind, w.width_param, w.max_width)
    a, ia, sa = oracle_lib.spd_direct(plane, 0.0, 1.0, widths)
    b, ib, sb = oracle_lib.spd_prefix(plane, 0.0, 1.0, widths)
    assert np.max(np.abs(a - b)) <= 1e-9
    clear = (a - sa) > 1e-9
    assert np.array_equal(ia[clear], ib[clear])


# --- candidate rule (reading A9): closed form on an isolated pulse ----------------------

def test_candidates_isolated_pulse_first_sample_of_plateau(oracle_lib):
    n_t, t0, S, snr_t = 400, 150, 20, 10.0
    widths = F.widths_pow2(64)
    x = _single_pulse_row(n_t, t0, S, snr_t)
    snr, idx, _ = oracle_lib.spd_direct(x, 0.0, 1.0, widths)
    # eq. (22): width 16 fits inside the pulse at n = t0..t0+4 -> five equal maxima of 16 A / 4
    peak = 16 * (snr_t / math.sqrt(S)) / 4.0
    assert np.allclose(snr[0][t0:t0 + 5], peak, rtol=1e-7) and snr[0].max() == pytest.approx(peak, rel=1e-7)
    count, c_dm, c_t, c_snr, c_w = oracle_lib.find_candidates(snr.astype(np.float32), idx, 0.9 * peak)
    assert count == 1 and c_dm[0] == 0 and c_t[0] == t0 and widths[c_w[0]] == 16
    assert c_snr[0] == pytest.approx(peak, rel=1e-6)


def test_candidates_rule_edges_and_capacity(oracle_lib):
    y = np.array([[7, 7, 3, 8, 8, 8, 2, 9],
                  [1, 2, 3, 4, 5, 6, 7, 8]], dtype=np.float32)
    wid = np.zeros_like(y, dtype=np.int32)
    count, c_dm, c_t, c_snr, _ = oracle_lib.find_candidates(y, wid, 6.0)
    # row 0: n=0 (7 > -inf, >= 7), n=3 (first of the 8-plateau), n=7 (9 > 2, right edge); row 1: n=7
    assert count == 4
    assert list(zip(c_dm.tolist(), c_t.tolist())) == [(0, 0), (0, 3), (0, 7), (1, 7)]
    count2, c_dm2, *_ = oracle_lib.find_candidates(y, wid, 6.0, capacity=2)
    assert count2 == 4 and len(c_dm2) == 2


# --- f2: per-width boxcar separation (the paper's decimated grids), oracle_spd_grid -----

def _slid_pulses(S, n_shifts, n_t, t_first, snr_t=16.0):
    """One noise-free row per shift of a width-S pulse (the paper's measurement method,
    PAPER.md:492-494; C = 16)."""
    x = np.zeros((n_shifts, n_t), dtype=np.float32)
    for s in range(n_shifts):
        x[s] = _single_pulse_row(n_t, t_first + s, S, snr_t)
    return x


@pytest.mark.parametrize("L,Ls", [(5, 3), (8, 8), (8, 4), (8, 2), (16, 16), (12, 4), (7, 7), (9, 2)])
def test_grid_single_width_recovers_eq30_and_eq23(oracle_lib, L, Ls):
    """Boxcars of one width L at every Ls-th sample: over all pulse shifts the best response
    per row has minimum eq. (30) and maximum eq. (23)."""
    for S in list(range(1, 3 * L + 2 * Ls, 2)) + [L, L + Ls]:
        n_t = 6 * (L + Ls) + 4 * S
        t_first = (2 * (L + Ls) + Ls - 1) // Ls * Ls          # a grid point, far from both ends
        x = _slid_pulses(S, Ls, n_t, t_first)
        snr, idx, _ = oracle_lib.spd_grid(x, 0.0, 1.0, [L], [Ls])
        per_shift = snr.max(axis=1) / 16.0
        assert per_shift.min() == pytest.approx(F.rsnr_min_single(S, L, Ls), abs=1e-6), (S, L, Ls)
        assert per_shift.max() == pytest.approx(F.rsnr_max_single(S, L), abs=1e-6), (S, L, Ls)
        off_grid = np.arange(n_t) % Ls != 0
        assert np.all(np.isneginf(snr[:, off_grid])) and np.all(idx[:, off_grid] == -1)


@pytest.mark.parametrize("name", ["DIT", "BOXDIT4", "BOXDIT8", "IGRID1x4"])
def test_grid_width_sets_lie_between_eq31_and_eq24(oracle_lib, name):
    """The bound test of PAPER.md:152, 512 on the paper's grids: measured worst response >=
    eq. (31), best == eq. (24); and both equal the shift scan written out in formulas.py."""
    widths, sep = {"DIT": (F.widths_pow2(64), lambda L: L),
                   "BOXDIT4": (F.widths_boxdit(4, 60), F.boxdit_separation(4)),
                   "BOXDIT8": (F.widths_boxdit(8, 56), F.boxdit_separation(8)),
                   "IGRID1x4": (F.widths_igrid(1, 64), F.igrid_separation(4))}[name]
    seps = [sep(L) for L in widths]
    period = max(seps)                                        # separations are powers of two
    for S in (1, 2, 3, 5, 7, 9, 12, 17, 20, 31, 33, 45, 64, 70):
        n_t = 4 * 64 + 2 * period + 2 * S
        t_first = 2 * period
        x = _slid_pulses(S, period, n_t, t_first)
        snr, _, _ = oracle_lib.spd_grid(x, 0.0, 1.0, widths, seps)
        per_shift = snr.max(axis=1) / 16.0
        lo, hi, mean = F.brute_force_response(S, widths, sep)
        assert per_shift.min() == pytest.approx(lo, abs=1e-6) and per_shift.max() == pytest.approx(hi, abs=1e-6)
        assert per_shift.mean() == pytest.approx(mean, abs=1e-6)
        assert per_shift.min() >= F.rsnr_min(S, widths, sep) - 1e-6
        assert per_shift.max() == pytest.approx(F.rsnr_max(S, widths), abs=1e-6)


def test_grid_paper_example_positions(oracle_lib):
    """with L_max = 4, widths 1..4 are calculated at every point, 6, 8, 10, 12 at
    every second point (and 16, 20, 24, 28 at every fourth).  On a constant offset
    SNR_L = a sqrt(L) / sigma grows with L, so the winner is the largest width whose grid
    contains n and whose window fits."""
    n_t, mu, sg, a = 131, 0.5, 2.0, 1.5
    widths = F.widths_boxdit(4, 28)
    assert widths == [1, 2, 3, 4, 6, 8, 10, 12, 16, 20, 24, 28]
    sepf = F.boxdit_separation(4)
    seps = [sepf(L) for L in widths]
    assert seps == [1, 1, 1, 1, 2, 2, 2, 2, 4, 4, 4, 4]
    x = np.full(n_t, mu + a, dtype=np.float32)
    snr, idx, _ = oracle_lib.spd_grid(x, mu, sg, widths, seps)
    for n in range(n_t):
        ok = [k for k, (L, s) in enumerate(zip(widths, seps)) if n % s == 0 and n + L <= n_t]
        assert idx[0][n] == ok[-1]
        assert snr[0][n] == pytest.approx(a * math.sqrt(widths[ok[-1]]) / sg, rel=1e-12)
    assert idx[0][1] == 3 and idx[0][2] == 7 and idx[0][4] == 11 and idx[0][6] == 7


def test_grid_with_unit_separations_is_direct(oracle_lib):
    rng = np.random.default_rng(5)
    x = rng.standard_normal((3, 300)).astype(np.float32)
    widths = F.widths_igrid(1, 64)
    a = oracle_lib.spd_direct(x, 0.1, 1.3, widths)
    b = oracle_lib.spd_grid(x, 0.1, 1.3, widths, [1] * len(widths))
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])


# --- f1 (second half): standard deviation per width from decimations --------

def test_width_sigma_is_numpy_on_hand_decimated_rows(oracle_lib):
    """Powers of two: numpy std of reshape(-1, 2^j).sum(1); a tiny row by hand; intermediate widths
    linear between the neighbouring powers of two; above the last level sqrt(L) from it (eq. 5)."""
    x = np.arange(1, 9, dtype=np.float32)[None, :]                 # 1..8
    sw = oracle_lib.width_sigma(x, [1, 2, 3, 4, 6, 8])
    s1 = np.std(np.arange(1, 9))                                   # 2.2913
    s2 = np.std([3, 7, 11, 15])                                    # sqrt(20)
    s4 = np.std([10, 26])                                          # 8
    assert sw[0, 0] == pytest.approx(s1) and sw[0, 1] == pytest.approx(math.sqrt(20.0))
    assert sw[0, 3] == pytest.approx(8.0)
    assert sw[0, 2] == pytest.approx(0.5 * (s2 + s4))              # L = 3: midway between 2 and 4
    assert sw[0, 4] == pytest.approx(s4 * math.sqrt(6 / 4))        # no level 8 (one element): sqrt law from 4
    assert sw[0, 5] == pytest.approx(s4 * math.sqrt(8 / 4))
    # rows too short for any level with two elements: a single sample has no deviation (numpy agrees)
    one = oracle_lib.width_sigma(np.array([[3.5]], dtype=np.float32), [1])
    assert one[0, 0] == 0.0 == np.std(np.array([3.5]))
    rng = np.random.default_rng(3)
    y = (rng.standard_normal((2, 4096 + 37)) * 2.5 + 7).astype(np.float32)
    widths = [1, 2, 4, 5, 8, 16, 24, 64, 100, 256]
    sw = oracle_lib.width_sigma(y, widths)
    for d in range(2):
        lev = {}
        for j in range(10):
            b = 1 << j
            m = y.shape[1] // b
            lev[b] = np.std(y[d, :m * b].astype(np.float64).reshape(m, b).sum(axis=1))
        for k, L in enumerate(widths):
            lo = 1 << (int(L).bit_length() - 1)
            want = lev[lo] + (lev[2 * lo] - lev[lo]) * (L - lo) / lo
            assert sw[d, k] == pytest.approx(want, rel=1e-12)


def test_width_sigma_white_noise_follows_eq5_and_ar1_follows_the_textbook(oracle_lib):
    """eq. (5): sigma_L = sqrt(L) sigma on white noise.  On an AR(1) series
    x[n] = rho x[n-1] + e[n] the variance of a sum of L samples is
    s^2 [L (1+rho)/(1-rho) - 2 rho (1 - rho^L)/(1-rho)^2] (textbook), i.e. NOT sqrt(L): the case the
    paper's measured sigma is for (Fig. 24)."""
    rng = np.random.default_rng(11)
    n = 1 << 20
    w = rng.standard_normal(n)
    widths = [1, 2, 4, 8, 16, 32, 64]
    sw = oracle_lib.width_sigma(w.astype(np.float32)[None, :], widths)[0]
    for L, s in zip(widths, sw):
        assert s == pytest.approx(math.sqrt(L), rel=4.0 * math.sqrt(L / (2.0 * n)) + 1e-3)
    rho = 0.6
    x = np.empty(n)
    x[0] = w[0] / math.sqrt(1 - rho * rho)
    for i in range(1, n):
        x[i] = rho * x[i - 1] + w[i]
    s2 = 1.0 / (1 - rho * rho)
    sw = oracle_lib.width_sigma(x.astype(np.float32)[None, :], widths)[0]
    for L, s in zip(widths, sw):
        var = s2 * (L * (1 + rho) / (1 - rho) - 2 * rho * (1 - rho ** L) / (1 - rho) ** 2)
        assert s == pytest.approx(math.sqrt(var), rel=0.02), L
    assert sw[-1] > 1.5 * math.sqrt(64) * math.sqrt(s2) * 0.9      # far from the white-noise law


def test_direct_with_white_noise_sigma_table_is_direct(oracle_lib):
    rng = np.random.default_rng(12)
    x = rng.standard_normal((2, 400)).astype(np.float32)
    widths = [1, 2, 3, 8, 20]
    sg = np.array([1.5, 0.7])
    table = sg[:, None] * np.sqrt(np.asarray(widths, dtype=np.float64))[None, :]
    a = oracle_lib.spd_direct(x, [0.1, -0.2], sg, widths)
    b = oracle_lib.spd_direct_sw(x, [0.1, -0.2], table, widths)
    assert np.allclose(a[0], b[0], rtol=1e-13, atol=1e-13) and np.array_equal(a[1], b[1])
    # halving one width's sigma doubles that width's SNR only
    table2 = table.copy()
    table2[:, 3] *= 0.5
    only8 = oracle_lib.spd_direct_sw(x, [0.1, -0.2], table2[:, 3:4], [8])
    ref8 = oracle_lib.spd_direct(x, [0.1, -0.2], sg, [8])
    assert np.allclose(only8[0][:, :392], 2.0 * ref8[0][:, :392], rtol=1e-13)


def test_grid_with_sigma_table_reduces_to_grid_and_to_direct_sw(oracle_lib):
    """oracle_spd_grid_sw: the table sqrt(L) sigma reproduces oracle_spd_grid bit for bit (same expression
    evaluated on the same doubles is not guaranteed, so: to 1e-13 and identical indices), separations all 1
    reproduce oracle_spd_direct_sw exactly, and halving one width's sigma doubles that width's SNR on its
    grid only."""
    rng = np.random.default_rng(21)
    x = rng.standard_normal((3, 500)).astype(np.float32)
    x[1, 200:230] += 2.0
    widths = [1, 2, 3, 4, 6, 8, 10, 12, 16, 24]
    seps = [1, 1, 1, 1, 2, 2, 2, 2, 4, 4]
    sg = np.array([1.5, 0.7, 1.0])
    mu = [0.1, -0.2, 0.0]
    table = sg[:, None] * np.sqrt(np.asarray(widths, dtype=np.float64))[None, :]
    a = oracle_lib.spd_grid(x, mu, sg, widths, seps)
    b = oracle_lib.spd_grid_sw(x, mu, table, widths, seps)
    fin = np.isfinite(a[0])
    assert np.array_equal(a[1], b[1]) and np.allclose(a[0][fin], b[0][fin], rtol=1e-13, atol=1e-13)
    rough = rng.uniform(0.5, 2.0, size=table.shape) * table
    c = oracle_lib.spd_direct_sw(x, mu, rough, widths)
    d = oracle_lib.spd_grid_sw(x, mu, rough, widths, [1] * len(widths))
    assert np.array_equal(c[0], d[0]) and np.array_equal(c[1], d[1]) and np.array_equal(c[2], d[2])
    # a single width on a grid: SNR only at multiples of its separation, scaled by 1 / sigma_w
    one = oracle_lib.spd_grid_sw(x, mu, 0.5 * table[:, 8:9], [16], [4])
    ref = oracle_lib.spd_grid(x, mu, sg, [16], [4])
    on = np.arange(500) % 4 == 0
    valid = on & (np.arange(500) + 16 <= 500)
    assert np.allclose(one[0][:, valid], 2.0 * ref[0][:, valid], rtol=1e-13)
    assert np.all(np.isneginf(one[0][:, ~on])) and np.all(one[1][:, ~on] == -1)


# --- f4: 2-D (DM x time) peaks over the 1-D candidates (reading A18) ----

def _cluster_brute(snr, widths, c_dm, c_t, c_w, R):
    """The rule of reading A18 written out with numpy windows."""
    n_dm, n_t = snr.shape
    keep = []
    for d, n, wi in zip(c_dm, c_t, c_w):
        L = int(widths[wi])
        d0, d1 = max(0, d - R), min(n_dm - 1, d + R)
        n0, n1 = max(0, n - L), min(n_t - 1, n + L)
        win = snr[d0:d1 + 1, n0:n1 + 1]
        v = snr[d, n]
        ok = not np.any(win > v)
        if ok:
            dd, nn = np.nonzero(win == v)
            first = min(zip(dd + d0, nn + n0))
            ok = first == (d, n)
        keep.append(ok)
    return np.array(keep, dtype=bool)


def test_cluster_one_pulse_smeared_over_dm_rows_is_one_cluster(oracle_lib):
    """A pulse seen in five neighbouring DM rows with SNR falling away from the middle row, each row a
    plateau with ripples: the 1-D rule (A9) reports several peaks per row, the 2-D rule (A18, dm_radius 1)
    keeps exactly one - the highest sample of the middle row, with its width index."""
    widths = [1, 2, 4, 8, 16, 32]
    n_dm, n_t = 9, 600
    snr = np.full((n_dm, n_t), 0.5, dtype=np.float32)
    wid = np.zeros((n_dm, n_t), dtype=np.int32)
    for d, amp in zip(range(2, 7), [7.0, 9.0, 12.0, 9.5, 6.5]):
        t = np.arange(280, 321)
        snr[d, t] = (amp - 0.02 * np.abs(t - 300) + 0.3 * ((t % 5) == 0)).astype(np.float32)
        wid[d, t] = 5                                   # best width 32
    cnt, c_dm, c_t, c_snr, c_w = oracle_lib.find_candidates(snr, wid, 6.0)
    assert cnt > 10                                     # ripples: many 1-D peaks
    keep = oracle_lib.cluster_candidates(snr, widths, c_dm, c_t, c_w, 1)
    assert keep.sum() == 1
    i = int(np.nonzero(keep)[0][0])
    assert (c_dm[i], c_t[i], c_w[i]) == (4, 300, 5) and c_snr[i] == np.float32(12.3)
    assert np.array_equal(keep, _cluster_brute(snr, widths, c_dm, c_t, c_w, 1))


def test_cluster_separation_ties_and_edges(oracle_lib):
    """Two pulses further apart than the window are two clusters, closer than it one (the larger);
    a pulse two rows away is separate at dm_radius 1 and merged at dm_radius 2; of two equal samples
    inside each other's window the first in (dm, t) order is kept; windows are clipped at the edges."""
    widths = [1, 2, 4, 8, 16]
    n_dm, n_t = 6, 400

    def run(points, R):
        snr = np.zeros((n_dm, n_t), dtype=np.float32)
        wid = np.zeros((n_dm, n_t), dtype=np.int32)
        for d, t, v, wi in points:
            snr[d, t] = v
            wid[d, t] = wi
        cnt, c_dm, c_t, c_snr, c_w = oracle_lib.find_candidates(snr, wid, 5.0)
        assert cnt == len(points)
        keep = oracle_lib.cluster_candidates(snr, widths, c_dm, c_t, c_w, R)
        assert np.array_equal(keep, _cluster_brute(snr, widths, c_dm, c_t, c_w, R))
        return {(int(a), int(b)) for a, b, k in zip(c_dm, c_t, keep) if k}

    assert run([(1, 100, 8.0, 3), (1, 109, 9.0, 3)], 1) == {(1, 100), (1, 109)}   # 9 > width 8: apart
    assert run([(1, 100, 8.0, 3), (1, 108, 9.0, 3)], 1) == {(1, 108)}             # 8 <= 8: one cluster
    assert run([(1, 100, 8.0, 0), (1, 108, 9.0, 4)], 1) == {(1, 100), (1, 108)}   # window = OWN width (1)
    assert run([(1, 100, 8.0, 3), (3, 100, 9.0, 3)], 1) == {(1, 100), (3, 100)}
    assert run([(1, 100, 8.0, 3), (3, 100, 9.0, 3)], 2) == {(3, 100)}
    assert run([(2, 50, 7.0, 2), (2, 53, 7.0, 2), (1, 52, 7.0, 2)], 1) == {(1, 52)}  # ties: first in (dm, t)
    assert run([(0, 0, 6.0, 4), (5, 399, 6.5, 4)], 3) == {(0, 0), (5, 399)}        # clipped windows


def test_cluster_random_planes_match_window_scan(oracle_lib):
    rng = np.random.default_rng(33)
    widths = [1, 2, 3, 5, 8, 13, 21]
    for R in (0, 1, 3):
        snr = rng.standard_normal((12, 700)).astype(np.float32) * 2.0
        snr = np.round(snr * 4) / 4                     # many exact ties
        wid = rng.integers(0, len(widths), size=snr.shape).astype(np.int32)
        cnt, c_dm, c_t, c_snr, c_w = oracle_lib.find_candidates(snr.astype(np.float32), wid, 2.0)
        keep = oracle_lib.cluster_candidates(snr.astype(np.float32), widths, c_dm, c_t, c_w, R)
        assert cnt > 50 and np.array_equal(keep, _cluster_brute(snr, widths, c_dm, c_t, c_w, R))


# --- output separated by iteration (eq. 12; Alg. 1, eq. 13-15) -----------------

def _boxdit_literal(x, mu, sg, l_max, n_iter):
    """Alg. 1 as printed, D = 2, in double: iteration i works on the decimated series x^i
    and on X^{i-1}, the longest boxcar of the iteration before;
        eq. (15)  X_L[n] = X^{i-1}[n] + sum_{j < m} x^i[n_s + j],  n_s = n / D^(i),  L = L_MAX^{i-1} + D^(i) m (eq. 14)
        eq. (13)  x^{i+1}[n - L_max / D] = x^i[D n] + x^i[D n + 1]
    Positions are kept in the iteration's own index q (sample n = 2^i q of the row).  Returns, per iteration,
    (Y^i, m^i) over the points whose windows fit the row, with m the winning 1-based position in the
    iteration's width list, plus the number of points."""
    xi = np.asarray(x, dtype=np.float64) - mu          # x^0, mean removed (eq. 4's numerator, per sample)
    n_t = xi.size
    X_prev = np.zeros(n_t)                             # X^{-1} = 0 at the points of iteration 0
    L_MAX_prev = 0
    out = []
    for i in range(n_iter):
        step = 1 << i
        n_pts = (n_t + step - 1) // step
        Y = np.full(n_pts, -np.inf)
        M = np.full(n_pts, -1, dtype=np.int64)
        X_long = np.zeros(n_pts)
        for q in range(n_pts):
            n = q * step
            acc = X_prev[q]
            for m in range(1, l_max + 1):
                L = L_MAX_prev + step * m                               # eq. (14)
                if n + L > n_t:
                    break
                acc = acc + xi[q + m - 1]                                # eq. (15): one more element of x^i
                snr = acc / (math.sqrt(L) * sg)                          # eq. (4) with eq. (5)
                if snr > Y[q]:
                    Y[q], M[q] = snr, m
                if m == l_max:
                    X_long[q] = acc
        out.append((Y, M, n_pts))
        # eq. (13): x^{i+1}[q'] = x^i[2 q' + l_max] + x^i[2 q' + l_max + 1]; X^i is handed on at every second point
        n_next = (n_t + 2 * step - 1) // (2 * step)
        nxt = np.zeros(n_next + l_max + 2)
        for qn in range(nxt.size):
            a, b = 2 * qn + l_max, 2 * qn + l_max + 1
            nxt[qn] = (xi[a] if a < xi.size else 0.0) + (xi[b] if b < xi.size else 0.0)
        xi = nxt
        X_prev = X_long[::2].copy()
        L_MAX_prev += step * l_max
    return out


@pytest.mark.parametrize("l_max,n_iter,n_t", [(4, 4, 203), (8, 3, 260), (4, 3, 64), (2, 5, 117)])
def test_grid_iter_equals_the_literal_boxdit_algorithm(oracle_lib, l_max, n_iter, n_t):
    """oracle_spd_grid_iter (direct summation of every window of an iteration) against Alg. 1 run step by step
    with eq. (13)'s shifted decimation and eq. (15): the same Y^i, W^i at every point of every iteration."""
    rng = np.random.default_rng(1000 + l_max + n_t)
    x = (rng.standard_normal(n_t) * 1.7 + 0.4).astype(np.float32)
    x[n_t // 3: n_t // 3 + 3 * l_max] += np.float32(2.0)
    mu, sg = 0.4, 1.7
    widths = [((1 << i) - 1) * l_max + (m << i) for i in range(n_iter) for m in range(1, l_max + 1)]
    seps = [1 << i for i in range(n_iter) for _ in range(l_max)]
    assert widths == F.widths_boxdit(l_max, widths[-1])
    its = oracle_lib.grid_iterations(seps)
    assert its == [(i * l_max, (i + 1) * l_max) for i in range(n_iter)]
    lit = _boxdit_literal(x, mu, sg, l_max, n_iter)
    for i, (kb, ke) in enumerate(its):
        snr, idx, _ = oracle_lib.spd_grid_iter(x, mu, sg, widths, seps, kb, ke)
        Y, M, n_pts = lit[i]
        assert snr.shape == (1, n_pts)
        fit = M >= 0
        assert np.array_equal(idx[0] >= 0, fit)
        assert np.array_equal(idx[0][fit], kb + M[fit] - 1)
        assert np.allclose(snr[0][fit], Y[fit], rtol=1e-12, atol=1e-12)
        assert np.all(np.isneginf(snr[0][~fit]))


def test_grid_iter_planes_merge_into_the_grid_plane(oracle_lib):
    """Reading A16: the merged plane of oracle_spd_grid is, at every sample, the maximum over the iterations
    whose grid holds the sample (ties: the earlier iteration, i.e. the smaller width) - for the BoxDIT, DIT and
    IGRID-layer grids."""
    rng = np.random.default_rng(77)
    x = rng.standard_normal((2, 333)).astype(np.float32)
    cases = [
        (F.widths_boxdit(8, 56), F.boxdit_separation(8)),
        ([1 << k for k in range(7)], lambda L: L),
        (F.widths_igrid(1, 64), F.igrid_separation(4)),
    ]
    for widths, sepf in cases:
        seps = [sepf(L) for L in widths]
        ref_snr, ref_idx, _ = oracle_lib.spd_grid(x, 0.2, 1.1, widths, seps)
        snr = np.full(x.shape, -np.inf)
        idx = np.full(x.shape, -1, dtype=np.int32)
        for kb, ke in oracle_lib.grid_iterations(seps):
            s = seps[kb]
            y, w, _ = oracle_lib.spd_grid_iter(x, 0.2, 1.1, widths, seps, kb, ke)
            assert y.shape[1] == (x.shape[1] + s - 1) // s
            better = y > snr[:, ::s]
            snr[:, ::s] = np.where(better, y, snr[:, ::s])
            idx[:, ::s] = np.where(better, w, idx[:, ::s])
        assert np.array_equal(snr, ref_snr) and np.array_equal(idx, ref_idx)


def test_grid_iter_paper_example_closed_form(oracle_lib):
    """PAPER.md:201 ("boxcar filters of width L = 1, 2, 3, 4 are calculated at every point; after decimation,
    boxcar filters of width L = 6, 8, 10, 12 are calculated at every second point and so on") on a constant
    offset a: SNR_L = a sqrt(L) / sigma, so every iteration's winner is its largest width that fits the row."""
    n_t, mu, sg, a = 131, 0.5, 2.0, 1.5
    widths = F.widths_boxdit(4, 28)
    seps = [F.boxdit_separation(4)(L) for L in widths]
    x = np.full(n_t, mu + a, dtype=np.float32)
    for i, (kb, ke) in enumerate(oracle_lib.grid_iterations(seps)):
        s = 1 << i
        snr, idx, sec = oracle_lib.spd_grid_iter(x, mu, sg, widths, seps, kb, ke)
        assert snr.shape == (1, (n_t + s - 1) // s)
        for m in range(snr.shape[1]):
            ok = [k for k in range(kb, ke) if s * m + widths[k] <= n_t]
            if not ok:
                assert idx[0][m] == -1 and np.isneginf(snr[0][m])
                continue
            assert idx[0][m] == ok[-1]
            assert snr[0][m] == pytest.approx(a * math.sqrt(widths[ok[-1]]) / sg, rel=1e-12)
            if len(ok) > 1:
                assert sec[0][m] == pytest.approx(a * math.sqrt(widths[ok[-2]]) / sg, rel=1e-12)
    # iteration 1 holds 6, 8, 10, 12 at samples 0, 2, 4, ...; its point 3 is sample 6
    y1, w1, _ = oracle_lib.spd_grid_iter(x, mu, sg, widths, seps, 4, 8)
    assert w1[0][3] == 7 and y1.shape[1] == 66
