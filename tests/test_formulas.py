"""Pins for oracle/formulas.py: the paper's printed numbers, hand values and a
brute-force scan over pulse shifts that shares no code with eq. (27)-(31)."""
import math

import pytest

from oracle import formulas as F


# --- P3: width-set generators against lists printed in the paper -----------------

def test_boxdit_widths_match_paper_example(paper_pins):
    p = paper_pins["boxdit_example_widths"]
    got = F.widths_boxdit(p["l_max"], 12)
    assert got == p["iteration0"] + p["iteration1"]


def test_igrid_widths_match_table1(paper_pins):
    t = paper_pins["igrid_table1"]
    for depth in (0, 1, 2, 3):
        got = [L for L in F.widths_igrid(depth, 31) if 16 <= L < 32]
        assert got == t[f"depth{depth}"]
    # IG(1) is {2^i, 3*2^(i-1)}
    assert F.widths_igrid(1, 64) == [1, 2, 3, 4, 6, 8, 12, 16, 24, 32, 48, 64]


def test_bd8_reaches_l_end_in_ten_iterations(paper_pins):
    p = paper_pins["bd8_iterations"]
    w = F.widths_boxdit(p["l_max"], p["l_end"])
    assert w[-1] == p["last_width"] == p["l_max"] * (2 ** p["iterations"] - 1)
    assert len(w) == p["l_max"] * p["iterations"]
    # nine iterations are not enough: 8*(2^9-1) = 4088 < 8192 (L_end is the
    # nearest boxcar to S_end)
    assert p["l_max"] * (2 ** (p["iterations"] - 1) - 1) < p["l_end"] // 2 + 1


def test_pow2_and_all_sets():
    assert F.widths_pow2(8192) == [2 ** i for i in range(14)]
    assert F.widths_all(64) == list(range(1, 65))
    assert F.width_set("POW2", 0, 256) == [1, 2, 4, 8, 16, 32, 64, 128, 256]
    g = F.widths_geometric(1.8, 8192)
    assert g[0] == 1 and g[-1] <= 8192 and all(b > a for a, b in zip(g, g[1:]))


# --- P4: eq. (23)/(24) hand values ---------------------------------------------------

def test_best_case_hand_values():
    w = F.widths_pow2(8192)
    assert F.rsnr_max(3, w) == pytest.approx(math.sqrt(3 / 4))
    assert F.rsnr_max(7, w) == pytest.approx(math.sqrt(7 / 8))
    assert F.rsnr_max(20, w) == pytest.approx(math.sqrt(16 / 20))
    assert F.rsnr_max(45, w) == pytest.approx(math.sqrt(32 / 45))
    for L in w:
        assert F.rsnr_max(L, w) == 1.0                       # S = L -> RSNR = C
    # worst systematic loss of the 2^i set tends to 1 - 2^(-1/4) (S ~ sqrt(2) 2^i)
    worst = max(F.systematic_loss(S, w) for S in range(1, 8193))
    assert worst <= 1 - 2 ** -0.25 + 1e-12
    assert worst == pytest.approx(1 - 2 ** -0.25, abs=2e-4)


def test_best_case_three_cases():
    # PAPER.md:858-860
    assert F.rsnr_max_single(5, 32) == pytest.approx(math.sqrt(5) / math.sqrt(32))
    assert F.rsnr_max_single(32, 32) == 1.0
    assert F.rsnr_max_single(50, 32) == pytest.approx(math.sqrt(32) / math.sqrt(50))
    assert F.rsnr(20, 16, 16) == pytest.approx(16 / math.sqrt(16 * 20))


# --- P5: L_s = 1 collapses the worst case onto the best case ------------------------

def test_separation_one_collapses_to_best_case():
    for L in (1, 2, 3, 5, 8, 16, 31, 64):
        for S in range(1, 200):
            assert F.rsnr_min_single(S, L, 1) == pytest.approx(F.rsnr_max_single(S, L), abs=1e-15)


# --- P1: eq. (27)-(30) against a brute-force scan over pulse shifts -----------------

@pytest.mark.parametrize("L,Ls", [(5, 3), (8, 8), (8, 4), (8, 2), (16, 16), (12, 4), (32, 8), (7, 7), (9, 2)])
def test_single_width_worst_case_equals_brute_force(L, Ls):
    for S in range(1, 4 * L + 2 * Ls):
        lo, hi, _ = F.brute_force_response(S, [L], Ls)
        assert lo == pytest.approx(F.rsnr_min_single(S, L, Ls), abs=1e-12), (S, L, Ls)
        assert hi == pytest.approx(F.rsnr_max_single(S, L), abs=1e-12), (S, L, Ls)


def test_paper_worked_figures_33_32():
    # Fig. 33: L = 5, Ls = 3, S = 4 lies between two boxcars;
    # Fig. 32: S = 8 >= L + Ls covers a boxcar fully, S = 2 <= L - Ls is fully covered.
    assert F.rsnr_min_single(8, 5, 3) == pytest.approx(math.sqrt(5) / math.sqrt(8))
    assert F.rsnr_min_single(2, 5, 3) == pytest.approx(math.sqrt(2) / math.sqrt(5))
    assert F.coverage_lt(4, 5, 3) == 3
    lo, _, _ = F.brute_force_response(4, [5], 3)
    assert lo == pytest.approx(3 / math.sqrt(20))


def test_set_response_bounds_brute_force():
    # measured responses must lie between eq. (31) and eq. (24)
    for widths, sep in ((F.widths_pow2(64), lambda L: L),
                        (F.widths_igrid(1, 64), F.igrid_separation(4)),
                        (F.widths_boxdit(4, 60), F.boxdit_separation(4))):
        for S in range(1, 80):
            lo, hi, _ = F.brute_force_response(S, widths, sep)
            assert lo >= F.rsnr_min(S, widths, sep) - 1e-12
            assert hi == pytest.approx(F.rsnr_max(S, widths), abs=1e-12)


def test_dit_losses_match_paper(paper_pins):
    p = paper_pins["dit_loss"]
    w = F.widths_pow2(8192)
    worst = max(F.worst_loss(S, w, lambda L: L) for S in range(1, 8193))
    assert abs(worst - p["worst"]) < p["tolerance"]              # 40.5 % vs "40 %"
    # position-averaged loss by brute force over every pulse shift (self-similar, so a
    # smaller S0 suffices), averaged over S by eq. (19)
    w256 = F.widths_pow2(256)
    avg = F.cumulative_mean_loss(lambda S: 1.0 - F.brute_force_response(S, w256, lambda L: L)[2], 256)
    assert abs(avg - p["average"]) < p["tolerance"]              # 19.9 % vs "20 %"


def test_configuration_losses_match_paper(paper_pins):
    p = paper_pins["configuration_losses"]
    S0 = 8192
    ig1 = F.widths_igrid(1, S0)
    worst_ig1 = max(F.worst_loss(S, ig1, F.igrid_separation(4)) for S in range(1, S0 + 1))
    assert abs(worst_ig1 - p["ig1"]) < 0.005                     # 12.6 % vs "12.5 %"
    ig3 = F.widths_igrid(3, S0)
    mean_ig3 = F.cumulative_mean_loss(lambda S: F.worst_loss(S, ig3, F.igrid_separation(16)), S0)
    assert abs(mean_ig3 - p["ig3"]) < 0.005                      # 2.2 % vs "2 %"
    bd32 = F.widths_boxdit(32, S0)
    mean_bd32 = F.cumulative_mean_loss(lambda S: F.worst_loss(S, bd32, F.boxdit_separation(32)), S0)
    assert abs(mean_bd32 - p["bd32"]) < 0.005                    # 1.1 % vs "1 %"


def test_cumulative_mean_is_eq19_as_printed():
    assert F.cumulative_mean_loss(lambda s: 0.5, 11) == pytest.approx(11 * 0.5 / 10)
    w = F.widths_pow2(8192)
    m = F.cumulative_mean_loss(lambda S: F.systematic_loss(S, w), 8192)
    assert 0.07 < m < 0.09          # the "about 7 %" regime of BASELINE.json config 3 (8.10 %)


def test_mean_loss_over_population():
    w = F.widths_pow2(64)
    pop = [1, 3, 7, 20, 45]
    expect = sum(1 - r for r in (1.0, math.sqrt(3 / 4), math.sqrt(7 / 8), math.sqrt(16 / 20), math.sqrt(32 / 45))) / 5
    assert F.mean_loss_over_widths(pop, w) == pytest.approx(expect)
