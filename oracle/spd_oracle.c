/*
 * ORACLE - TEST INFRASTRUCTURE ONLY.  Not part of the product.
 *
 * A plain, slow, double-precision CPU statement of what the single-pulse-
 * detection (SPD) hot path computes, written from /root/reference/PAPER.md
 * (Adamek & Armour 2020).  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.
 * It shares no code, header, table or helper with the CUDA path under
 * paper_1910_08324_b200/csrc/.
 *
 * What is computed, per DM trial d and time sample n:
 *
 *   X_L[n]   = sum_{j=0}^{L-1} x[d, n+j]                      eq. (2)
 *   SNR_L[n] = (X_L[n] - mu(X_L)) / sigma(X_L)                eq. (4)
 *   mu(X_L)  = L mu_d ,  sigma(X_L) = sqrt(L) sigma_d         eq. (5)
 *   Y[n]     = max_{L in B} SNR_L[n],  W[n] = that L's index  eq. (12)
 *
 * Widths are visited in ascending order and the best is replaced only by a
 * strictly higher SNR ("If the new SNR is higher than the old SNR ...",
 * PAPER.md:287), so the smallest width wins exact ties (reading A4).
 * Windows that would cross the end of the row are skipped (reading A3:
 * valid-only); if no width fits, Y = -inf and W = -1.
 *
 *   oracle_spd_direct  : the definition, every boxcar by direct summation
 *                        (the "ideal SPD algorithm" route).
 *   oracle_spd_prefix  : same quantities via a double-precision running sum
 *                        C[n] of (x - mu) and X'_L[n] = C[n+L] - C[n]; a faster
 *                        route used on full planes, itself pinned to
 *                        oracle_spd_direct in tests (<= 1e-9).
 *   oracle_spd_grid    : oracle_spd_direct with a boxcar separation per width (the
 *                        paper's decimated grids, merged into one plane; reading A16).
 *   oracle_spd_grid_iter: the output separated by iteration (eq. 12): one decimated plane per
 *                        run of widths that share a separation, direct summation.
 *   oracle_width_sigma : standard deviation per width from power-of-two decimations,
 *                        interpolated (reading A17); oracle_spd_direct_sw uses it.
 *   oracle_snr_of_width: SNR_L[n] for one width at listed samples (near-tie checks).
 *   oracle_row_stats   : per-row mean and population standard deviation (reading A6).
 *   oracle_spd_grid_sw : oracle_spd_grid with a measured standard deviation per width.
 *   oracle_row_stats_clipped: mean / sigma with point-wise outlier rejection, a given number
 *                        of passes or "until convergence" (reading A14),
 *                        everything in double.
 *   oracle_find_candidates: threshold + 1-D local-peak rule (reading A9).
 *   oracle_cluster_candidates: 2-D (DM x time) peak rule over the 1-D candidates (reading A18).
 *
 * Pins: tests/test_oracle_pins.py (closed form eq. 22 on single-pulse planes,
 * numpy.convolve for single widths, constant / ramp / impulse closed forms,
 * affine and shift invariances, white-noise statistics, brute force, the
 * Fig. 17 worked example PAPER.md:587,605, eq. 24 on noise-free twins).
 * oracle_row_stats(_clipped): numpy mean / std; exact two-valued rows with outliers;
 * the textbook variance of a normal distribution truncated at +-c sigma.
 * oracle_find_candidates: the rule is this project's reading A9 (the paper
 * names "peak-finding" only) - pinned by closed form on
 * isolated pulses; otherwise "parity unpinned by the paper".
 * oracle_cluster_candidates: reading A18, this project's definition as well (same passages):
 * pinned on hand-built planes (a pulse smeared over neighbouring DM rows gives one cluster at
 * its peak; two pulses further apart than the window give two; exact ties keep the first in
 * (dm, t) order) and against a brute-force window scan; "parity unpinned by the paper".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Direct summation over samples [t0, t1) of every row.  Outputs are
 * [n_dm][t1 - t0]; out_second (may be NULL) receives the best SNR among all
 * widths other than the arg-max one (-inf if none). */
void oracle_spd_direct(const float* x, int64_t n_dm, int64_t n_t,
                       const double* mean, const double* sigma,
                       const int32_t* widths, int32_t n_w,
                       int64_t t0, int64_t t1,
                       double* out_snr, int32_t* out_width, double* out_second) {
    const int64_t span = t1 - t0;
#pragma omp parallel for collapse(2) schedule(dynamic, 256)
    for (int64_t d = 0; d < n_dm; ++d) {
        for (int64_t n = t0; n < t1; ++n) {
            const float* row = x + d * n_t;
            double best = -INFINITY, second = -INFINITY;
            int32_t idx = -1;
            for (int32_t k = 0; k < n_w; ++k) {
                const int64_t L = widths[k];
                if (n + L > n_t) break;                       /* valid windows only (A3) */
                double X = 0.0;
                for (int64_t j = 0; j < L; ++j) X += (double)row[n + j];      /* eq. (2) */
                const double snr = (X - (double)L * mean[d]) / (sqrt((double)L) * sigma[d]); /* eq. (4),(5) */
                if (snr > best) {                              /* strict '>' (A4) */
                    second = best;
                    best = snr;
                    idx = k;
                } else if (snr > second) {
                    second = snr;
                }
            }
            const int64_t o = d * span + (n - t0);
            out_snr[o] = best;
            out_width[o] = idx;
            if (out_second) out_second[o] = second;
        }
    }
}

/* Per-width boxcar separation (the paper's lossy grids): width k is
 * evaluated only at the samples n that are multiples of its separation L_s[k]
 * ("boxcar filters of width L=6,8,10,12 are calculated at every second point", PAPER.md:201;
 * BoxDIT iteration i works at every D^(i)-th point, Alg. 1; DIT width 2^i at
 * every 2^i-th point, Alg. 3; IGRID with P layers at 2^i / P).
 * Reading A16: one merged full-resolution plane, Y[n] = max over the widths whose grid
 * contains n (eq. 12 restricted to them), -inf / -1 where none does; everything else
 * (eq. 2, 4, 5, valid windows only, strict '>' in ascending width order) as oracle_spd_direct.
 * Pins (tests/test_oracle_pins.py): pulses slid over all shifts recover exactly the
 * worst / best responses of eq. (27)-(31) and (24); the constant-offset
 * closed form reproduces the example grid of PAPER.md:201; separations all 1 = oracle_spd_direct. */
void oracle_spd_grid(const float* x, int64_t n_dm, int64_t n_t,
                     const double* mean, const double* sigma,
                     const int32_t* widths, const int32_t* seps, int32_t n_w,
                     int64_t t0, int64_t t1,
                     double* out_snr, int32_t* out_width, double* out_second) {
    const int64_t span = t1 - t0;
#pragma omp parallel for collapse(2) schedule(dynamic, 256)
    for (int64_t d = 0; d < n_dm; ++d) {
        for (int64_t n = t0; n < t1; ++n) {
            const float* row = x + d * n_t;
            double best = -INFINITY, second = -INFINITY;
            int32_t idx = -1;
            for (int32_t k = 0; k < n_w; ++k) {
                const int64_t L = widths[k];
                if (n + L > n_t) break;                       /* valid windows only (A3) */
                if (n % (int64_t)seps[k] != 0) continue;      /* n is not on this width's grid */
                double X = 0.0;
                for (int64_t j = 0; j < L; ++j) X += (double)row[n + j];      /* eq. (2) */
                const double snr = (X - (double)L * mean[d]) / (sqrt((double)L) * sigma[d]); /* eq. (4),(5) */
                if (snr > best) {                              /* strict '>' (A4) */
                    second = best;
                    best = snr;
                    idx = k;
                } else if (snr > second) {
                    second = snr;
                }
            }
            const int64_t o = d * span + (n - t0);
            out_snr[o] = best;
            out_width[o] = idx;
            if (out_second) out_second[o] = second;
        }
    }
}

/* Output separated by iteration, eq. (12): "the output for ith iteration is
 * Y^i[n] = max_{L in B^i} SNR(X^i_L[n])", with "the width of the boxcar which produced the highest SNR
 * value W^i"; Y^i has N / D^(i) samples.  An iteration here is a run of consecutive
 * widths [kb, ke) of a grid plan that share one separation s = seps[kb] (BoxDIT iteration i: s = D^(i),
 * widths of eq. 14; DIT: one width per iteration; IGRID: the widths of one step).  Point m of the
 * iteration's plane is sample n = s m of the row, m < ceil(n_t / s):
 *     Y^i[m] = max over k in [kb, ke) with n + L_k <= n_t of (X_{L_k}[n] - L_k mu) / (sqrt(L_k) sigma),
 * X by direct summation (eq. 2), W^i[m] = that k (index in the plan's width set; -1 and -inf where no
 * width of the iteration fits the row, reading A3), strict '>' in ascending order (A4).
 * out_* are [n_dm][n_pts], n_pts = ceil(n_t / s).
 * Pins (tests/test_oracle_pins.py): a literal transcription of Alg. 1 with eq. (13)'s shifted decimation
 * and eq. (15) (x^{i+1}, X^i carried from iteration to iteration) gives the same planes; the maximum over
 * the iterations at a sample is oracle_spd_grid's merged plane (reading A16); the constant-offset closed
 * form on the example of PAPER.md:201 (widths 1..4 at every point, 6, 8, 10, 12 at every second). */
void oracle_spd_grid_iter(const float* x, int64_t n_dm, int64_t n_t,
                          const double* mean, const double* sigma,
                          const int32_t* widths, const int32_t* seps, int32_t kb, int32_t ke,
                          double* out_snr, int32_t* out_width, double* out_second) {
    const int64_t s = seps[kb];
    const int64_t n_pts = (n_t + s - 1) / s;
#pragma omp parallel for collapse(2) schedule(dynamic, 256)
    for (int64_t d = 0; d < n_dm; ++d) {
        for (int64_t m = 0; m < n_pts; ++m) {
            const float* row = x + d * n_t;
            const int64_t n = s * m;
            double best = -INFINITY, second = -INFINITY;
            int32_t idx = -1;
            for (int32_t k = kb; k < ke; ++k) {
                const int64_t L = widths[k];
                if (n + L > n_t) break;                       /* valid windows only (A3) */
                double X = 0.0;
                for (int64_t j = 0; j < L; ++j) X += (double)row[n + j];      /* eq. (2) */
                const double snr = (X - (double)L * mean[d]) / (sqrt((double)L) * sigma[d]); /* eq. (4),(5) */
                if (snr > best) {                              /* strict '>' (A4) */
                    second = best;
                    best = snr;
                    idx = k;
                } else if (snr > second) {
                    second = snr;
                }
            }
            const int64_t o = d * n_pts + m;
            out_snr[o] = best;
            out_width[o] = idx;
            if (out_second) out_second[o] = second;
        }
    }
}

/* Standard deviation per boxcar width on real (non-white) data, PAPER.md:728:
 * "we calculate values of the standard deviation only for time-series which are decimations of the
 * input time-series in time, i.e. ... only for boxcar filters of width that are equal to a powers of
 * two.  We then interpolate values of standard deviation for all intermediate boxcar widths."
 * Reading A17: level j = the series of sums of 2^j consecutive samples, x^j[m] = sum_{i<2^j} x[2^j m + i],
 * m < floor(n_t / 2^j) (eq. 13 with D = 2, without its shift); sigma_j = its population
 * standard deviation; for 2^j <= L < 2^(j+1) sigma_L is linear in L between sigma_j and sigma_(j+1);
 * above the last level with at least two elements it follows eq. (5)'s sqrt(L) from that level.
 * out_sigma_w is [n_dm][n_w].  Pins: numpy on hand-decimated rows, eq. (5) on white noise, the
 * textbook variance of block sums of an AR(1) process, exact interpolation midpoints. */
void oracle_width_sigma(const float* x, int64_t n_dm, int64_t n_t,
                        const int32_t* widths, int32_t n_w, double* out_sigma_w) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t d = 0; d < n_dm; ++d) {
        const float* row = x + d * n_t;
        double sig[40];
        int n_lev = 0;
        for (int j = 0; j < 40; ++j) {
            const int64_t blk = (int64_t)1 << j;
            const int64_t cnt = n_t / blk;
            if (cnt < 2) break;
            double s1 = 0.0;
            for (int64_t m = 0; m < cnt; ++m) {
                double v = 0.0;
                for (int64_t i = 0; i < blk; ++i) v += (double)row[m * blk + i];
                s1 += v;
            }
            const double mean = s1 / (double)cnt;
            double s2 = 0.0;
            for (int64_t m = 0; m < cnt; ++m) {
                double v = 0.0;
                for (int64_t i = 0; i < blk; ++i) v += (double)row[m * blk + i];
                s2 += (v - mean) * (v - mean);
            }
            sig[j] = sqrt(s2 / (double)cnt);
            n_lev = j + 1;
        }
        for (int32_t k = 0; k < n_w; ++k) {
            const int64_t L = widths[k];
            int j = 0;
            while (((int64_t)2 << j) <= L) ++j;               /* 2^j <= L < 2^(j+1) */
            double s;
            if (n_lev == 0) {
                s = 0.0;                                      /* a one-sample row has no deviation */
            } else if (j + 1 < n_lev) {
                const double lo = (double)((int64_t)1 << j);
                s = sig[j] + (sig[j + 1] - sig[j]) * ((double)L - lo) / lo;
            } else {
                const int jj = n_lev - 1;
                s = sig[jj] * sqrt((double)L / (double)((int64_t)1 << jj));
            }
            out_sigma_w[d * n_w + k] = s;
        }
    }
}

/* oracle_spd_direct with a measured standard deviation per width:
 * SNR_L[n] = (X_L[n] - L mu_d) / sigma_{d,L}   (eq. 4, with mu(X_L) = L mu of eq. 5). */
void oracle_spd_direct_sw(const float* x, int64_t n_dm, int64_t n_t,
                          const double* mean, const double* sigma_w,
                          const int32_t* widths, int32_t n_w,
                          int64_t t0, int64_t t1,
                          double* out_snr, int32_t* out_width, double* out_second) {
    const int64_t span = t1 - t0;
#pragma omp parallel for collapse(2) schedule(dynamic, 256)
    for (int64_t d = 0; d < n_dm; ++d) {
        for (int64_t n = t0; n < t1; ++n) {
            const float* row = x + d * n_t;
            double best = -INFINITY, second = -INFINITY;
            int32_t idx = -1;
            for (int32_t k = 0; k < n_w; ++k) {
                const int64_t L = widths[k];
                if (n + L > n_t) break;
                double X = 0.0;
                for (int64_t j = 0; j < L; ++j) X += (double)row[n + j];
                const double snr = (X - (double)L * mean[d]) / sigma_w[d * n_w + k];
                if (snr > best) {
                    second = best;
                    best = snr;
                    idx = k;
                } else if (snr > second) {
                    second = snr;
                }
            }
            const int64_t o = d * span + (n - t0);
            out_snr[o] = best;
            out_width[o] = idx;
            if (out_second) out_second[o] = second;
        }
    }
}

/* oracle_spd_grid with a measured standard deviation per width (rows f1 + f2 together):
 * SNR_L[n] = (X_L[n] - L mu_d) / sigma_{d,L} (eq. 4; sigma(X_L) measured and interpolated,
 * PAPER.md:728) for the widths whose grid contains n (reading A16).  Pins: with sigma_w = sqrt(L) sigma
 * it reproduces oracle_spd_grid bit for bit; with separations all 1 it reproduces oracle_spd_direct_sw. */
void oracle_spd_grid_sw(const float* x, int64_t n_dm, int64_t n_t,
                        const double* mean, const double* sigma_w,
                        const int32_t* widths, const int32_t* seps, int32_t n_w,
                        int64_t t0, int64_t t1,
                        double* out_snr, int32_t* out_width, double* out_second) {
    const int64_t span = t1 - t0;
#pragma omp parallel for collapse(2) schedule(dynamic, 256)
    for (int64_t d = 0; d < n_dm; ++d) {
        for (int64_t n = t0; n < t1; ++n) {
            const float* row = x + d * n_t;
            double best = -INFINITY, second = -INFINITY;
            int32_t idx = -1;
            for (int32_t k = 0; k < n_w; ++k) {
                const int64_t L = widths[k];
                if (n + L > n_t) break;                       /* valid windows only (A3) */
                if (n % (int64_t)seps[k] != 0) continue;      /* n is not on this width's grid (A16) */
                double X = 0.0;
                for (int64_t j = 0; j < L; ++j) X += (double)row[n + j];      /* eq. (2) */
                const double snr = (X - (double)L * mean[d]) / sigma_w[d * n_w + k];  /* eq. (4) */
                if (snr > best) {
                    second = best;
                    best = snr;
                    idx = k;
                } else if (snr > second) {
                    second = snr;
                }
            }
            const int64_t o = d * span + (n - t0);
            out_snr[o] = best;
            out_width[o] = idx;
            if (out_second) out_second[o] = second;
        }
    }
}

/* Same quantities through a double-precision running sum of (x - mu). */
void oracle_spd_prefix(const float* x, int64_t n_dm, int64_t n_t,
                       const double* mean, const double* sigma,
                       const int32_t* widths, int32_t n_w,
                       double* out_snr, int32_t* out_width, double* out_second) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t d = 0; d < n_dm; ++d) {
        const float* row = x + d * n_t;
        double* C = (double*)malloc((size_t)(n_t + 1) * sizeof(double));
        C[0] = 0.0;
        for (int64_t n = 0; n < n_t; ++n) C[n + 1] = C[n] + ((double)row[n] - mean[d]);
        for (int64_t n = 0; n < n_t; ++n) {
            double best = -INFINITY, second = -INFINITY;
            int32_t idx = -1;
            for (int32_t k = 0; k < n_w; ++k) {
                const int64_t L = widths[k];
                if (n + L > n_t) break;
                const double snr = (C[n + L] - C[n]) / (sqrt((double)L) * sigma[d]);
                if (snr > best) {
                    second = best;
                    best = snr;
                    idx = k;
                } else if (snr > second) {
                    second = snr;
                }
            }
            const int64_t o = d * n_t + n;
            out_snr[o] = best;
            out_width[o] = idx;
            if (out_second) out_second[o] = second;
        }
        free(C);
    }
}

/* SNR_L[n] by direct summation for one row, one width, at listed samples
 * (NaN where the window does not fit). */
void oracle_snr_of_width(const float* row, int64_t n_t, double mean, double sigma,
                         int64_t L, const int64_t* samples, int64_t count, double* out) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < count; ++i) {
        const int64_t n = samples[i];
        if (n < 0 || n + L > n_t) { out[i] = NAN; continue; }
        double X = 0.0;
        for (int64_t j = 0; j < L; ++j) X += (double)row[n + j];
        out[i] = (X - (double)L * mean) / (sqrt((double)L) * sigma);
    }
}

/* Per-row mean and population standard deviation (ddof = 0), two passes in
 * double (reading A6 of SURVEY.md sec. 8(c) for "computed from the plane"). */
void oracle_row_stats(const float* x, int64_t n_dm, int64_t n_t, double* mean, double* sigma) {
#pragma omp parallel for schedule(static)
    for (int64_t d = 0; d < n_dm; ++d) {
        const float* row = x + d * n_t;
        double s = 0.0;
        for (int64_t n = 0; n < n_t; ++n) s += (double)row[n];
        const double m = s / (double)n_t;
        double v = 0.0;
        for (int64_t n = 0; n < n_t; ++n) {
            const double e = (double)row[n] - m;
            v += e * e;
        }
        mean[d] = m;
        sigma[d] = sqrt(v / (double)n_t);
    }
}

/* Mean and standard deviation with point-wise outlier rejection (sec. 4.6.2:
 * "Each point is compared with the current estimate of the mean and standard deviation and
 * rejected if it is significantly different (the threshold is user defined).  This is repeated
 * until convergence."; reading A14).  Everything in double:
 *   pass 0: mean and population sigma of all samples of the row;
 *   pass i >= 1: keep x iff |x - mu| <= clip * sigma with mu, sigma of pass i-1; mean and sigma
 *           of the kept samples by the plain two-pass definition.
 * Stops after max_reject_passes rejection passes or - "until convergence" - after the first
 * pass that changes neither estimate by more than rel_tol * sigma(previous pass)
 * (|mu_i - mu_(i-1)| and |sigma_i - sigma_(i-1)|; rel_tol < 0 never stops early, so that the
 * pass count is the caller's).  A pass that rejects every sample keeps the previous estimate
 * and stops.  n_passes[d] (may be NULL) receives the rejection passes done.
 * n_border[d] (may be NULL) counts, over all passes, the samples within border_eps * sigma of
 * the rejection limit: the samples whose side a single-precision implementation may decide
 * differently (tests/ bound the CUDA path's deviation by it). */
void oracle_row_stats_clipped(const float* x, int64_t n_dm, int64_t n_t, double clip,
                              int32_t max_reject_passes, double rel_tol, double border_eps,
                              double* mean, double* sigma, int32_t* n_passes, int64_t* n_border) {
#pragma omp parallel for schedule(static)
    for (int64_t d = 0; d < n_dm; ++d) {
        const float* row = x + d * n_t;
        double mu = 0.0, sg = 0.0;
        int32_t done = 0;
        int64_t border = 0;
        for (int32_t pass = 0; pass <= max_reject_passes; ++pass) {
            const double lim = clip * sg;
            double s = 0.0;
            int64_t cnt = 0;
            for (int64_t n = 0; n < n_t; ++n) {
                const double dev = fabs((double)row[n] - mu);
                if (pass > 0 && fabs(dev - lim) <= border_eps * sg) ++border;
                if (pass == 0 || dev <= lim) {
                    s += (double)row[n];
                    ++cnt;
                }
            }
            if (cnt == 0) break;
            const double m = s / (double)cnt;
            double v = 0.0;
            for (int64_t n = 0; n < n_t; ++n) {
                if (pass == 0 || fabs((double)row[n] - mu) <= lim) {
                    const double e = (double)row[n] - m;
                    v += e * e;
                }
            }
            const double sg_new = sqrt(v / (double)cnt);
            const int converged = pass > 0 && fabs(m - mu) <= rel_tol * sg && fabs(sg_new - sg) <= rel_tol * sg;
            mu = m;
            sg = sg_new;
            if (pass > 0) done = pass;
            if (converged) break;
        }
        mean[d] = mu;
        sigma[d] = sg;
        if (n_passes) n_passes[d] = done;
        if (n_border) n_border[d] = border;
    }
}

/* Candidate rule (reading A9): (d, n) is a candidate iff Y[d,n] >= thr and
 * Y[d,n] > Y[d,n-1] and Y[d,n] >= Y[d,n+1], row ends comparing against -inf
 * (first sample of a plateau).  Candidates are emitted in (d, n) order; the
 * return value counts all of them, the arrays receive the first `capacity`. */
int64_t oracle_find_candidates(const float* snr, const int32_t* width, int64_t n_dm, int64_t n_t,
                               float thr, int64_t capacity,
                               int32_t* c_dm, int32_t* c_t, float* c_snr, int32_t* c_width) {
    int64_t count = 0;
    for (int64_t d = 0; d < n_dm; ++d) {
        const float* y = snr + d * n_t;
        for (int64_t n = 0; n < n_t; ++n) {
            const float v = y[n];
            const float left = (n > 0) ? y[n - 1] : -INFINITY;
            const float right = (n + 1 < n_t) ? y[n + 1] : -INFINITY;
            if (v >= thr && v > left && v >= right) {
                if (count < capacity) {
                    c_dm[count] = (int32_t)d;
                    c_t[count] = (int32_t)n;
                    c_snr[count] = v;
                    c_width[count] = width[d * n_t + n];
                }
                ++count;
            }
        }
    }
    return count;
}

/* 2-D (DM x time) peak rule over the 1-D candidates (the paper names the
 * stage only: "lastly candidates are selected using a peak-finding algorithm").
 * Reading A18 (this project's definition): a 1-D candidate (d, n) with best width L = widths[W[d,n]]
 * is kept iff no sample of the window |d' - d| <= dm_radius, |n' - n| <= L (clipped to the plane)
 * has a larger Y, and no sample of the window that comes EARLIER in (d, n) order has an equal Y
 * (the first of an exact tie is the peak).  The half-width L ties the window to the width being
 * tested, as a 3 x 3 neighbourhood on a plane decimated by the boxcar separation would.
 * Inputs: the float32 planes and the candidate list (c_dm, c_t, c_width index into widths), any
 * order; keep[i] receives 1 / 0.  Returns the number kept. */
int64_t oracle_cluster_candidates(const float* snr, int64_t n_dm, int64_t n_t,
                                  const int32_t* widths, int32_t n_w,
                                  const int32_t* c_dm, const int32_t* c_t, const int32_t* c_width,
                                  int64_t n_cand, int32_t dm_radius, uint8_t* keep) {
    int64_t kept = 0;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : kept)
    for (int64_t i = 0; i < n_cand; ++i) {
        const int64_t d = c_dm[i], n = c_t[i];
        const int32_t wi = c_width[i];
        const int64_t L = (wi >= 0 && wi < n_w) ? widths[wi] : 1;
        const float v = snr[d * n_t + n];
        const int64_t d_lo = d - dm_radius < 0 ? 0 : d - dm_radius;
        const int64_t d_hi = d + dm_radius >= n_dm ? n_dm - 1 : d + dm_radius;
        const int64_t n_lo = n - L < 0 ? 0 : n - L;
        const int64_t n_hi = n + L >= n_t ? n_t - 1 : n + L;
        int ok = 1;
        for (int64_t dd = d_lo; dd <= d_hi && ok; ++dd) {
            const float* y = snr + dd * n_t;
            for (int64_t nn = n_lo; nn <= n_hi; ++nn) {
                const float u = y[nn];
                if (u > v || (u == v && (dd < d || (dd == d && nn < n)))) {
                    ok = 0;
                    break;
                }
            }
        }
        keep[i] = (uint8_t)ok;
        kept += ok;
    }
    return kept;
}
