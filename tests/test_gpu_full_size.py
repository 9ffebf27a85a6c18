"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(spd_run_flagged + spd_find_candidates_flagged through the C ABI).

EVERY sample of configs 2-5 is compared with oracle B (the double-precision running sum, SURVEY.md
sec. 8(c) "Oracle B (accelerated, full planes)"), block-wise: <= 64 Mi samples of rows go to the
host at a time, the oracle runs on them, and its three outputs go back to the device where the
comparison rule of parity.py is evaluated with float64 tensor ops (the near-ties it leaves are settled
on the host by direct summation of the chosen width).  Oracle B itself is pinned at this size by
oracle A (direct summation) on sampled windows - around injected pulses, at row starts and row
tails, across the kernel's chunk, segment and piece boundaries, and at random places.  A window is a piece of one row
copied to the host together with the max_width - 1 samples that follow it, so every boxcar of
every compared sample lies inside the piece (windows that reach the end of the row exercise the
valid-windows-only rule instead).  Properties that hold at any size are checked on the whole
plane with integer / comparison tensor ops: width indices in range, Y finite, Y >= SNR of width 1
(width 1 is in every set used here), last sample of each row takes width 1, and the candidate list
equals the reading-A9 rule applied to the CUDA plane (exact integer comparison).
"""
import numpy as np
import pytest

import parity

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def spd():
    import paper_1910_08324_b200 as spd
    spd.build()
    spd.load()
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    return spd


def _window_list(w, info, pulses, rng, n_random):
    """(row, t0, span, kind) windows; span samples are compared."""
    M, n_t, n_dm = w.max_width, w.n_t, w.n_dm
    chunk = max(info["chunk"], 1)
    segs = max(info["segments_per_row"], 1)
    out = []
    direct_span = 1536 if M <= 8192 else 512
    # injected pulses: start of the pulse, its matched boxcars begin up to M samples earlier
    for p in pulses[:: max(1, len(pulses) // 12)]:
        t0 = max(0, p.t0 - direct_span // 2)
        out.append((p.dm, t0, min(direct_span, n_t - t0), "pulse"))
    # row starts and row tails (tail rule A3)
    for d in (0, n_dm - 1, int(rng.integers(0, n_dm))):
        out.append((d, 0, direct_span, "row-start"))
        out.append((d, n_t - direct_span, direct_span, "row-tail"))
        out.append((d, n_t - M - direct_span // 2, direct_span, "tail-onset"))
    # segment and chunk boundaries of the launch configuration
    chunks_per_row = (n_t + chunk - 1) // chunk
    seg_chunks = (chunks_per_row + segs - 1) // segs
    for s in range(1, segs)[:3]:
        b = s * seg_chunks * chunk
        out.append((int(rng.integers(0, n_dm)), b - direct_span // 2, direct_span, "segment-boundary"))
    # warp-per-stream kernel: the plane's steps are cut into pieces in row-major order
    piece = info.get("piece_chunks", 0)
    if piece > 0:
        n_pieces = (n_dm * chunks_per_row + piece - 1) // piece
        for pi in sorted({1, n_pieces // 3, n_pieces // 2, n_pieces - 1}):
            if 0 < pi < n_pieces:
                d, c = divmod(pi * piece, chunks_per_row)
                out.append((d, max(0, c * chunk - direct_span // 2), direct_span, "piece-boundary"))
    for _ in range(3):
        b = int(rng.integers(1, chunks_per_row)) * chunk
        out.append((int(rng.integers(0, n_dm)), b - direct_span // 2, direct_span, "chunk-boundary"))
    for _ in range(n_random):
        t0 = int(rng.integers(0, n_t - direct_span))
        out.append((int(rng.integers(0, n_dm)), t0, direct_span, "random"))
    return out


def _check_window(oracle, plane, snr, idx, mean_h, sigma_h, widths, M, row, t0, span, direct, what):
    n_t = plane.shape[1]
    t0 = max(0, min(int(t0), n_t - 1))
    span = int(min(span, n_t - t0))
    t_end = min(n_t, t0 + span + M - 1)
    seg = plane[row, t0:t_end].cpu().numpy()[None, :]
    got_snr = snr[row, t0:t0 + span].cpu().numpy()[None, :]
    got_idx = idx[row, t0:t0 + span].cpu().numpy()[None, :]
    mu, sg = float(mean_h[row]), float(sigma_h[row])
    if direct:
        ref_snr, ref_idx, ref_sec = oracle.spd_direct(seg, mu, sg, widths, 0, span)
    else:
        ref_snr, ref_idx, ref_sec = oracle.spd_prefix(seg, mu, sg, widths)
        ref_snr, ref_idx, ref_sec = ref_snr[:, :span], ref_idx[:, :span], ref_sec[:, :span]
    return parity.assert_parity(oracle, seg, mu, sg, widths, got_snr, got_idx, ref_snr, ref_idx, ref_sec,
                                what=f"{what} row {row} t0 {t0}")


def _prefix_oracle_block(oracle, x, mu, sg, widths):
    """oracle.spd_prefix on a block of whole rows.  The oracle runs one row per thread; a block of fewer rows
    than threads (config 5: one row of 2^26 samples) is cut into time segments that each carry the
    max_width - 1 samples that follow them, so that every window of a compared sample lies inside its segment;
    the last segment of a row keeps the row's real end (valid-windows-only rule)."""
    r, n_t = x.shape
    M = int(max(widths))
    n_seg = max(1, min(oracle.num_threads() * 2 // r, n_t // (8 * M)))
    if n_seg <= 1:
        return oracle.spd_prefix(x, mu, sg, widths)
    span = -(-n_t // n_seg)
    outs = [np.empty((r, n_t), dtype=np.float64), np.empty((r, n_t), dtype=np.int32),
            np.empty((r, n_t), dtype=np.float64)]
    n_full = (n_t - (M - 1)) // span               # segments that have their whole look-ahead inside the row
    n_full = min(n_full, n_seg - 1)
    if n_full > 0:
        seg = np.stack([x[d, s * span: s * span + span + M - 1] for d in range(r) for s in range(n_full)])
        res = oracle.spd_prefix(seg, np.repeat(mu, n_full), np.repeat(sg, n_full), widths)
        for o, a in zip(outs, res):
            o[:, : n_full * span] = a[:, :span].reshape(r, n_full * span)
    t0 = n_full * span
    res = oracle.spd_prefix(np.ascontiguousarray(x[:, t0:]), mu, sg, widths)
    for o, a in zip(outs, res):
        o[:, t0:] = a
    return tuple(outs)


def _full_plane_parity(oracle, plane, snr, idx, mean_h, sigma_h, widths, what):
    """parity.assert_parity's rule on every sample of the plane against oracle.spd_prefix, in row blocks."""
    n_dm, n_t = plane.shape
    dev = plane.device
    rows = max(1, min(n_dm, (1 << 26) // n_t))
    wl = np.asarray(sorted(set(int(v) for v in widths)), dtype=np.int64)
    worst, n_diff, n_cmp = 0.0, 0, 0
    ninf = float("-inf")
    for r0 in range(0, n_dm, rows):
        r1 = min(n_dm, r0 + rows)
        x = plane[r0:r1].cpu().numpy()
        ref_snr, ref_idx, ref_sec = _prefix_oracle_block(oracle, x, mean_h[r0:r1], sigma_h[r0:r1], widths)
        with np.errstate(invalid="ignore"):
            gap_h = (ref_snr - ref_sec).astype(np.float32)          # inf where there is no runner-up
        rs = torch.from_numpy(ref_snr).to(dev)
        ri = torch.from_numpy(ref_idx).to(dev)
        gap = torch.from_numpy(gap_h).to(dev)
        y = snr[r0:r1].double()
        k = idx[r0:r1].to(torch.int32)
        nofit = ri < 0
        if bool(nofit.any()):
            assert bool((y[nofit] == ninf).all()) and bool((k[nofit] == -1).all()), f"{what}: no-fit samples"
        ok = ~nofit
        assert bool(torch.isfinite(y[ok]).all()), f"{what}: non-finite SNR"
        tol = parity.SNR_RTOL * torch.clamp(torch.where(ok, rs, torch.zeros_like(rs)).abs(), min=1.0)
        ratio = torch.where(ok, (y - rs).abs() / tol, torch.zeros_like(rs))
        w_blk = float(ratio.max())
        if w_blk > 1.0:
            i = int(torch.argmax(ratio))
            raise AssertionError(f"{what}: SNR mismatch at row {r0 + i // n_t} sample {i % n_t}: cuda "
                                 f"{float(y.flatten()[i])!r} oracle {float(rs.flatten()[i])!r} (err/tol {w_blk:.3g})")
        worst = max(worst, w_blk)
        assert bool(((k >= 0) & (k < len(wl)))[ok].all()), f"{what}: width index out of range"
        diff = ok & (k != ri)
        decisive = diff & (gap.double() > tol)
        if bool(decisive.any()):
            i = int(torch.nonzero(decisive.flatten())[0])
            raise AssertionError(f"{what}: width index mismatch at row {r0 + i // n_t} sample {i % n_t} where the "
                                 f"oracle's top two differ by more than the tolerance ({int(decisive.sum())} such)")
        rr, cc = torch.nonzero(diff, as_tuple=True)
        if rr.numel():
            rr_h, cc_h = rr.cpu().numpy(), cc.cpu().numpy()
            kk_h = k[rr, cc].cpu().numpy()
            tol_h = tol[rr, cc].cpu().numpy()
            for row in np.unique(rr_h):
                sel = rr_h == row
                for kw in np.unique(kk_h[sel]):
                    m = sel & (kk_h == kw)
                    s_w = oracle.snr_of_width(x[row], float(mean_h[r0 + row]), float(sigma_h[r0 + row]),
                                              int(wl[kw]), cc_h[m].astype(np.int64))
                    bad = ~(np.abs(s_w - ref_snr[row, cc_h[m]]) <= tol_h[m])
                    assert not bad.any(), (f"{what}: near-tie width {wl[kw]} at row {r0 + row} sample "
                                           f"{cc_h[m][bad][0]} is not within tolerance of the best")
            n_diff += int(rr.numel())
        n_cmp += (r1 - r0) * n_t
        del rs, ri, gap, y, k, tol, ratio, diff, decisive
    return worst, n_diff, n_cmp


def _whole_plane_properties(plane, mean, sigma, snr, idx, n_widths, rows_per_block=64):
    n_dm, n_t = plane.shape
    for r0 in range(0, n_dm, rows_per_block):
        r1 = min(n_dm, r0 + rows_per_block)
        y, k = snr[r0:r1], idx[r0:r1]
        assert bool(torch.isfinite(y).all()), "non-finite SNR"
        assert int(k.min()) >= 0 and int(k.max()) < n_widths, "width index out of range"
        # width 1 is in the set: Y >= (x - mu) / sigma within the tolerance
        s1 = (plane[r0:r1] - mean[r0:r1, None]) / sigma[r0:r1, None]
        tol = parity.SNR_RTOL * torch.clamp(s1.abs(), min=1.0)
        assert bool((y >= s1 - tol).all()), "best SNR below the width-1 SNR"
        del s1, tol
        assert bool((k[:, -1] == 0).all()), "last sample of a row must take width 1 (reading A3)"


def _rule_candidates(snr, thr, rows_per_block=64):
    """Reading A9 on the CUDA plane with comparison ops only -> sorted int64 keys dm * n_t + t."""
    n_dm, n_t = snr.shape
    keys = []
    ninf = torch.full((1,), float("-inf"), device=snr.device)
    for r0 in range(0, n_dm, rows_per_block):
        y = snr[r0:r0 + rows_per_block]
        prev = torch.cat([ninf.expand(y.shape[0], 1), y[:, :-1]], dim=1)
        nxt = torch.cat([y[:, 1:], ninf.expand(y.shape[0], 1)], dim=1)
        hit = (y >= thr) & (y > prev) & (y >= nxt)
        del prev, nxt
        rr, tt = torch.nonzero(hit, as_tuple=True)
        keys.append((rr + r0) * n_t + tt)
    return torch.sort(torch.cat(keys))[0]


@pytest.mark.parametrize("cfg,width_kind", [(2, None), (3, None), (4, None), (5, None), (3, "IGRID"), (4, "IGRID")])
def test_full_size_config(spd, oracle_lib, cfg, width_kind):
    from dataclasses import replace
    from workloads import get_workload, make_plane_torch
    w = get_workload(cfg)
    if width_kind:  # the paper's IG(1) width set (IGRID streaming tree) on the same plane
        w = replace(w, width_kind=width_kind, width_param=1)
    dev = torch.device("cuda:0")
    free, _ = torch.cuda.mem_get_info(dev)
    need = 13 * w.n_samples + (6 << 30)
    if free < need:
        pytest.skip(f"config {cfg} needs {need >> 30} GiB of device memory, {free >> 30} GiB free")
    widths = spd.spd_width_set_generate(w.width_kind, w.width_param, w.max_width)
    plane, pulses = make_plane_torch(w, dev)
    if w.stats == "measured":  # reading A6: per-row mean and population sigma, in double
        mean = torch.cat([plane[r:r + 64].double().mean(dim=1) for r in range(0, w.n_dm, 64)]).float()
        sigma = torch.cat([plane[r:r + 64].double().std(dim=1, unbiased=False)
                           for r in range(0, w.n_dm, 64)]).float()
    else:
        mean = torch.zeros(w.n_dm, device=dev)
        sigma = torch.ones(w.n_dm, device=dev)
    thr = w.candidate_threshold if w.candidate_threshold is not None else 6.0
    cap = 1 << 22
    with spd.Plan(w.n_dm, w.n_t, widths, w.max_width) as plan:
        info = dict(plan.info)
        assert info["path"] == (spd.SPD_PATH_IGRID_TREE if width_kind else spd.SPD_PATH_DYADIC_TREE)
        snr, idx, act = plan.run_flagged(plane, mean, sigma, thr)
        lst, n_found = plan.find_candidates_flagged(snr, idx, act, thr, cap)
        torch.cuda.synchronize()
        count, cands = spd.candidates_to_numpy(lst, n_found, cap)

    # ---- sampled windows against the oracle ------------------------------------------------
    mean_h, sigma_h = mean.cpu().numpy().astype(np.float64), sigma.cpu().numpy().astype(np.float64)
    rng = np.random.default_rng(w.seed + 17)
    worst, n_cmp = 0.0, 0
    for row, t0, span, kind in _window_list(w, info, pulses, rng, n_random=6):
        st = _check_window(oracle_lib, plane, snr, idx, mean_h, sigma_h, widths, w.max_width, row, t0, span,
                           direct=True, what=f"config {cfg} {kind}")
        worst, n_cmp = max(worst, st.max_err_over_tol), n_cmp + st.n
    # longer windows with the running-sum oracle (itself pinned to direct summation)
    for _ in range(4):
        row = int(rng.integers(0, w.n_dm))
        span = min(1 << 18, w.n_t - w.max_width)
        t0 = int(rng.integers(0, w.n_t - span - w.max_width + 1))
        st = _check_window(oracle_lib, plane, snr, idx, mean_h, sigma_h, widths, w.max_width, row, t0, span,
                           direct=False, what=f"config {cfg} long")
        worst, n_cmp = max(worst, st.max_err_over_tol), n_cmp + st.n
    row = int(rng.integers(0, w.n_dm))
    span = min(1 << 18, w.n_t)
    st = _check_window(oracle_lib, plane, snr, idx, mean_h, sigma_h, widths, w.max_width, row, w.n_t - span, span,
                       direct=False, what=f"config {cfg} long-tail")
    worst, n_cmp = max(worst, st.max_err_over_tol), n_cmp + st.n
    assert worst <= 1.0 and n_cmp > 1 << 19

    # ---- every sample against oracle B --------------------------------------------------------
    worst_all, n_near, n_all = _full_plane_parity(oracle_lib, plane, snr, idx, mean_h, sigma_h, widths,
                                                  f"config {cfg} full plane")
    assert n_all == w.n_dm * w.n_t and worst_all <= 1.0
    print(f"config {cfg}{' IG(1)' if width_kind else ''}: {n_all} samples compared, max |dSNR|/tol = {worst_all:.3g}, "
          f"{n_near} near-tie width differences (all valid)")

    # ---- properties of the whole plane ------------------------------------------------------
    _whole_plane_properties(plane, mean, sigma, snr, idx, len(widths))

    # ---- candidate list = the rule on the CUDA plane (exact) --------------------------------
    ref_keys = _rule_candidates(snr, thr)
    assert count == int(ref_keys.numel()), f"config {cfg}: {count} candidates, rule gives {ref_keys.numel()}"
    if count <= cap:
        got_keys = torch.from_numpy(cands["dm"].astype(np.int64) * w.n_t + cands["t"].astype(np.int64)).to(dev)
        assert torch.equal(torch.sort(got_keys)[0], ref_keys)
        sel = torch.from_numpy(cands["dm"].astype(np.int64)).to(dev), torch.from_numpy(cands["t"].astype(np.int64)).to(dev)
        assert torch.equal(snr[sel], torch.from_numpy(cands["snr"]).to(dev))
        assert torch.equal(idx[sel], torch.from_numpy(cands["width_idx"]).to(dev))
    else:
        assert len(cands) == cap
    # every injected pulse clear of the threshold is detected near its start
    if count <= cap:
        hit = 0
        strong = [p for p in pulses if p.snr_t >= thr + 4.0]
        for p in strong:
            m = (cands["dm"] == p.dm) & (np.abs(cands["t"].astype(np.int64) - p.t0) <= 2 * p.width + 4)
            hit += bool(m.any())
        assert hit >= 0.95 * len(strong), f"config {cfg}: only {hit} of {len(strong)} strong pulses detected"


@pytest.mark.parametrize("kind,param", [("POW2", 0), ("IGRID", 1)])
def test_longest_row(spd, oracle_lib, kind, param):
    """Maximum row length of the C ABI (n_t <= 2^31 - 1): one DM trial of 2^31 - 4 samples (8.6 GB),
    widths up to 8192.  Windows at the row start, across the 2^30 and 2^31 - 2^28 marks, at segment
    boundaries and at the very end are compared with the oracle; the whole row is checked for
    Y >= SNR of width 1 and index range."""
    dev = torch.device("cuda:0")
    n_t = (1 << 31) - 4
    free, _ = torch.cuda.mem_get_info(dev)
    if free < 13 * n_t + (8 << 30):
        pytest.skip("not enough device memory")
    gen = torch.Generator(device=dev)
    gen.manual_seed(20260101)
    plane = torch.empty((1, n_t), dtype=torch.float32, device=dev)
    plane.normal_(generator=gen)
    for t0, S in ((5, 3000), ((1 << 30) - 1500, 3000), (n_t - 40000, 6000), (n_t - 2500, 2500)):
        plane[0, t0:t0 + S] += 12.0 / float(np.sqrt(S))
    mean = torch.zeros(1, device=dev)
    sigma = torch.ones(1, device=dev)
    widths = spd.spd_width_set_generate(kind, param, 8192)
    with spd.Plan(1, n_t, widths, 8192) as plan:
        info = dict(plan.info)
        snr, idx, act = plan.run_flagged(plane, mean, sigma, 6.0)
        lst, n_found = plan.find_candidates_flagged(snr, idx, act, 6.0, 1 << 20)
        torch.cuda.synchronize()
        count, cands = spd.candidates_to_numpy(lst, n_found, 1 << 20)
    mean_h, sigma_h = np.zeros(1), np.ones(1)
    chunk, segs = info["chunk"], max(info["segments_per_row"], 1)
    chunks_per_row = (n_t + chunk - 1) // chunk
    seg_chunks = (chunks_per_row + segs - 1) // segs
    starts = [0, (1 << 30) - 2000, (1 << 31) - (1 << 28) - 700, n_t - 8192 - 1000, n_t - 1536]
    starts += [s * seg_chunks * chunk - 700 for s in range(1, segs)][:3]
    if info.get("piece_chunks", 0) > 0:  # one row: pieces are stretches of this row
        n_pieces = (chunks_per_row + info["piece_chunks"] - 1) // info["piece_chunks"]
        starts += [pi * info["piece_chunks"] * chunk - 700 for pi in sorted({1, n_pieces // 2, n_pieces - 1})
                   if 0 < pi < n_pieces]
    worst = 0.0
    for t0 in starts:
        st = _check_window(oracle_lib, plane, snr, idx, mean_h, sigma_h, widths, 8192, 0, t0, 1536, direct=True,
                           what=f"longest row {kind}")
        worst = max(worst, st.max_err_over_tol)
    st = _check_window(oracle_lib, plane, snr, idx, mean_h, sigma_h, widths, 8192, 0, n_t - (1 << 18), 1 << 18,
                       direct=False, what=f"longest row {kind} tail")
    assert max(worst, st.max_err_over_tol) <= 1.0
    # whole row, in pieces
    piece = 1 << 28
    for a in range(0, n_t, piece):
        b = min(n_t, a + piece)
        y, k = snr[0, a:b], idx[0, a:b]
        assert bool(torch.isfinite(y).all()) and int(k.min()) >= 0 and int(k.max()) < len(widths)
        assert bool((y >= plane[0, a:b] - 1e-4 * torch.clamp(plane[0, a:b].abs(), min=1.0)).all())
    # the four injected pulses are in the candidate list
    for t0 in (5, (1 << 30) - 1500, n_t - 40000, n_t - 2500):
        assert bool(((cands["t"].astype(np.int64) - t0) ** 2 < 8192 ** 2).any()), t0
    assert count == len(cands) or count > (1 << 20)


@pytest.mark.parametrize("wkind,wparam,gkind,gparam", [("BOXDIT", 8, "BOXDIT", 8), ("IGRID", 1, "IGRID", 4)])
def test_full_size_config3_on_the_paper_grids(spd, oracle_lib, wkind, wparam, gkind, gparam):
    """Row f2 at BASELINE's config-3 size, in the configuration `bench.py --grid` times: sampled
    windows (injected pulses, row starts and tails, tile boundaries, random) against
    oracle_spd_grid, and whole-plane properties that hold at any size."""
    from dataclasses import replace
    from workloads import get_workload, make_plane_torch
    w = replace(get_workload(3), width_kind=wkind, width_param=wparam)
    dev = torch.device("cuda:0")
    free, _ = torch.cuda.mem_get_info(dev)
    if free < 13 * w.n_samples + (6 << 30):
        pytest.skip("not enough device memory")
    widths = spd.spd_width_set_generate(w.width_kind, w.width_param, w.max_width)
    seps = spd.spd_separation_generate(gkind, gparam, widths)
    plane, pulses = make_plane_torch(w, dev)
    mean, sigma = torch.zeros(w.n_dm, device=dev), torch.ones(w.n_dm, device=dev)
    with spd.Plan(w.n_dm, w.n_t, widths, w.max_width, separations=seps) as plan:
        info = dict(plan.info)
        assert info["path"] == spd.SPD_PATH_GRID
        snr, idx = plan.run(plane, mean, sigma)
        torch.cuda.synchronize()
    tile, M, n_t = info["chunk"], w.max_width, w.n_t
    rng = np.random.default_rng(w.seed + 23)
    span = 768
    wins = [(p.dm, max(0, p.t0 - span // 2)) for p in pulses[:: max(1, len(pulses) // 10)]]
    wins += [(0, 0), (w.n_dm - 1, n_t - span), (7, n_t - M - span // 2)]
    wins += [(int(rng.integers(0, w.n_dm)), int(rng.integers(1, n_t // tile)) * tile - span // 2) for _ in range(3)]
    wins += [(int(rng.integers(0, w.n_dm)), int(rng.integers(0, n_t - span))) for _ in range(4)]
    worst = 0.0
    for row, t0 in wins:
        t0 = t0 // 8192 * 8192 if t0 % 2 else t0          # keep a few windows on coarse grid points
        t1 = min(n_t, t0 + span)
        # the row up to t1 + M: every window of a sample < t1 ends inside it, or at the row's real end
        seg = plane[row, : min(n_t, t1 + M)].cpu().numpy()[None, :]
        ref_snr, ref_idx, ref_sec = oracle_lib.spd_grid(seg, 0.0, 1.0, widths, seps, t0, t1)
        st = parity.assert_parity(oracle_lib, seg, 0.0, 1.0, widths, snr[row, t0:t1].cpu().numpy()[None, :],
                                  idx[row, t0:t1].cpu().numpy()[None, :], ref_snr, ref_idx, ref_sec, t0=t0,
                                  what=f"grid {gkind}:{gparam} row {row} t0 {t0}")
        worst = max(worst, st.max_err_over_tol)
    assert worst <= 1.0
    # whole plane: finite, indices in range, width 1 is on every sample's grid, chosen widths on their grid
    sp = torch.from_numpy(np.asarray(seps)).to(dev)
    n = torch.arange(n_t, device=dev)
    for r0 in range(0, w.n_dm, 64):
        y, k = snr[r0:r0 + 64], idx[r0:r0 + 64]
        assert bool(torch.isfinite(y).all()) and int(k.min()) >= 0 and int(k.max()) < len(widths)
        assert bool((y >= plane[r0:r0 + 64] - 1e-4 * torch.clamp(plane[r0:r0 + 64].abs(), min=1.0)).all())
        assert bool((n[None, :] % sp[k.long()] == 0).all())


def test_full_size_config3_sigma_per_width(spd, oracle_lib):
    """Row f1 at config 3's size, as `bench.py` runs it: spd_width_sigma on the whole plane checked against the
    oracle on sampled rows, then spd_run_sigma_w (warp-per-stream kernel) against direct summation with the
    same table on sampled windows, and eq. (5) as a property of the white-noise plane."""
    from workloads import get_workload, make_plane_torch
    w = get_workload(3)
    dev = torch.device("cuda:0")
    free, _ = torch.cuda.mem_get_info(dev)
    if free < 13 * w.n_samples + (6 << 30):
        pytest.skip("not enough device memory")
    widths = spd.spd_width_set_generate(w.width_kind, w.width_param, w.max_width)
    plane, pulses = make_plane_torch(w, dev)
    with spd.Plan(w.n_dm, w.n_t, widths, w.max_width) as plan:
        assert plan.info["tree_kernel"] == 2
        mean, sigma = plan.row_stats(plane)
        sw = plan.width_sigma(plane, mean)
        snr, idx = plan.run_sigma_w(plane, mean, sw)
        torch.cuda.synchronize()
    sw_h = sw.cpu().numpy().astype(np.float64)
    # the plane is white noise (+ a few pulses): sigma_L = sqrt(L) sigma to the sampling error of each level
    L = np.asarray(widths, dtype=np.float64)
    rel = sw_h / (sigma.cpu().numpy().astype(np.float64)[:, None] * np.sqrt(L)[None, :]) - 1.0
    quiet = np.ones(w.n_dm, dtype=bool)
    quiet[[p.dm for p in pulses]] = False     # an injected pulse is an outlier of the level near its width
    assert quiet.sum() > w.n_dm // 2
    assert np.all(np.abs(rel[quiet]) < 6.0 * np.sqrt(L / (2.0 * w.n_t))[None, :] + 0.02)
    rng = np.random.default_rng(w.seed + 31)
    rows = sorted({0, w.n_dm - 1, pulses[0].dm, int(rng.integers(0, w.n_dm))})
    for r in rows:
        ref = oracle_lib.width_sigma(plane[r].cpu().numpy()[None, :], widths)[0]
        assert np.allclose(sw_h[r], ref, rtol=2e-5, atol=0), (r, np.abs(sw_h[r] / ref - 1).max())
    mean_h = mean.cpu().numpy().astype(np.float64)
    M, n_t, span = w.max_width, w.n_t, 1024
    wins = [(p.dm, max(0, p.t0 - span // 2)) for p in pulses[:: max(1, len(pulses) // 6)]]
    wins += [(0, 0), (w.n_dm - 1, n_t - span), (5, n_t - M - span // 2), (int(rng.integers(0, w.n_dm)), int(rng.integers(0, n_t - span)))]
    for row, t0 in wins:
        t1 = min(n_t, t0 + span)
        lo, hi = t0, min(n_t, t1 + M)
        seg = plane[row, lo:hi].cpu().numpy()[None, :]
        if hi < n_t:   # not the row's end: every window of a sample < t1 must count as fitting
            seg = np.concatenate([seg, np.zeros((1, 1), np.float32)], axis=1)
        ref_snr, ref_idx, ref_sec = oracle_lib.spd_direct_sw(seg, mean_h[row], sw_h[row][None, :], widths, 0, t1 - t0)
        got_snr = snr[row, t0:t1].cpu().numpy()[None, :]
        got_idx = idx[row, t0:t1].cpu().numpy()[None, :]
        tol = parity.snr_tolerance(ref_snr)
        assert np.all(np.abs(got_snr - ref_snr) <= tol), (row, t0)
        decisive = (ref_snr - ref_sec) > tol
        assert np.array_equal(got_idx[decisive], ref_idx[decisive]), (row, t0)
