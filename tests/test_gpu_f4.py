"""SURVEY.md sec. 8(f) row f4 on the GPU: the compact (uint8) width index, the 2-D (DM x time) peak stage over
the 1-D candidates (reading A18), and the end-to-end entry point that returns the candidate list."""
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


@pytest.mark.parametrize("K", [1, 3, 8, 9, 11, 14, 15, 16])
def test_uint8_width_plane_equals_int32_plane(spd, oracle_lib, K):
    """SPD_FLAG_WIDTH_U8: the same kernels store W as one byte per sample (4 per 32-bit store); Y is
    bit-identical, W equal value for value (no-fit samples: 255 for -1), on both tree kernels, with a ragged
    tail and several segments; candidates read the byte plane."""
    M = 1 << (K - 1)
    n_dm, n_t = 3, max(2048 * 5 + 4 * 9, 2 * M + 2048 + 12)
    rng = np.random.default_rng(60 + K)
    x = rng.standard_normal((n_dm, n_t)).astype(np.float32)
    x[1, n_t // 2: n_t // 2 + max(1, M // 2)] += np.float32(14.0 / np.sqrt(max(1, M // 2)))
    widths = [1 << k for k in range(K)]
    if K > 1:
        widths_no1 = None
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    mean = torch.zeros(n_dm, device=dev)
    sigma = torch.full((n_dm,), 1.25, device=dev)
    with spd.Plan(n_dm, n_t, widths, M) as p32, spd.Plan(n_dm, n_t, widths, M, flags=spd.SPD_FLAG_WIDTH_U8) as p8:
        assert p8.info["width_bytes"] == 1 and p32.info["width_bytes"] == 4
        assert p8.info["tree_kernel"] == p32.info["tree_kernel"]
        for segs in (0, 2):
            p32.set_option(spd.SPD_OPT_SEGMENTS_PER_ROW, segs)
            p8.set_option(spd.SPD_OPT_SEGMENTS_PER_ROW, segs)
            s32, w32, a32 = p32.run_flagged(plane, mean, sigma, 5.0)
            s8, w8, a8 = p8.run_flagged(plane, mean, sigma, 5.0)
            assert w8.dtype == torch.uint8 and w8.shape == (n_dm, n_t)
            assert torch.equal(s32, s8) and torch.equal(a32, a8)
            assert torch.equal(w32.to(torch.int64), w8.to(torch.int64))
            l32, n32 = p32.find_candidates_flagged(s32, w32, a32, 5.0, 1 << 16)
            l8, n8 = p8.find_candidates_flagged(s8, w8, a8, 5.0, 1 << 16)
            c32, g32 = spd.candidates_to_numpy(l32, n32, 1 << 16)
            c8, g8 = spd.candidates_to_numpy(l8, n8, 1 << 16)
            assert c32 == c8 and c8 > 0 and np.array_equal(g32, g8)
            ld, nd = p8.find_candidates(s8, w8, 5.0, 1 << 16)
            cd, gd = spd.candidates_to_numpy(ld, nd, 1 << 16)
            assert cd == c8 and np.array_equal(gd, g8)
        got_snr, got_idx = s8.cpu().numpy(), w8.cpu().numpy().astype(np.int32)
    ref = oracle_lib.spd_prefix(x, 0.0, 1.25, widths)
    parity.assert_parity(oracle_lib, x, 0.0, 1.25, widths, got_snr, got_idx, *ref, what=f"uint8 index K={K}")


def test_uint8_width_plane_needs_a_tree_plan(spd):
    with pytest.raises(spd.SpdError):
        spd.Plan(2, 4096, [1, 2, 3], 3, flags=spd.SPD_FLAG_WIDTH_U8)
    with pytest.raises(spd.SpdError):
        spd.Plan(2, 4096, [1, 2, 4], 4, flags=spd.SPD_FLAG_WIDTH_U8 | spd.SPD_FLAG_FORCE_GENERIC)
    with pytest.raises(spd.SpdError):
        spd.Plan(2, 4098, [1, 2, 4], 4, flags=spd.SPD_FLAG_WIDTH_U8)          # n_t % 4 != 0: any-width-set path


def _cluster_both(spd, oracle_lib, plan, snr, idx, act, thr, R, cap=1 << 20):
    lst, n_f = plan.find_candidates_flagged(snr, idx, act, thr, cap)
    count, cands = spd.candidates_to_numpy(lst, n_f, cap)
    lst2, n2 = plan.cluster_candidates(snr, lst, n_f, cap, R, cap)
    kept_count, kept = spd.candidates_to_numpy(lst2, n2, cap)
    keep = oracle_lib.cluster_candidates(snr.cpu().numpy(), plan.widths, cands["dm"], cands["t"], cands["width_idx"], R)
    want = cands[keep]
    assert kept_count == int(keep.sum()), (kept_count, int(keep.sum()), count)
    assert np.array_equal(kept, want)
    return count, kept


@pytest.mark.parametrize("cfg,n_dm,n_t,thr,R", [(3, 8, 262144, 6.0, 1), (3, 5, 65536 + 4 * 7, 4.0, 2),
                                                 (2, 16, 65536, 5.0, 0), (5, 4, 262144, 6.0, 1)])
def test_cluster_stage_matches_oracle_on_the_cuda_plane(spd, oracle_lib, cfg, n_dm, n_t, thr, R):
    """Row f4: spd_cluster_candidates against oracle_cluster_candidates (reading A18) on the plane the CUDA
    path produced - bit-exact list.  Config recipes with pulses; config 5's drift floods the threshold."""
    from workloads import get_workload, make_plane_numpy
    w = get_workload(cfg).scaled(n_dm, n_t, 10)
    x, pulses = make_plane_numpy(w)
    widths = spd.spd_width_set_generate(w.width_kind, w.width_param, min(w.max_width, 8192))
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    mean, sigma = torch.zeros(n_dm, device=dev), torch.ones(n_dm, device=dev)
    with spd.Plan(n_dm, n_t, widths) as plan:
        snr, idx, act = plan.run_flagged(plane, mean, sigma, thr)
        count, kept = _cluster_both(spd, oracle_lib, plan, snr, idx, act, thr, R)
    assert 0 < len(kept) < count
    if cfg == 3 and thr >= 6.0:
        # every injected pulse above the threshold leaves at least one cluster at its place, and the
        # list has the order of magnitude of the pulse count, not of the 1-D peak count
        assert len(kept) <= 4 * len(pulses) + 8 and count > 5 * len(kept)


def test_cluster_stage_smeared_pulse_and_ties(spd, oracle_lib):
    """A pulse smeared over neighbouring DM rows collapses to the single highest sample (dm_radius 1); with
    dm_radius 0 every row keeps its own peak; exact ties (noise-free plateaus) keep the first in (dm, t)."""
    n_dm, n_t = 7, 16384
    x = np.zeros((n_dm, n_t), dtype=np.float32)
    for d, amp in zip(range(1, 6), [1.0, 1.6, 2.2, 1.7, 0.9]):
        x[d, 5000 + 3 * d: 5000 + 3 * d + 64] = np.float32(amp)
    x[6, 12000:12016] = np.float32(2.0)
    x[0, 12000:12016] = np.float32(2.0)
    widths = [1 << k for k in range(10)]
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    mean, sigma = torch.zeros(n_dm, device=dev), torch.ones(n_dm, device=dev)
    with spd.Plan(n_dm, n_t, widths) as plan:
        snr, idx, act = plan.run_flagged(plane, mean, sigma, 5.0)
        _, kept1 = _cluster_both(spd, oracle_lib, plan, snr, idx, act, 5.0, 1)
        _, kept0 = _cluster_both(spd, oracle_lib, plan, snr, idx, act, 5.0, 0)
    big = kept1[(kept1["t"] > 4000) & (kept1["t"] < 6000)]
    assert len(big) == 1 and big[0]["dm"] == 3 and big[0]["t"] == 5009 and widths[big[0]["width_idx"]] == 64
    rows0 = sorted(set(kept0[(kept0["t"] > 4000) & (kept0["t"] < 6000)]["dm"].tolist()))
    assert rows0 == [1, 2, 3, 4, 5]
    far = kept1[kept1["t"] > 11000]
    assert sorted(far["dm"].tolist()) == [0, 6] and set(far["t"].tolist()) == {12000}


@pytest.mark.parametrize("cfg,n_dm,n_t,R", [(3, 40, 131072, 1), (2, 24, 65536, -1), (4, 6, 262144, 0)])
def test_run_host_candidates_equals_the_device_path(spd, oracle_lib, cfg, n_dm, n_t, R):
    """spd_run_host_candidates (H2D of row blocks, rows a1-a8 per block, row f4 over the whole list, D2H of the
    list only) returns the list the device-buffer calls give on the same plane; several row blocks."""
    from workloads import get_workload, make_plane_numpy
    w = get_workload(cfg).scaled(n_dm, n_t, 12)
    x, _ = make_plane_numpy(w)
    widths = spd.spd_width_set_generate(w.width_kind, w.width_param, min(w.max_width, n_t // 4))
    rng = np.random.default_rng(5)
    mu = (0.02 * rng.standard_normal(n_dm)).astype(np.float32)
    sg = (1.0 + 0.2 * rng.random(n_dm)).astype(np.float32)
    dev = torch.device("cuda:0")
    cap = 1 << 18
    with spd.Plan(n_dm, n_t, widths) as plan:
        plane = torch.from_numpy(x).to(dev)
        mean, sigma = torch.from_numpy(mu).to(dev), torch.from_numpy(sg).to(dev)
        snr, idx, act = plan.run_flagged(plane, mean, sigma, 6.0)
        lst, n_f = plan.find_candidates_flagged(snr, idx, act, 6.0, cap)
        count1, want = spd.candidates_to_numpy(lst, n_f, cap)
        if R >= 0:
            lst2, n2 = plan.cluster_candidates(snr, lst, n_f, cap, R, cap)
            _, want = spd.candidates_to_numpy(lst2, n2, cap)
        n_found, n_1d, got = plan.run_host_candidates(x, mu, sg, 6.0, R, cap)
        assert n_1d == count1 and n_found == len(want) and n_found > 0
        assert np.array_equal(got, want)
        # several row blocks (a ragged last one), alternating between the two staging streams
        plan.set_option(spd.SPD_OPT_HOST_ROWS_PER_BLOCK, 7)
        n_found, n_1d, got = plan.run_host_candidates(x, mu, sg, 6.0, R, cap)
        assert n_1d == count1 and n_found == len(want) and np.array_equal(got, want)
        # and the plane-returning host call agrees with the device planes
        out_snr = np.empty((n_dm, n_t), dtype=np.float32)
        out_idx = np.empty((n_dm, n_t), dtype=np.int32)
        plan.run_host(x, mu, sg, out_snr, out_idx)
        assert np.array_equal(out_snr, snr.cpu().numpy()) and np.array_equal(out_idx, idx.cpu().numpy())
