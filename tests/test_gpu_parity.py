"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element,
on the same seeded inputs.  Sizes here are ones the oracle finishes in seconds; the
full BASELINE.json sizes are in test_gpu_full_size.py.
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


def run_gpu(spd, x: np.ndarray, mu, sg, widths, max_width=None, flags=0, segs=0):
    """One spd_run through the binding; returns (snr f32, idx i32) numpy arrays and plan info.
    segs > 0: SPD_OPT_SEGMENTS_PER_ROW (every row cut into that many streams); 0: the default work split."""
    n_dm, n_t = x.shape
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32)).to(dev)
    mean = torch.from_numpy(np.broadcast_to(np.asarray(mu, dtype=np.float32), (n_dm,)).copy()).to(dev)
    sigma = torch.from_numpy(np.broadcast_to(np.asarray(sg, dtype=np.float32), (n_dm,)).copy()).to(dev)
    with spd.Plan(n_dm, n_t, widths, max_width, flags) as plan:
        if segs:
            plan.set_option(spd.SPD_OPT_SEGMENTS_PER_ROW, segs)
        snr, idx = plan.run(plane, mean, sigma)
        torch.cuda.synchronize()
        return snr.cpu().numpy().astype(np.float32), idx.cpu().numpy().astype(np.int32), dict(plan.info)


def check(spd, oracle, x, mu, sg, widths, what, direct=False, flags=0, expect_path=None, segs=0,
          direct_windows=()):
    """Element-by-element parity of one run against oracle B (running sum) or, direct=True, oracle A (direct
    summation); direct_windows = [(t0, t1), ...] adds oracle A on those sample ranges of every row."""
    got_snr, got_idx, info = run_gpu(spd, x, mu, sg, widths, flags=flags, segs=segs)
    if expect_path is not None:
        assert info["path"] == expect_path, f"{what}: plan took path {info['path']}"
    # both sides see the float32-rounded mu / sigma the C ABI takes
    mu64 = np.broadcast_to(np.asarray(mu, dtype=np.float32), (x.shape[0],)).astype(np.float64)
    sg64 = np.broadcast_to(np.asarray(sg, dtype=np.float32), (x.shape[0],)).astype(np.float64)
    fn = oracle.spd_direct if direct else oracle.spd_prefix
    ref_snr, ref_idx, ref_sec = fn(x, mu64, sg64, widths)
    st = parity.assert_parity(oracle, x, mu64, sg64, widths, got_snr, got_idx, ref_snr, ref_idx, ref_sec,
                              what=what)
    for t0, t1 in direct_windows:
        d_snr, d_idx, d_sec = oracle.spd_direct(x, mu64, sg64, widths, t0, t1)
        parity.assert_parity(oracle, x, mu64, sg64, widths, got_snr[:, t0:t1], got_idx[:, t0:t1], d_snr, d_idx,
                             d_sec, t0=t0, what=f"{what} direct [{t0}, {t1})")
    return st


def test_config1_tiny_lossless_full_plane(spd, oracle_lib):
    """BASELINE.json configs[0], whole plane, against the direct-summation oracle."""
    from workloads import get_workload, make_plane_numpy
    w = get_workload(1)
    x, _ = make_plane_numpy(w)
    widths = spd.spd_width_set_generate(w.width_kind, w.width_param, w.max_width)
    assert list(widths) == list(range(1, 65))
    st = check(spd, oracle_lib, x, 0.0, 1.0, widths, "config1/all-widths", direct=True,
               expect_path=spd.SPD_PATH_GENERIC)
    assert st.n == 64 * 16384


def test_config1_plane_dyadic_set_direct_oracle(spd, oracle_lib):
    from workloads import get_workload, make_plane_numpy
    x, _ = make_plane_numpy(get_workload(1))
    widths = spd.spd_width_set_generate("POW2", 0, 64)
    check(spd, oracle_lib, x, 0.0, 1.0, widths, "config1/pow2", direct=True, expect_path=spd.SPD_PATH_DYADIC_TREE)


@pytest.mark.parametrize("segs", [0, 3])
@pytest.mark.parametrize("K", list(range(1, 17)))
def test_dyadic_tree_every_depth_ragged(spd, oracle_lib, K, segs):
    """Every kernel instantiation (widths 1..2^(K-1)); n_t spans several chunks plus a ragged
    tail that is not a multiple of the chunk; with the default work split (segs 0) and with several
    segments per row, so that interior segments replay their look-ahead."""
    M = 1 << (K - 1)
    T = 128 if K <= 14 else (256 if K == 15 else 512)
    chunk = 16 * T
    n_t = max(5 * chunk + 4 * 37, 2 * M + chunk + 4 * 5)
    rng = np.random.default_rng(1000 + K)
    x = rng.standard_normal((3, n_t), dtype=np.float32)
    x[1, n_t // 3: n_t // 3 + max(1, M // 2)] += np.float32(12.0 / np.sqrt(max(1, M // 2)))
    x[2, n_t - M // 2 - 3:] += np.float32(0.7)  # a pulse running off the end of the row
    widths = [1 << k for k in range(K)]
    check(spd, oracle_lib, x, 0.0, 1.0, widths, f"tree K={K} segs={segs}", expect_path=spd.SPD_PATH_DYADIC_TREE,
          segs=segs)


@pytest.mark.parametrize("segs", [0, 3])
@pytest.mark.parametrize("K", list(range(5, 17)))
def test_igrid_tree_every_depth_ragged(spd, oracle_lib, K, segs):
    """Every instantiation of the IGRID depth-1 streaming tree (widths 2^k and 3 * 2^m up to 2^(K-1)):
    several chunks, ragged tail, several segments per row, pulses of non-power-of-two widths."""
    M = 1 << (K - 1)
    chunk = 4096
    n_t = max(5 * chunk + 4 * 37, 2 * M + chunk + 4 * 5)
    rng = np.random.default_rng(2000 + K)
    x = rng.standard_normal((3, n_t), dtype=np.float32)
    S = max(1, 3 * M // 8)
    x[1, n_t // 3: n_t // 3 + S] += np.float32(12.0 / np.sqrt(S))
    x[2, n_t - M // 2 - 3:] += np.float32(0.7)  # a pulse running off the end of the row
    widths = spd.spd_width_set_generate("IGRID", 1, M)
    assert len(widths) == 2 * K - 2
    check(spd, oracle_lib, x, 0.0, 1.0, widths, f"igrid tree K={K} segs={segs}",
          expect_path=spd.SPD_PATH_IGRID_TREE, segs=segs)


@pytest.mark.parametrize("segs", [1, 2, 5])
def test_igrid_tree_segmentation_and_statistics(spd, oracle_lib, segs):
    rng = np.random.default_rng(78)
    n_t = 2048 * 19 + 4 * 3
    x = (rng.standard_normal((2, n_t)) * 3.1 - 17.0).astype(np.float32)
    x[0, 9000:9000 + 96] += np.float32(4.0)  # width 96 = 3 * 32 is in the set
    mu, sg = oracle_lib.row_stats(x)
    widths = spd.spd_width_set_generate("IGRID", 1, 4096)
    check(spd, oracle_lib, x, mu, sg, widths, f"igrid tree segs={segs}", expect_path=spd.SPD_PATH_IGRID_TREE,
          segs=segs)


def test_igrid_tree_exact_ties_and_plateau(spd, oracle_lib):
    """Zero background: exact ties resolve to the smallest width; a width-24 pulse is recovered exactly
    by the width-24 boxcar (index 8 of 1,2,3,4,6,8,12,16,24)."""
    n_t = 8192
    x = np.zeros((2, n_t), dtype=np.float32)
    x[1, 1000:1024] = np.float32(2.0)
    widths = list(spd.spd_width_set_generate("IGRID", 1, 64))
    got_snr, got_idx, info = run_gpu(spd, x, 0.0, 1.0, widths)
    assert info["path"] == spd.SPD_PATH_IGRID_TREE
    assert np.all(got_snr[0] == 0.0) and np.all(got_idx[0, : n_t - 64] == 0)
    assert got_idx[1, 1000] == widths.index(24)
    assert abs(got_snr[1, 1000] - 2.0 * np.sqrt(24.0)) < 1e-4 * 2.0 * np.sqrt(24.0)
    ref_snr, ref_idx, ref_sec = oracle_lib.spd_direct(x, 0.0, 1.0, widths)
    parity.assert_parity(oracle_lib, x, 0.0, 1.0, widths, got_snr, got_idx, ref_snr, ref_idx, ref_sec, what="ig ties")


def test_igrid_tree_flagged_candidates(spd, oracle_lib):
    from workloads import get_workload, make_plane_numpy
    w = get_workload(3).scaled(4, 131072, 10)
    x, _ = make_plane_numpy(w)
    widths = spd.spd_width_set_generate("IGRID", 1, 8192)
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    mean, sigma = torch.zeros(4, device=dev), torch.ones(4, device=dev)
    with spd.Plan(4, 131072, widths) as plan:
        assert plan.info["path"] == spd.SPD_PATH_IGRID_TREE
        snr, idx, act = plan.run_flagged(plane, mean, sigma, 6.0)
        lst, n_f = plan.find_candidates_flagged(snr, idx, act, 6.0, 1 << 16)
        count, got = spd.candidates_to_numpy(lst, n_f, 1 << 16)
        ref_count, c_dm, c_t, c_snr, c_w = oracle_lib.find_candidates(snr.cpu().numpy(), idx.cpu().numpy(), 6.0)
        assert count == ref_count and count > 0
        assert np.array_equal(got["dm"], c_dm) and np.array_equal(got["t"], c_t)


@pytest.mark.parametrize("seed", list(range(10)))
def test_random_shapes_and_statistics(spd, oracle_lib, seed):
    """Seeded fuzz over plane shapes, depths, segmentation, width-set family and statistics: row lengths
    that are not multiples of the chunk, rows shorter than a chunk or barely longer than max_width."""
    rng = np.random.default_rng(9000 + seed)
    family = ["POW2", "IGRID"][seed % 2]
    K = int(rng.integers(5, 15))
    M = 1 << (K - 1)
    n_dm = int(rng.integers(1, 6))
    n_t = 4 * int(rng.integers((M + 3) // 4, (M + 3) // 4 + 6000))
    x = (rng.standard_normal((n_dm, n_t)) * rng.uniform(0.5, 4.0) + rng.uniform(-30, 30)).astype(np.float32)
    for _ in range(3):
        S = int(rng.integers(1, M + 1))
        t0 = int(rng.integers(0, n_t - 1))
        x[int(rng.integers(0, n_dm)), t0:t0 + S] += np.float32(rng.uniform(5, 15) / np.sqrt(S) * x.std())
    mu, sg = oracle_lib.row_stats(x)
    segs = int(rng.integers(0, 5))  # 0: the default work split
    widths = spd.spd_width_set_generate(family, 1 if family == "IGRID" else 0, M)
    check(spd, oracle_lib, x, mu, sg, widths, f"fuzz seed={seed} {family} K={K} {n_dm}x{n_t} segs={segs}",
          expect_path=spd.SPD_PATH_IGRID_TREE if family == "IGRID" else spd.SPD_PATH_DYADIC_TREE, segs=segs)


@pytest.mark.parametrize("segs", [1, 2, 7])
def test_dyadic_tree_segmentation_is_invisible(spd, oracle_lib, segs):
    rng = np.random.default_rng(77)
    n_t = 2048 * 23 + 4 * 3
    x = rng.standard_normal((2, n_t), dtype=np.float32)
    check(spd, oracle_lib, x, 0.0, 1.0, [1 << k for k in range(12)], f"tree segs={segs}", segs=segs)


def test_small_lossy_measured_statistics(spd, oracle_lib):
    """Config-2 recipe on a reduced plane: mu, sigma measured by the oracle's definition
    (reading A6) on data with a large offset and scale."""
    from workloads import get_workload, make_plane_numpy
    w = get_workload(2).scaled(16, 65536, 8)
    x, _ = make_plane_numpy(w)
    x = (x * np.float32(3.7) + np.float32(41.5)).astype(np.float32)
    mu, sg = oracle_lib.row_stats(x)
    widths = spd.spd_width_set_generate(w.width_kind, w.width_param, w.max_width)
    check(spd, oracle_lib, x, mu, sg, widths, "config2-recipe/tree")
    check(spd, oracle_lib, x, mu, sg, widths, "config2-recipe/generic", flags=spd.SPD_FLAG_FORCE_GENERIC,
          expect_path=spd.SPD_PATH_GENERIC)


@pytest.mark.parametrize("kind,param,max_width", [("IGRID", 1, 256), ("IGRID", 2, 512), ("BOXDIT", 8, 300),
                                                    ("GEOMETRIC", 1800, 1000), ("ALL", 0, 37)])
def test_generic_width_sets(spd, oracle_lib, kind, param, max_width):
    rng = np.random.default_rng(5)
    x = rng.standard_normal((5, 10007), dtype=np.float32)  # n_t odd: tree not applicable anyway
    x[2, 5000:5100] += np.float32(1.5)
    widths = spd.spd_width_set_generate(kind, param, max_width)
    # oracle B on the whole plane, oracle A (direct summation) around the pulse and on the row tail
    check(spd, oracle_lib, x, 0.0, 1.0, widths, f"generic {kind}({param})<= {max_width}",
          expect_path=spd.SPD_PATH_GENERIC, direct_windows=[(4900, 5200), (10007 - 300, 10007)])


DENSE_SETS = {"all64": list(range(1, 65)), "all37": list(range(1, 38)), "one": [1], "only64": [64],
              "fib": [1, 2, 3, 5, 8, 13, 21, 34, 55], "odd": list(range(3, 64, 2)), "boxdit4": None}


@pytest.mark.parametrize("n_t", [4, 60, 1024, 1028, 2048 + 64, 10008])
@pytest.mark.parametrize("name", list(DENSE_SETS))
def test_dense_kernel_small_width_sets(spd, oracle_lib, name, n_t):
    """Width sets with max_width <= 64 (config 1's family) run on spd_dense_kernel (running sums in registers,
    one 1024-sample tile per block): direct-summation oracle on every sample, row lengths inside one tile, on a
    tile boundary, just past it (a one-float4 last tile) and with a look-ahead that ends inside the halo; sets
    without width 1 leave -inf / -1 at the row's end (reading A3)."""
    widths = [L for L in DENSE_SETS[name] or spd.spd_width_set_generate("BOXDIT", 4, 64) if L <= n_t]
    if not widths:
        pytest.skip("no width of the set fits the row")
    rng = np.random.default_rng(n_t + len(widths))
    x = (rng.standard_normal((3, n_t)) * 2.0 + 7.0).astype(np.float32)
    if n_t > 200:
        x[1, 100:140] += np.float32(3.0)
        x[2, n_t - 30:] += np.float32(2.0)
    mu, sg = oracle_lib.row_stats(x)
    force = spd.SPD_FLAG_FORCE_GENERIC   # [1] is also a {2^k} set
    with spd.Plan(3, n_t, widths, flags=force) as plan:
        assert plan.info["path"] == spd.SPD_PATH_GENERIC and plan.info["threads_per_block"] == 256
        assert plan.info["launches_per_run"] == 1 and plan.info["blocks"] == 3 * ((n_t + 1023) // 1024)
    check(spd, oracle_lib, x, mu, sg, widths, f"dense {name} n_t={n_t}", direct=True, flags=force,
          expect_path=spd.SPD_PATH_GENERIC)


def test_dense_kernel_with_measured_sigma_per_width(spd, oracle_lib):
    """spd_run_sigma_w on the dense kernel: all 64 widths (more than the tile kernel's table holds)."""
    n_dm, n_t = 3, 20000
    x = _plane_for_sigma_w(n_dm, n_t, 41)
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    widths = list(range(1, 65))
    with spd.Plan(n_dm, n_t, widths) as plan:
        mean, _ = plan.row_stats(plane)
        sw = plan.width_sigma(plane, mean)
        snr, idx = plan.run_sigma_w(plane, mean, sw)
        torch.cuda.synchronize()
    mu64 = mean.cpu().numpy().astype(np.float64)
    sw64 = sw.cpu().numpy().astype(np.float64)
    ref = oracle_lib.spd_direct_sw(x, mu64, sw64, widths)
    parity.assert_parity_table(oracle_lib, x, mu64, sw64, widths, None, snr.cpu().numpy(), idx.cpu().numpy(), *ref,
                               what="sigma_w dense")


def test_generic_tile_kernel_wide_sets_and_tile_boundaries(spd, oracle_lib):
    """Any-width-set tile kernel: max_width in the thousands (several tiles per row, ragged last tile,
    look-ahead longer than the tile's remainder), on drifting data with a large offset."""
    rng = np.random.default_rng(31)
    n_dm, n_t = 3, 150001
    x = (rng.standard_normal((n_dm, n_t)) + 0.2 * np.sin(np.arange(n_t) / 9000.0) + 25.0).astype(np.float32)
    x[1, 60000:63000] += np.float32(0.4)
    x[2, n_t - 2500:] += np.float32(0.3)  # runs off the end of the row
    mu, sg = oracle_lib.row_stats(x)
    for kind, param, mw in [("IGRID", 1, 8192), ("BOXDIT", 16, 3000), ("GEOMETRIC", 1500, 20000)]:
        widths = spd.spd_width_set_generate(kind, param, mw)
        st = check(spd, oracle_lib, x, mu, sg, widths, f"tile {kind}({param})<= {mw}",
                   expect_path=spd.SPD_PATH_GENERIC, direct_windows=[(62900, 63100), (n_t - 150, n_t)])
        assert st.max_err_over_tol < 0.5


def test_generic_workspace_fallback(spd, oracle_lib):
    """The running-sum-in-device-memory kernels (used when max_width does not fit a shared-memory tile;
    SPD_FLAG_GENERIC_WORKSPACE selects them on a small plane)."""
    rng = np.random.default_rng(32)
    x = rng.standard_normal((4, 30011), dtype=np.float32)
    x[3, 1000:1400] += np.float32(0.8)
    widths = spd.spd_width_set_generate("IGRID", 2, 1024)
    got_snr, got_idx, info = run_gpu(spd, x, 0.0, 1.0, widths, flags=spd.SPD_FLAG_GENERIC_WORKSPACE)
    assert info["launches_per_run"] == 4 and info["workspace_bytes"] > 8 * 4 * 30011
    got_snr2, got_idx2, info2 = run_gpu(spd, x, 0.0, 1.0, widths)
    assert info2["launches_per_run"] == 1
    ref_snr, ref_idx, ref_sec = oracle_lib.spd_prefix(x, 0.0, 1.0, widths)
    d_snr, d_idx, d_sec = oracle_lib.spd_direct(x, 0.0, 1.0, widths, 900, 1500)   # oracle A around the pulse
    for gs, gi, what in ((got_snr, got_idx, "workspace"), (got_snr2, got_idx2, "tile")):
        parity.assert_parity(oracle_lib, x, 0.0, 1.0, widths, gs, gi, ref_snr, ref_idx, ref_sec, what=what)
        parity.assert_parity(oracle_lib, x, 0.0, 1.0, widths, gs[:, 900:1500], gi[:, 900:1500], d_snr, d_idx, d_sec,
                             t0=900, what=what + " direct")


def test_width_set_generators_agree_with_formula_module(spd):
    from oracle import formulas
    for kind, param, mw in [("ALL", 0, 64), ("POW2", 0, 8192), ("BOXDIT", 4, 12), ("BOXDIT", 8, 8192),
                            ("IGRID", 1, 8192), ("IGRID", 3, 32768), ("GEOMETRIC", 1800, 8192)]:
        assert list(spd.spd_width_set_generate(kind, param, mw)) == formulas.width_set(kind, param, mw), (kind, param)


def test_tail_rule_without_width_one(spd, oracle_lib):
    """Reading A3: widths that do not fit are skipped; with 1 not in the set the last samples
    have no valid width: -inf / -1."""
    rng = np.random.default_rng(9)
    x = rng.standard_normal((2, 64), dtype=np.float32)
    got_snr, got_idx, _ = run_gpu(spd, x, 0.0, 1.0, [4, 8])
    assert np.all(np.isneginf(got_snr[:, 61:])) and np.all(got_idx[:, 61:] == -1)
    check(spd, oracle_lib, x, 0.0, 1.0, [4, 8], "tail/no-width-1", direct=True)


@pytest.mark.parametrize("n_t", [4, 8, 64, 2044, 2048, 2052])
def test_tiny_and_chunk_boundary_lengths(spd, oracle_lib, n_t):
    rng = np.random.default_rng(n_t)
    x = rng.standard_normal((1, n_t), dtype=np.float32)
    K = min(4, int(np.log2(n_t)) + 1)
    check(spd, oracle_lib, x, 0.0, 1.0, [1 << k for k in range(K)], f"tree n_t={n_t}", direct=True,
          expect_path=spd.SPD_PATH_DYADIC_TREE)


def test_max_width_equals_row_length(spd, oracle_lib):
    rng = np.random.default_rng(3)
    x = rng.standard_normal((2, 4096), dtype=np.float32)
    check(spd, oracle_lib, x, 0.0, 1.0, [1 << k for k in range(13)], "tree M == n_t", direct=True)


def test_exact_ties_take_the_smallest_width(spd, oracle_lib):
    """Zero background (every SNR exactly 0) and a noise-free pulse: exact ties resolve to
    the smallest width on both paths (reading A4)."""
    n_t = 8192
    x = np.zeros((2, n_t), dtype=np.float32)
    x[1, 1000:1016] = np.float32(2.0)
    for f in (0, spd.SPD_FLAG_FORCE_GENERIC):
        got_snr, got_idx, _ = run_gpu(spd, x, 0.0, 1.0, [1, 2, 4, 8, 16, 32, 64], flags=f)
        assert np.all(got_snr[0] == 0.0) and np.all(got_idx[0, : n_t - 64] == 0)
        ref_snr, ref_idx, ref_sec = oracle_lib.spd_direct(x, 0.0, 1.0, [1, 2, 4, 8, 16, 32, 64])
        parity.assert_parity(oracle_lib, x, 0.0, 1.0, [1, 2, 4, 8, 16, 32, 64], got_snr, got_idx, ref_snr,
                             ref_idx, ref_sec, what=f"ties flags={f}")
        # exact comparison of the index on the noise-free plane, away from float near-ties:
        # dyadic sums of 2.0 are exact in fp32, so the decision is exact on both sides
        assert np.array_equal(got_idx, ref_idx)


def test_constant_offset_closed_form(spd):
    """x = mu + a: SNR_L = a sqrt(L) / sigma, so the largest width that fits wins (pin P10)."""
    n_t, a, sg = 4096, 0.25, 2.0
    x = np.full((1, n_t), 10.0 + a, dtype=np.float32)
    widths = [1 << k for k in range(9)]
    got_snr, got_idx, _ = run_gpu(spd, x, 10.0, sg, widths)
    room = n_t - np.arange(n_t)
    exp_idx = np.minimum(8, np.floor(np.log2(room)).astype(np.int64))
    exp_snr = a * np.sqrt(2.0 ** exp_idx) / sg
    assert np.array_equal(got_idx[0], exp_idx)
    assert np.all(np.abs(got_snr[0] - exp_snr) <= 1e-4 * np.maximum(1, exp_snr))


@pytest.mark.parametrize("shape", ["gauss", "double_gauss"])
@pytest.mark.parametrize("kind,param", [("POW2", 0), ("IGRID", 1)])
def test_other_pulse_shapes_parity(spd, oracle_lib, shape, kind, param):
    """Row f3: Gaussian and double-Gaussian pulses of the config-3 recipe, on a zero
    background and on noise - CUDA planes against the oracle's (no closed form exists for these shapes:
    the oracle itself is pinned to the paper's worked example in test_oracle_pins.py)."""
    from workloads import get_workload
    from workloads.generate import make_shaped_pulse_plane_numpy
    w = get_workload(3).scaled(4, 131072, 12)
    widths = spd.spd_width_set_generate(kind, param, w.max_width)
    for noise in (False, True):
        x, pulses = make_shaped_pulse_plane_numpy(w, shape, noise=noise)
        st = check(spd, oracle_lib, x, 0.0, 1.0, widths, f"{shape} {kind} noise={noise}")
        assert st.max_err_over_tol < 0.5
    # on the zero background every isolated pulse is recovered ABOVE its SNR_T or within the set's loss of it
    x, pulses = make_shaped_pulse_plane_numpy(w, shape, noise=False)
    got_snr, got_idx, _ = run_gpu(spd, x, 0.0, 1.0, widths)
    for p in pulses:
        if p.width < 8:
            continue
        lo, hi = max(0, p.t0 - w.max_width), min(w.n_t, p.t0 + p.width)
        assert float(got_snr[p.dm, lo:hi].max()) > 0.9 * p.snr_t


@pytest.mark.parametrize("kind", ["config", "IGRID1"])
@pytest.mark.parametrize("cfg,n_dm,n_t,n_pulses", [(2, 8, 32768, 16), (3, 4, 262144, 12), (4, 2, 524288, 6)])
def test_noise_free_twin_loss_matches_eq24(spd, cfg, n_dm, n_t, n_pulses, kind):
    """Pin P14 through the CUDA path: on a zero-background plane each injected rectangular
    pulse is recovered at exactly eq. (24)'s fraction of its true SNR,
    and the mean loss equals the formula's mean over the injected widths."""
    from oracle import formulas
    from workloads import get_workload, make_pulse_only_plane_numpy
    w = get_workload(cfg).scaled(n_dm, n_t, n_pulses)
    x, pulses = make_pulse_only_plane_numpy(w)
    if kind == "IGRID1":  # the paper's IG(1) width set on the same pulses (IGRID streaming tree)
        widths = list(spd.spd_width_set_generate("IGRID", 1, w.max_width))
    else:
        widths = list(spd.spd_width_set_generate(w.width_kind, w.width_param, w.max_width))
    got_snr, _, info = run_gpu(spd, x, 0.0, 1.0, widths)
    assert info["path"] == (spd.SPD_PATH_IGRID_TREE if kind == "IGRID1" else spd.SPD_PATH_DYADIC_TREE)
    losses, predicted = [], []
    for p in pulses:
        others = [q for q in pulses if q is not p and q.dm == p.dm and
                  abs(q.t0 - p.t0) < 2 * w.max_width + p.width + q.width]
        if others:
            continue  # overlapping pulses do not follow the single-pulse formula
        lo, hi = max(0, p.t0 - w.max_width), min(n_t, p.t0 + p.width + 1)
        rec = float(got_snr[p.dm, lo:hi].max()) / p.snr_t
        exp = formulas.rsnr_max(p.width, widths)
        assert abs(rec - exp) <= 2e-4, (p, rec, exp)
        losses.append(1.0 - rec)
        predicted.append(1.0 - exp)
    assert len(losses) >= n_pulses // 2
    assert abs(np.mean(losses) - np.mean(predicted)) <= 1e-4


def test_candidates_match_rule_on_cuda_plane(spd, oracle_lib):
    """Row a8: on the SNR plane the CUDA path produced, the candidate list equals the
    reading-A9 rule evaluated by the oracle on that same float32 plane - bit-exact."""
    from workloads import get_workload, make_plane_numpy
    w = get_workload(5).scaled(4, 262144, 24)
    x, _ = make_plane_numpy(w)
    widths = spd.spd_width_set_generate(w.width_kind, w.width_param, w.max_width)
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    mean = torch.zeros(4, device=dev)
    sigma = torch.ones(4, device=dev)
    with spd.Plan(4, 262144, widths) as plan:
        snr, idx = plan.run(plane, mean, sigma)
        cap = 1 << 20  # the config-5 drift floods the threshold: stay below capacity
        lst, n_found = plan.find_candidates(snr, idx, 6.0, cap)
        count, got = spd.candidates_to_numpy(lst, n_found, cap)
        assert count <= cap
        snr_h, idx_h = snr.cpu().numpy(), idx.cpu().numpy()
        ref_count, c_dm, c_t, c_snr, c_w = oracle_lib.find_candidates(snr_h, idx_h, 6.0)
        assert count == ref_count and count > 0
        assert np.array_equal(got["dm"], c_dm) and np.array_equal(got["t"], c_t)
        assert np.array_equal(got["snr"], c_snr) and np.array_equal(got["width_idx"], c_w)
        # overflow: the count keeps running past a small capacity
        lst2, n2 = plan.find_candidates(snr, idx, 6.0, 5)
        count2, got2 = spd.candidates_to_numpy(lst2, n2, 5)
        assert count2 == ref_count and len(got2) == 5


def test_candidates_against_oracle_plane_tolerance_aware(spd, oracle_lib):
    """Candidates of the CUDA planes vs candidates of the ORACLE's planes (reading A9's
    tolerance-aware rule): every oracle candidate clear of the threshold has a CUDA candidate
    in the same row within +-width samples and SNR tolerance, and vice versa."""
    from workloads import get_workload, make_plane_numpy
    w = get_workload(2).scaled(8, 65536, 16)
    x, _ = make_plane_numpy(w)
    widths = list(spd.spd_width_set_generate(w.width_kind, w.width_param, w.max_width))
    thr = 6.0
    dev = torch.device("cuda:0")
    with spd.Plan(8, 65536, widths) as plan:
        snr, idx = plan.run(torch.from_numpy(x).to(dev), torch.zeros(8, device=dev), torch.ones(8, device=dev))
        lst, n_found = plan.find_candidates(snr, idx, thr, 1 << 16)
        count, got = spd.candidates_to_numpy(lst, n_found, 1 << 16)
    ref_snr, ref_idx, _ = oracle_lib.spd_prefix(x, 0.0, 1.0, widths)
    _, o_dm, o_t, o_snr, o_w = oracle_lib.find_candidates(ref_snr.astype(np.float32), ref_idx, thr)
    assert count > 0 and len(o_dm) > 0

    def covered(a_dm, a_t, a_snr, a_w, b_dm, b_t, b_snr):
        for d, t, s, k in zip(a_dm, a_t, a_snr, a_w):
            tol = parity.SNR_RTOL * max(1.0, abs(float(s)))
            if s < thr + 2 * tol:
                continue
            m = (b_dm == d) & (np.abs(b_t - t) <= widths[k]) & (np.abs(b_snr - s) <= 2 * tol)
            assert m.any(), f"candidate (dm={d}, t={t}, snr={s}, width={widths[k]}) has no counterpart"

    covered(o_dm, o_t, o_snr, o_w, got["dm"], got["t"], got["snr"])
    covered(got["dm"], got["t"], got["snr"], got["width_idx"], o_dm, o_t, o_snr)


def _activity_truth(snr_h, block, per_row, thr):
    """Per-block 'some Y >= thr' map of a host SNR plane."""
    n_dm, n_t = snr_h.shape
    pad = per_row * block - n_t
    y = np.pad(snr_h, ((0, 0), (0, pad)), constant_values=-np.inf) if pad else snr_h
    return (y.reshape(n_dm, per_row, block) >= thr).any(axis=2)


@pytest.mark.parametrize("cfg,n_dm,n_t,thr,segs", [(3, 6, 262144 + 4 * 11, 6.0, 0), (5, 4, 262144, 6.0, 3),
                                                     (2, 8, 65536, 4.5, 0), (3, 3, 40000, 3.0, 2)])
def test_flagged_run_equals_plain_run_and_dense_candidates(spd, oracle_lib, cfg, n_dm, n_t, thr, segs):
    """Row a8 fused: spd_run_flagged writes the same Y, W as spd_run; its activity map marks every block
    that holds a sample >= threshold (and may mark no block whose samples are all clearly below it);
    spd_find_candidates_flagged returns exactly the list of the visit-everything kernel, which equals
    the reading-A9 rule evaluated by the oracle on that plane."""
    from workloads import get_workload, make_plane_numpy
    w = get_workload(cfg).scaled(n_dm, n_t, 12)
    x, _ = make_plane_numpy(w)
    widths = spd.spd_width_set_generate(w.width_kind, w.width_param, min(w.max_width, 8192))
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    rng = np.random.default_rng(3)
    mean = torch.from_numpy((0.01 * rng.standard_normal(n_dm)).astype(np.float32)).to(dev)
    sigma = torch.from_numpy((1.0 + 0.3 * rng.random(n_dm)).astype(np.float32)).to(dev)
    cap = 1 << 20
    with spd.Plan(n_dm, n_t, widths) as plan:
        assert plan.info["path"] == spd.SPD_PATH_DYADIC_TREE
        if segs:
            plan.set_option(spd.SPD_OPT_SEGMENTS_PER_ROW, segs)
            assert plan.info["segments_per_row"] == segs
        snr0, idx0 = plan.run(plane, mean, sigma)
        snr, idx, act = plan.run_flagged(plane, mean, sigma, thr)
        assert torch.equal(snr0, snr) and torch.equal(idx0, idx)
        block, per_row = plan.info["activity_block"], plan.info["activity_per_row"]
        assert plan.info["activity_bytes"] % 128 == 0 and plan.info["activity_bytes"] >= n_dm * per_row
        snr_h = snr.cpu().numpy()
        act_h = act.cpu().numpy()
        assert not act_h[n_dm * per_row:].any(), "padding of the activity map must be cleared"
        got_map = act_h[: n_dm * per_row].reshape(n_dm, per_row) != 0
        must = _activity_truth(snr_h, block, per_row, thr)
        may = _activity_truth(snr_h, block, per_row, thr * (1 - 1e-5) - 1e-5)
        assert not (must & ~got_map).any(), "a block holding a sample >= threshold is not marked"
        assert not (got_map & ~may).any(), "a block clearly below the threshold is marked"
        lst_d, n_d = plan.find_candidates(snr, idx, thr, cap)
        count_d, dense = spd.candidates_to_numpy(lst_d, n_d, cap)
        lst_f, n_f = plan.find_candidates_flagged(snr, idx, act, thr, cap)
        count_f, flagged = spd.candidates_to_numpy(lst_f, n_f, cap)
        assert count_f == count_d and count_d > 0
        assert np.array_equal(dense, flagged)
        ref_count, c_dm, c_t, c_snr, c_w = oracle_lib.find_candidates(snr_h, idx.cpu().numpy(), thr)
        assert count_f == ref_count
        assert np.array_equal(flagged["dm"], c_dm) and np.array_equal(flagged["t"], c_t)
        assert np.array_equal(flagged["snr"], c_snr) and np.array_equal(flagged["width_idx"], c_w)
        # a higher threshold with the same (lower-threshold) map is allowed
        lst_h, n_h = plan.find_candidates_flagged(snr, idx, act, thr + 2.0, cap)
        count_h, _ = spd.candidates_to_numpy(lst_h, n_h, cap)
        assert count_h == oracle_lib.find_candidates(snr_h, idx.cpu().numpy(), thr + 2.0)[0]
        # overflow keeps counting
        lst_o, n_o = plan.find_candidates_flagged(snr, idx, act, thr, 3)
        count_o, got_o = spd.candidates_to_numpy(lst_o, n_o, 3)
        assert count_o == ref_count and len(got_o) == min(3, ref_count)


def test_flagged_run_generic_path_marks_everything(spd, oracle_lib):
    rng = np.random.default_rng(21)
    x = rng.standard_normal((3, 20001), dtype=np.float32)
    x[1, 7000:7030] += np.float32(2.0)
    widths = spd.spd_width_set_generate("IGRID", 1, 64)
    dev = torch.device("cuda:0")
    with spd.Plan(3, 20001, widths) as plan:
        assert plan.info["path"] == spd.SPD_PATH_GENERIC
        snr, idx, act = plan.run_flagged(torch.from_numpy(x).to(dev), torch.zeros(3, device=dev),
                                         torch.ones(3, device=dev), 5.0)
        assert bool((act != 0).all())
        lst, n_found = plan.find_candidates_flagged(snr, idx, act, 5.0, 1 << 16)
        count, got = spd.candidates_to_numpy(lst, n_found, 1 << 16)
        ref_count, c_dm, c_t, c_snr, c_w = oracle_lib.find_candidates(snr.cpu().numpy(), idx.cpu().numpy(), 5.0)
        assert count == ref_count and count > 0
        assert np.array_equal(got["dm"], c_dm) and np.array_equal(got["t"], c_t)


def test_flagged_no_detections_and_all_detections(spd):
    """Degenerate maps: nothing above the threshold (empty list, empty map) and everything above it."""
    rng = np.random.default_rng(22)
    x = (0.01 * rng.standard_normal((2, 32768))).astype(np.float32)
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    mean, sigma = torch.zeros(2, device=dev), torch.ones(2, device=dev)
    with spd.Plan(2, 32768, [1 << k for k in range(8)]) as plan:
        snr, idx, act = plan.run_flagged(plane, mean, sigma, 6.0)
        assert not bool(act.any())
        _, n0 = plan.find_candidates_flagged(snr, idx, act, 6.0, 16)
        assert int(n0.item()) == 0
        snr, idx, act = plan.run_flagged(plane, mean, sigma, -1e30)
        per_row = plan.info["activity_per_row"]
        assert bool((act[: 2 * per_row] != 0).all())
        _, n1 = plan.find_candidates_flagged(snr, idx, act, -1e30, 16)
        lst_d, n_d = plan.find_candidates(snr, idx, -1e30, 16)
        assert int(n1.item()) == int(n_d.item()) > 0


def _stats_plane(n_dm, n_t, seed):
    rng = np.random.default_rng(seed)
    x = (rng.standard_normal((n_dm, n_t)) * 2.5 + 11.0).astype(np.float32)
    x[0, n_t // 4: n_t // 4 + max(4, n_t // 50)] += np.float32(40.0)  # a strong wide pulse
    x[n_dm - 1, ::97] -= np.float32(25.0)                             # scattered outliers
    return x


def _assert_stats_close(got_mu, got_sg, ref_mu, ref_sg, n_border, n_t, clip):
    """The oracle decides |x - mu| <= clip sigma in double on unrounded estimates, the kernel in float32 on the
    float32 estimates it hands out.  Rows without a border-line sample (none within 1e-6 sigma of a limit in
    any pass) must agree to 2e-6 sigma; every border-line sample may change sides and then moves the mean
    by at most clip sigma / n_kept and sigma by about (clip^2 + 1) sigma / (2 n_kept)."""
    base = 2e-6 * ref_sg + 1e-7 * np.abs(ref_mu)
    per_flip = (clip * clip + 2.0) * ref_sg / (0.5 * n_t)
    tol = base + n_border * per_flip
    assert np.all(np.abs(got_mu - ref_mu) <= tol), float(np.max(np.abs(got_mu - ref_mu) / tol))
    assert np.all(np.abs(got_sg - ref_sg) <= tol), float(np.max(np.abs(got_sg - ref_sg) / tol))
    if n_t <= 100000:
        assert np.mean(n_border == 0) > 0.5, "the tight comparison must cover most rows"


@pytest.mark.parametrize("n_dm,n_t", [(16, 65536), (5, 10007), (300, 4096 + 4), (2, 1 << 21)])
@pytest.mark.parametrize("clip,passes", [(0.0, 0), (2.0, 1), (2.5, 4), (3.0, 8)])
def test_row_stats_against_oracle(spd, oracle_lib, n_dm, n_t, clip, passes):
    """Row f1: per-DM mean / sigma with point-wise outlier rejection (reading A14) against
    the double-precision oracle; see _assert_stats_close for the bound."""
    x = _stats_plane(n_dm, n_t, n_dm * 31 + passes)
    dev = torch.device("cuda:0")
    widths = [1, 2, 4] if n_t % 4 == 0 else [1, 3]
    with spd.Plan(n_dm, n_t, widths) as plan:
        mean, sigma = plan.row_stats(torch.from_numpy(x).to(dev), clip, passes)
        got_mu, got_sg = mean.cpu().numpy().astype(np.float64), sigma.cpu().numpy().astype(np.float64)
    ref_mu, ref_sg, n_pass, n_border = oracle_lib.row_stats_clipped(x, clip, passes, border_eps=1e-6, details=True)
    _assert_stats_close(got_mu, got_sg, ref_mu, ref_sg, n_border, n_t, clip)


@pytest.mark.parametrize("n_dm,n_t,clip,rel_tol", [(24, 65536, 2.0, 1e-4), (7, 30001, 2.5, 1e-3), (64, 8192, 3.0, 0.0),
                                                    (3, 1 << 20, 2.0, 1e-5)])
def test_row_stats_until_convergence(spd, oracle_lib, n_dm, n_t, clip, rel_tol):
    """spd_row_stats_converge ("repeated until convergence"): the device-side stop against the
    oracle's, rule stated in double there.  Pass counts agree (a row whose last change is within 2e-6 of the
    tolerance may stop one pass apart), estimates within the border-line bound, and a row that has stopped
    is not touched by later passes (same result with a larger pass limit)."""
    x = _stats_plane(n_dm, n_t, 4000 + n_dm)
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    widths = [1, 2, 4] if n_t % 4 == 0 else [1, 3]
    with spd.Plan(n_dm, n_t, widths) as plan:
        mean, sigma, n_p = plan.row_stats_converge(plane, clip, 40, rel_tol)
        got_mu, got_sg = mean.cpu().numpy().astype(np.float64), sigma.cpu().numpy().astype(np.float64)
        got_p = n_p.cpu().numpy()
        mean2, sigma2, n_p2 = plan.row_stats_converge(plane, clip, 64, rel_tol)
        assert torch.equal(mean, mean2) and torch.equal(sigma, sigma2) and torch.equal(n_p, n_p2)
        # the caller's fixed count reproduces it where the counts agree
        mean3, sigma3 = plan.row_stats(plane, clip, int(got_p.max()))
        with pytest.raises(spd.SpdError):
            plan.row_stats_converge(plane, clip, 0, rel_tol)       # needs at least one rejection pass
        with pytest.raises(spd.SpdError):
            plan.row_stats_converge(plane, clip, 8, -1.0)
    ref_mu, ref_sg, ref_p, n_border = oracle_lib.row_stats_clipped(x, clip, 40, rel_tol=rel_tol, border_eps=1e-6,
                                                                  details=True)
    assert np.all(got_p >= 1) and np.all(got_p < 40), "the iteration must stop on its own"
    same = got_p == ref_p
    assert np.all(np.abs(got_p - ref_p) <= 1) and same.mean() > 0.8, (got_p, ref_p)
    _assert_stats_close(got_mu[same], got_sg[same], ref_mu[same], ref_sg[same], n_border[same], n_t, clip)
    # one pass apart: both sides are within the tolerance of the fixed point
    assert np.all(np.abs(got_sg - ref_sg)[~same] <= (2.0 * rel_tol + 1e-5) * ref_sg[~same])
    top = got_p == got_p.max()
    assert np.array_equal(mean3.cpu().numpy()[top], mean.cpu().numpy()[top])


def test_row_stats_feed_the_hot_path(spd, oracle_lib):
    """mu, sigma from spd_row_stats (no rejection = reading A6) go straight into spd_run on the device."""
    from workloads import get_workload, make_plane_numpy
    w = get_workload(2).scaled(8, 65536, 8)
    x, _ = make_plane_numpy(w)
    x = (x * np.float32(1.9) - np.float32(7.0)).astype(np.float32)
    widths = spd.spd_width_set_generate(w.width_kind, w.width_param, w.max_width)
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    with spd.Plan(8, 65536, widths) as plan:
        mean, sigma = plan.row_stats(plane)
        snr, idx = plan.run(plane, mean, sigma)
        got_snr, got_idx = snr.cpu().numpy(), idx.cpu().numpy()
        mu64, sg64 = mean.cpu().numpy().astype(np.float64), sigma.cpu().numpy().astype(np.float64)
    ref_mu, ref_sg = oracle_lib.row_stats(x)
    assert np.allclose(mu64, ref_mu, rtol=0, atol=2e-6 * ref_sg.max()) and np.allclose(sg64, ref_sg, rtol=2e-6)
    ref_snr, ref_idx, ref_sec = oracle_lib.spd_prefix(x, mu64, sg64, widths)
    parity.assert_parity(oracle_lib, x, mu64, sg64, widths, got_snr, got_idx, ref_snr, ref_idx, ref_sec,
                         what="row_stats -> spd_run")


def test_row_stats_argument_checks(spd):
    dev = torch.device("cuda:0")
    plane = torch.zeros((2, 1024), device=dev)
    with spd.Plan(2, 1024, [1, 2]) as plan:
        with pytest.raises(spd.SpdError):
            plan.row_stats(plane, 0.0, 2)      # rejection needs a positive threshold
        with pytest.raises(spd.SpdError):
            plan.row_stats(plane, 2.0, -1)


@pytest.mark.parametrize("kind,param,max_width", [("POW2", 0, 8192), ("IGRID", 1, 8192), ("POW2", 0, 32768)])
def test_repeated_runs_are_bit_identical(spd, kind, param, max_width):
    """Race check by repetition (compute-sanitizer is not available on this pool): the kernels have
    no atomics on the data path, so every run of the same plan on the same input must give the same
    bits - a shared-memory or halo race would show up as a difference between runs."""
    rng = np.random.default_rng(41)
    n_dm, n_t = 24, 1 << 19
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(rng.standard_normal((n_dm, n_t), dtype=np.float32)).to(dev)
    mean = torch.from_numpy((0.1 * rng.standard_normal(n_dm)).astype(np.float32)).to(dev)
    sigma = torch.from_numpy((1.0 + rng.random(n_dm)).astype(np.float32)).to(dev)
    widths = spd.spd_width_set_generate(kind, param, max_width)
    with spd.Plan(n_dm, n_t, widths) as plan:
        ref = plan.run_flagged(plane, mean, sigma, 4.0)
        ref = [t.clone() for t in ref]
        streams = [torch.cuda.Stream() for _ in range(2)]
        torch.cuda.synchronize()
        for i in range(8):
            st = streams[i % 2]
            with torch.cuda.stream(st):
                act = torch.empty_like(ref[2])
                got = plan.run_flagged(plane, mean, sigma, 4.0, activity=act, stream=st)
            st.synchronize()
            for a, b in zip(ref, got):
                assert torch.equal(a, b), f"run {i} differs"


@pytest.mark.parametrize("kind,param,n_t", [("POW2", 0, 1 << 20), ("IGRID", 1, 1 << 20), ("IGRID", 2, (1 << 18) + 3)])
def test_run_host_equals_device_run(spd, kind, param, n_t):
    """The end-to-end host entry point (several row blocks) returns exactly what spd_run does
    (both streaming trees and the any-width-set tile kernel)."""
    rng = np.random.default_rng(11)
    n_dm = 6
    x = rng.standard_normal((n_dm, n_t), dtype=np.float32)
    mu = rng.standard_normal(n_dm).astype(np.float32) * 0.01
    sg = (1.0 + 0.1 * rng.random(n_dm)).astype(np.float32)
    widths = spd.spd_width_set_generate(kind, param, 8192 if kind != "IGRID" or param == 1 else 512)
    got_snr, got_idx, _ = run_gpu(spd, x, mu, sg, widths)
    out_snr = np.empty((n_dm, n_t), dtype=np.float32)
    out_idx = np.empty((n_dm, n_t), dtype=np.int32)
    with spd.Plan(n_dm, n_t, widths) as plan:
        plan.run_host(x, mu, sg, out_snr, out_idx)
    assert np.array_equal(out_snr, got_snr) and np.array_equal(out_idx, got_idx)


def test_concurrent_streams_share_a_plan(spd):
    rng = np.random.default_rng(12)
    x = rng.standard_normal((8, 65536), dtype=np.float32)
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    mean, sigma = torch.zeros(8, device=dev), torch.ones(8, device=dev)
    with spd.Plan(8, 65536, [1 << k for k in range(10)]) as plan:
        a = plan.run(plane, mean, sigma)
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        torch.cuda.synchronize()
        with torch.cuda.stream(s1):
            b = plan.run(plane, mean, sigma, stream=s1)
        with torch.cuda.stream(s2):
            c = plan.run(plane, mean, sigma, stream=s2)
        torch.cuda.synchronize()
        assert torch.equal(a[0], b[0]) and torch.equal(a[0], c[0])
        assert torch.equal(a[1], b[1]) and torch.equal(a[1], c[1])


def test_invalid_arguments_fail_loudly(spd):
    with pytest.raises(spd.SpdError):
        spd.spd_plan_create(4, 1024, [], 8)
    with pytest.raises(spd.SpdError):
        spd.spd_plan_create(4, 1024, [0, 2], 8)
    with pytest.raises(spd.SpdError):
        spd.spd_plan_create(4, 1024, [16], 8)      # width above max_width
    with pytest.raises(spd.SpdError):
        spd.spd_plan_create(4, 64, [1, 2], 128)    # max_width above n_t
    with pytest.raises(spd.SpdError):
        spd.spd_width_set_generate(99, 0, 8)
    assert "unknown" in spd.spd_last_error_string()


# --- row f2: per-width boxcar separation (the paper's decimated grids), spd_plan_create_grid ----

def run_gpu_grid(spd, x, mu, sg, widths, seps, max_width=None):
    n_dm, n_t = x.shape
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32)).to(dev)
    mean = torch.from_numpy(np.broadcast_to(np.asarray(mu, dtype=np.float32), (n_dm,)).copy()).to(dev)
    sigma = torch.from_numpy(np.broadcast_to(np.asarray(sg, dtype=np.float32), (n_dm,)).copy()).to(dev)
    with spd.Plan(n_dm, n_t, widths, max_width, separations=seps) as plan:
        assert plan.info["path"] == spd.SPD_PATH_GRID
        snr, idx = plan.run(plane, mean, sigma)
        torch.cuda.synchronize()
        return snr.cpu().numpy(), idx.cpu().numpy(), dict(plan.info)


GRIDS = [("BOXDIT", 8, "BOXDIT", 8), ("BOXDIT", 16, "BOXDIT", 16), ("BOXDIT", 32, "BOXDIT", 32),
         ("POW2", 0, "DIT", 0), ("IGRID", 1, "IGRID", 4), ("IGRID", 2, "IGRID", 8), ("IGRID", 3, "IGRID", 16)]


@pytest.mark.parametrize("wkind,wparam,gkind,gparam", GRIDS)
def test_grid_plans_match_oracle(spd, oracle_lib, wkind, wparam, gkind, gparam):
    """The paper's BoxDIT / DIT / IGRID grids on noise + pulses: several
    tiles, a ragged row length, pulses of widths between grid widths; the generators agree with
    the formula module; a chosen width is always one whose grid contains the sample."""
    from oracle import formulas as F
    M = 600
    widths = spd.spd_width_set_generate(wkind, wparam, M)
    seps = spd.spd_separation_generate(gkind, gparam, widths)
    sepf = {"BOXDIT": F.boxdit_separation(gparam) if gkind == "BOXDIT" else None, "DIT": (lambda L: L),
            "IGRID": F.igrid_separation(gparam) if gkind == "IGRID" else None}[gkind]
    assert [int(s) for s in seps] == [sepf(int(L)) for L in widths]
    rng = np.random.default_rng(4242 + int(widths.size))
    n_t = 11 * 1024 + 317
    x = rng.standard_normal((3, n_t)).astype(np.float32)
    for d, (t0, S) in enumerate([(1000, 23), (5003, 150), (n_t - 300, 290)]):
        x[d, t0:t0 + S] += np.float32(14.0 / np.sqrt(S))
    mu, sg = 0.25, 1.5
    got_snr, got_idx, info = run_gpu_grid(spd, x + np.float32(mu), mu, sg, widths, seps, M)
    mu64 = np.full(3, np.float32(mu), dtype=np.float64)
    sg64 = np.full(3, np.float32(sg), dtype=np.float64)
    xs = (x + np.float32(mu)).astype(np.float32)
    ref_snr, ref_idx, ref_sec = oracle_lib.spd_grid(xs, mu64, sg64, widths, seps)
    parity.assert_parity(oracle_lib, xs, mu64, sg64, widths, got_snr, got_idx, ref_snr, ref_idx, ref_sec,
                         what=f"grid {gkind}:{gparam}")
    n = np.arange(n_t)[None, :]
    on = got_idx >= 0
    assert np.all((n % np.asarray(seps)[np.where(on, got_idx, 0)] == 0) | ~on)


@pytest.mark.parametrize("segs", [0, 3])
@pytest.mark.parametrize("B,M,n_t", [(4, 200, 8192 + 4 * 33), (8, 8192, 40000), (8, 300, 4096), (8, 8, 1000),
                                     (16, 5000, 3 * 4096 + 4), (16, 700, 20004), (32, 8192, 30000), (32, 1000, 9000),
                                     (4, 8188, 25000)])
def test_boxdit_kernel_matches_oracle(spd, oracle_lib, B, M, n_t, segs):
    """Alg. 1's widths (eq. 14) on Alg. 1's grids run on spd_boxdit_kernel: every sample against
    oracle_spd_grid (direct summation on each width's own grid) - 1 to 11 iterations, width sets cut by max_width
    inside the last iteration, rows of one partial chunk up to several chunks with a ragged end, the default work
    split and three segments per row (the warm-up replay), a drifting baseline with an offset, pulses between the
    grid widths and one that runs off the row's end; the same plan with SPD_FLAG_FORCE_GENERIC stays on
    grid_tile_kernel."""
    widths = spd.spd_width_set_generate("BOXDIT", B, M)
    seps = spd.spd_separation_generate("BOXDIT", B, widths)
    rng = np.random.default_rng(B * 1000 + M + n_t)
    x = (rng.standard_normal((3, n_t)) + 0.3 * np.sin(np.arange(n_t) / 3000.0) + 11.0).astype(np.float32)
    for d, (t0, S) in enumerate([(n_t // 3, 23), (n_t // 2 + 1, 150), (n_t - 200, 400)]):
        x[d, t0:t0 + S] += np.float32(14.0 / np.sqrt(S))
    mu, sg = oracle_lib.row_stats(x)
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    mean = torch.from_numpy(mu.astype(np.float32)).to(dev)
    sigma = torch.from_numpy(sg.astype(np.float32)).to(dev)
    with spd.Plan(3, n_t, widths, int(widths[-1]), separations=seps) as plan:
        info = plan.info
        assert info["path"] == spd.SPD_PATH_GRID and info["threads_per_block"] == 256 and info["chunk"] == 4096
        if segs:
            plan.set_option(spd.SPD_OPT_SEGMENTS_PER_ROW, segs)
            chunks = (n_t + 4095) // 4096
            assert plan.info["segments_per_row"] == -(-chunks // -(-chunks // segs))
        snr, idx = plan.run(plane, mean, sigma)
        torch.cuda.synchronize()
    with spd.Plan(3, n_t, widths, int(widths[-1]), separations=seps, flags=spd.SPD_FLAG_FORCE_GENERIC) as plan:
        assert plan.info["threads_per_block"] == 1024
    mu64 = mean.cpu().numpy().astype(np.float64)
    sg64 = sigma.cpu().numpy().astype(np.float64)
    ref_snr, ref_idx, ref_sec = oracle_lib.spd_grid(x, mu64, sg64, widths, seps)
    got_snr, got_idx = snr.cpu().numpy(), idx.cpu().numpy()
    st = parity.assert_parity(oracle_lib, x, mu64, sg64, widths, got_snr, got_idx, ref_snr, ref_idx, ref_sec,
                              what=f"boxdit B={B} M={M} n_t={n_t} segs={segs}")
    assert st.n == 3 * n_t
    n = np.arange(n_t)[None, :]
    assert np.all(n % np.asarray(seps)[got_idx] == 0)   # width 1 always fits: every sample has a width


@pytest.mark.parametrize("B,M", [(8, 2000), (16, 8192)])
def test_boxdit_kernel_with_measured_sigma_per_width(spd, oracle_lib, B, M):
    """spd_run_sigma_w on the BoxDIT kernel, every sample against oracle_spd_grid_sw with the
    table the device measured."""
    n_dm, n_t = 3, 24000
    x = _plane_for_sigma_w(n_dm, n_t, 5 + B)
    widths = spd.spd_width_set_generate("BOXDIT", B, M)
    seps = spd.spd_separation_generate("BOXDIT", B, widths)
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    with spd.Plan(n_dm, n_t, widths, int(widths[-1]), separations=seps) as plan:
        assert plan.info["threads_per_block"] == 256
        mean, _ = plan.row_stats(plane)
        sw = plan.width_sigma(plane, mean)
        snr, idx = plan.run_sigma_w(plane, mean, sw)
        torch.cuda.synchronize()
    mu64 = mean.cpu().numpy().astype(np.float64)
    sw64 = sw.cpu().numpy().astype(np.float64)
    ref = oracle_lib.spd_grid_sw(x, mu64, sw64, widths, seps)
    st = parity.assert_parity_table(oracle_lib, x, mu64, sw64, widths, seps, snr.cpu().numpy(), idx.cpu().numpy(),
                                    *ref, what=f"sigma_w boxdit B={B}")
    assert st.n == n_dm * n_t


@pytest.mark.parametrize("wkind,wparam,gkind,gparam", [("BOXDIT", 8, "BOXDIT", 8), ("IGRID", 1, "IGRID", 4),
                                                       ("POW2", 0, "DIT", 0)])
def test_grid_sliding_pulses_recover_the_paper_bounds(spd, wkind, wparam, gkind, gparam):
    """a pulse slid over every shift; the best response per shift lies
    between eq. (31) and eq. (24), its maximum equals eq. (24) and its minimum / mean equal the
    shift scan of the formula module (itself pinned to the paper's printed losses)."""
    from oracle import formulas as F
    M = 120
    widths = spd.spd_width_set_generate(wkind, wparam, M)
    seps = spd.spd_separation_generate(gkind, gparam, widths)
    sepd = {int(L): int(s) for L, s in zip(widths, seps)}
    period = int(max(seps))
    for S in (3, 9, 20, 33, 47, 100):
        n_t = 4 * M + 2 * period + 2 * S
        x = np.zeros((period, n_t), dtype=np.float32)
        for s in range(period):
            x[s, 2 * period + s: 2 * period + s + S] = np.float32(16.0 / np.sqrt(S))
        got_snr, _, _ = run_gpu_grid(spd, x, 0.0, 1.0, widths, seps, M)
        per_shift = got_snr.max(axis=1).astype(np.float64) / 16.0
        lo, hi, mean = F.brute_force_response(S, [int(L) for L in widths], sepd)
        assert abs(per_shift.min() - lo) < 1e-4 and abs(per_shift.max() - hi) < 1e-4
        assert abs(per_shift.mean() - mean) < 1e-4
        assert per_shift.min() >= F.rsnr_min(S, [int(L) for L in widths], sepd) - 1e-4
        assert abs(per_shift.max() - F.rsnr_max(S, [int(L) for L in widths])) < 1e-4


def test_grid_first_separation_above_one_and_flagged_candidates(spd, oracle_lib):
    """Samples on no width's grid are -inf / -1; the flagged run and the candidate stage work on a grid plan."""
    rng = np.random.default_rng(99)
    n_t = 5000
    x = rng.standard_normal((2, n_t)).astype(np.float32)
    x[1, 2048:2048 + 64] += np.float32(2.0)
    widths, seps = [4, 8, 16, 64], [2, 2, 4, 16]
    got_snr, got_idx, _ = run_gpu_grid(spd, x, 0.0, 1.0, widths, seps, 64)
    ref_snr, ref_idx, ref_sec = oracle_lib.spd_grid(x, 0.0, 1.0, widths, seps)
    parity.assert_parity(oracle_lib, x, 0.0, 1.0, widths, got_snr, got_idx, ref_snr, ref_idx, ref_sec, what="grid sep>1")
    assert np.all(got_idx[:, 1::2] == -1) and np.all(np.isneginf(got_snr[:, 1::2]))
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    mean, sigma = torch.zeros(2, device=dev), torch.ones(2, device=dev)
    with spd.Plan(2, n_t, widths, 64, separations=seps) as plan:
        snr, idx, act = plan.run_flagged(plane, mean, sigma, 8.0)
        lst, n_found = plan.find_candidates_flagged(snr, idx, act, 8.0, 4096)
        torch.cuda.synchronize()
        count, cands = spd.candidates_to_numpy(lst, n_found, 4096)
    assert np.array_equal(snr.cpu().numpy(), got_snr)
    ref_count = oracle_lib.find_candidates(got_snr, got_idx, 8.0)[0]
    assert count == ref_count and count >= 1
    assert np.any((cands["dm"] == 1) & (np.abs(cands["t"].astype(np.int64) - 2048) <= 64))


def test_grid_invalid_arguments(spd):
    with pytest.raises(spd.SpdError):
        spd.Plan(1, 1000, [1, 2, 4], 4, separations=[1, 3, 4])       # not a power of two
    with pytest.raises(spd.SpdError):
        spd.Plan(1, 1000, [1, 2, 4], 4, separations=[2, 1, 4])       # decreasing
    with pytest.raises(spd.SpdError):
        spd.Plan(1, 1000, [1, 4, 2], 4, separations=[1, 1, 1])       # widths not ascending
    with pytest.raises(spd.SpdError):
        spd.Plan(1, 100000, [1, 60000], 60000, separations=[1, 1])   # max_width beyond the tile kernel
    with pytest.raises(spd.SpdError):
        spd.spd_separation_generate("DIT", 0, [1, 2, 3])


# --- the two dyadic-tree kernels: warp-per-stream pieces spanning rows, and the A/B hook -------------

@pytest.mark.parametrize("K", [9, 10, 11, 12, 13, 14])
def test_warp_stream_kernel_pieces_span_rows(spd, oracle_lib, K):
    """Default work split of the warp-per-stream kernel: the plane's steps cut in row-major order into
    pieces that start and stop inside rows (each interior stop replays look-ahead), many short rows with a
    ragged tail, pulses across row ends.  Checked on every sample against the oracle."""
    M = 1 << (K - 1)
    n_dm = 37 if K <= 12 else 11
    n_t = max(512 * 23 + 4 * 5, 3 * M + 512 + 4 * 3)
    rng = np.random.default_rng(500 + K)
    x = rng.standard_normal((n_dm, n_t)).astype(np.float32)
    x[1, n_t // 2: n_t // 2 + M // 2] += np.float32(12.0 / np.sqrt(M // 2))
    x[n_dm - 1, n_t - M // 3:] += np.float32(0.9)
    x[0, :7] += np.float32(4.0)
    got_snr, got_idx, info = run_gpu(spd, x, 0.0, 1.0, [1 << k for k in range(K)])
    assert info["tree_kernel"] == 2 and info["piece_chunks"] > 0 and info["segments_per_row"] == 0
    chunks_per_row = (n_t + info["chunk"] - 1) // info["chunk"]
    assert info["piece_chunks"] % chunks_per_row != 0, "pieces were meant to stop inside rows"
    ref_snr, ref_idx, ref_sec = oracle_lib.spd_prefix(x, 0.0, 1.0, [1 << k for k in range(K)])
    parity.assert_parity(oracle_lib, x, 0.0, 1.0, [1 << k for k in range(K)], got_snr, got_idx, ref_snr, ref_idx,
                         ref_sec, what=f"warp-stream K={K}")


@pytest.mark.parametrize("K", [9, 12, 14])
def test_igrid_block_and_warp_kernels_agree_and_take_a_sigma_table(spd, oracle_lib, K):
    """The IGRID depth-1 widths run on the warp-per-stream kernel for 9 <= K <= 14 levels (tree_kernel 2) and on
    the block-per-stream kernel with SPD_FLAG_BLOCK_TREE (tree_kernel 1): both pass parity on the same plane.
    spd_run_sigma_w on the former (PAPER.md:728 for the paper's IG(1) set) against direct summation with the
    same table on every sample; the table sqrt(L) sigma reproduces spd_run."""
    M = 1 << (K - 1)
    rng = np.random.default_rng(300 + K)
    n_dm, n_t = 3, max(512 * 17 + 12, 2 * M + 600)
    x = rng.standard_normal((n_dm, n_t))
    x[1] = np.convolve(x[1], np.ones(5) / 2.0, mode="same")
    S = max(1, 3 * M // 8)
    x[2, n_t // 3: n_t // 3 + S] += 11.0 / np.sqrt(S)
    x = (x + np.array([0.0, 2.0, -1.0])[:, None]).astype(np.float32)
    widths = spd.spd_width_set_generate("IGRID", 1, M)
    a_snr, a_idx, a_info = run_gpu(spd, x, 0.0, 1.0, widths)
    b_snr, b_idx, b_info = run_gpu(spd, x, 0.0, 1.0, widths, flags=spd.SPD_FLAG_BLOCK_TREE)
    assert a_info["path"] == b_info["path"] == spd.SPD_PATH_IGRID_TREE
    assert a_info["tree_kernel"] == 2 and b_info["tree_kernel"] == 1
    ref = oracle_lib.spd_prefix(x, 0.0, 1.0, widths)
    for snr, idx, name in ((a_snr, a_idx, "warp"), (b_snr, b_idx, "block")):
        parity.assert_parity(oracle_lib, x, 0.0, 1.0, widths, snr, idx, *ref, what=f"igrid {name} K={K}")
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    with spd.Plan(n_dm, n_t, widths, M) as plan:
        mean, sigma = plan.row_stats(plane)
        sw = plan.width_sigma(plane, mean)
        snr, idx = plan.run_sigma_w(plane, mean, sw)
        white = (sigma[:, None] * torch.sqrt(torch.tensor(widths, dtype=torch.float32, device=dev))[None, :]).contiguous()
        snr_w, idx_w = plan.run_sigma_w(plane, mean, white)
        snr_0, idx_0 = plan.run(plane, mean, sigma)
        torch.cuda.synchronize()
    mu64 = mean.cpu().numpy().astype(np.float64)
    sw64 = sw.cpu().numpy().astype(np.float64)
    if K <= 12:   # direct summation of every sample: seconds
        ref_sw = oracle_lib.spd_direct_sw(x, mu64, sw64, widths)
        parity.assert_parity_table(oracle_lib, x, mu64, sw64, widths, None, snr.cpu().numpy(), idx.cpu().numpy(),
                                   *ref_sw, what=f"igrid sigma_w K={K}")
    else:
        for t0, t1 in [(n_t // 3 - 400, n_t // 3 + 400), (n_t - 600, n_t), (0, 400)]:
            r = oracle_lib.spd_direct_sw(x, mu64, sw64, widths, t0, t1)
            tol = parity.snr_tolerance(r[0])
            fit = r[1] >= 0
            assert np.all(np.abs(snr.cpu().numpy()[:, t0:t1] - r[0])[fit] <= tol[fit])
            dec = fit & ((r[0] - r[2]) > tol)
            assert np.array_equal(idx.cpu().numpy()[:, t0:t1][dec], r[1][dec])
    a, b = snr_w.cpu().numpy(), snr_0.cpu().numpy()
    assert np.all(np.abs(a - b) <= 1e-5 * np.maximum(1.0, np.abs(b)))
    assert np.mean(idx_w.cpu().numpy() == idx_0.cpu().numpy()) > 0.999


@pytest.mark.parametrize("K,flags", [(6, 0), (8, 0), (11, "block"), (15, 0), (16, 0)])
def test_igrid_block_kernel_with_measured_sigma_per_width(spd, oracle_lib, K, flags):
    """spd_run_sigma_w on the block-per-stream IGRID kernel (max_width < 256 or > 8192, or SPD_FLAG_BLOCK_TREE):
    PAPER.md:728 applies the interpolated sigma to every width of the IG(1) set.  Every sample against direct
    summation with the same table where that takes seconds, windows otherwise; the table sqrt(L) sigma
    reproduces spd_run."""
    M = 1 << (K - 1)
    rng = np.random.default_rng(900 + K)
    n_dm = 3
    n_t = 4 * ((max(2048 * 5 + 12, 2 * M + 600) + 3) // 4)
    x = rng.standard_normal((n_dm, n_t))
    x[1] = np.convolve(x[1], np.ones(5) / 2.0, mode="same")   # coloured row: sigma_L != sqrt(L) sigma
    S = max(1, 3 * M // 8)
    x[2, n_t // 3: n_t // 3 + S] += 11.0 / np.sqrt(S)
    x = (x + np.array([0.0, 2.0, -1.0])[:, None]).astype(np.float32)
    widths = spd.spd_width_set_generate("IGRID", 1, M)
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    fl = spd.SPD_FLAG_BLOCK_TREE if flags == "block" else 0
    with spd.Plan(n_dm, n_t, widths, M, flags=fl) as plan:
        assert plan.info["path"] == spd.SPD_PATH_IGRID_TREE and plan.info["tree_kernel"] == 1
        mean, sigma = plan.row_stats(plane)
        sw = plan.width_sigma(plane, mean)
        snr, idx = plan.run_sigma_w(plane, mean, sw)
        white = (sigma[:, None] * torch.sqrt(torch.tensor(widths, dtype=torch.float32, device=dev))[None, :]).contiguous()
        snr_w, idx_w = plan.run_sigma_w(plane, mean, white)
        snr_0, idx_0 = plan.run(plane, mean, sigma)
        torch.cuda.synchronize()
    mu64 = mean.cpu().numpy().astype(np.float64)
    sw64 = sw.cpu().numpy().astype(np.float64)
    if K <= 11:   # direct summation of every sample: seconds
        ref_sw = oracle_lib.spd_direct_sw(x, mu64, sw64, widths)
        parity.assert_parity_table(oracle_lib, x, mu64, sw64, widths, None, snr.cpu().numpy(), idx.cpu().numpy(),
                                   *ref_sw, what=f"igrid block sigma_w K={K}")
    else:
        for t0, t1 in [(n_t // 3 - 300, n_t // 3 + 300), (n_t - 500, n_t), (0, 300), (n_t - M - 150, n_t - M + 150)]:
            r = oracle_lib.spd_direct_sw(x, mu64, sw64, widths, t0, t1)
            tol = parity.snr_tolerance(r[0])
            fit = r[1] >= 0
            assert np.all(np.abs(snr.cpu().numpy()[:, t0:t1] - r[0])[fit] <= tol[fit])
            dec = fit & ((r[0] - r[2]) > tol)
            assert np.array_equal(idx.cpu().numpy()[:, t0:t1][dec], r[1][dec])
    a, b = snr_w.cpu().numpy(), snr_0.cpu().numpy()
    assert np.all(np.abs(a - b) <= 1e-5 * np.maximum(1.0, np.abs(b)))
    assert np.mean(idx_w.cpu().numpy() == idx_0.cpu().numpy()) > 0.999


@pytest.mark.parametrize("K,layers", [(9, 4), (12, 4), (14, 4), (13, 16), (11, 1)])
def test_igrid_widths_on_layer_grids_run_on_the_tree_kernel(spd, oracle_lib, K, layers):
    """The paper's IG(1) grids (widths 2^k and 3 * 2^m with the widths of step 2^i on P layers):
    the warp-per-stream kernel forms a level's keys on its grid points only; every sample against
    oracle_spd_grid (direct summation on the grid), pieces stopping inside rows, a ragged tail."""
    M = 1 << (K - 1)
    widths = spd.spd_width_set_generate("IGRID", 1, M)
    seps = spd.spd_separation_generate("IGRID", layers, widths)
    rng = np.random.default_rng(700 + K)
    n_dm, n_t = 3, max(512 * 9 + 20, 2 * M + 1100)
    x = rng.standard_normal((n_dm, n_t)).astype(np.float32)
    S = max(1, 3 * M // 8)
    x[1, (n_t // 3) // 64 * 64: (n_t // 3) // 64 * 64 + S] += np.float32(12.0 / np.sqrt(S))
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    mean, sigma = torch.zeros(n_dm, device=dev), torch.ones(n_dm, device=dev)
    with spd.Plan(n_dm, n_t, widths, M, separations=seps) as plan:
        assert plan.info["path"] == spd.SPD_PATH_GRID and plan.info["tree_kernel"] == 2
        snr, idx, act = plan.run_flagged(plane, mean, sigma, 6.0)
        lst, n_f = plan.find_candidates_flagged(snr, idx, act, 6.0, 1 << 16)
        count, got = spd.candidates_to_numpy(lst, n_f, 1 << 16)
        got_snr, got_idx = snr.cpu().numpy(), idx.cpu().numpy()
    if K <= 12:
        ref = oracle_lib.spd_grid(x, 0.0, 1.0, widths, seps)
        parity.assert_parity(oracle_lib, x, 0.0, 1.0, widths, got_snr, got_idx, *ref, what=f"igrid grid K={K} P={layers}")
    else:
        for t0, t1 in [(n_t // 3 - 600, n_t // 3 + 600), (n_t - 700, n_t), (0, 500), (n_t // 2, n_t // 2 + 512)]:
            ref = oracle_lib.spd_grid(x, 0.0, 1.0, widths, seps, t0, t1)
            parity.assert_parity(oracle_lib, x, 0.0, 1.0, widths, got_snr[:, t0:t1], got_idx[:, t0:t1], *ref, t0=t0,
                                 what=f"igrid grid K={K} P={layers} [{t0}, {t1})")
    ref_count, c_dm, c_t, _, _ = oracle_lib.find_candidates(got_snr, got_idx, 6.0)
    assert count == ref_count and count > 0 and np.array_equal(got["dm"], c_dm) and np.array_equal(got["t"], c_t)


@pytest.mark.parametrize("K", [9, 14])
def test_block_and_warp_kernels_agree(spd, oracle_lib, K):
    """SPD_FLAG_BLOCK_TREE keeps the block-per-stream kernel: both kernels pass parity on the same plane, and
    their SNR planes differ by no more than the tag perturbation (31 ulp)."""
    rng = np.random.default_rng(77 + K)
    n_t = 512 * 40 + 12
    x = rng.standard_normal((4, n_t)).astype(np.float32)
    widths = [1 << k for k in range(K)]
    a_snr, a_idx, a_info = run_gpu(spd, x, 0.0, 1.0, widths)
    b_snr, b_idx, b_info = run_gpu(spd, x, 0.0, 1.0, widths, flags=spd.SPD_FLAG_BLOCK_TREE)
    assert a_info["tree_kernel"] == 2 and b_info["tree_kernel"] == 1
    ref = oracle_lib.spd_prefix(x, 0.0, 1.0, widths)
    for snr, idx, name in ((a_snr, a_idx, "warp"), (b_snr, b_idx, "block")):
        parity.assert_parity(oracle_lib, x, 0.0, 1.0, widths, snr, idx, *ref, what=f"{name} K={K}")
    assert np.all(np.abs(a_snr - b_snr) <= 64 * np.spacing(np.abs(b_snr)) + 1e-30)


# --- row f1, second half: standard deviation per width from decimations ----------

@pytest.mark.parametrize("n_dm,n_t,kind,param,M", [(3, 8192 * 5 + 1234, "IGRID", 1, 256), (2, 300001, "POW2", 0, 32768),
                                                   (5, 4100, "ALL", 0, 48), (1, 8192 * 19, "BOXDIT", 8, 8184),
                                                   (2, 700, "POW2", 0, 512)])
def test_width_sigma_matches_oracle(spd, oracle_lib, n_dm, n_t, kind, param, M):
    """White and red (random-walk-like) rows, ragged lengths, levels above the 8192-sample super-block,
    rows too short for the upper levels (sqrt law from the last measured level)."""
    rng = np.random.default_rng(n_t)
    x = rng.standard_normal((n_dm, n_t))
    x[0] = np.convolve(x[0], np.ones(9) / 3.0, mode="same") + 5.0          # correlated: sigma_L is not sqrt(L)
    x = x.astype(np.float32)
    widths = spd.spd_width_set_generate(kind, param, min(M, n_t))
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    with spd.Plan(n_dm, n_t, widths, int(widths.max()), flags=spd.SPD_FLAG_FORCE_GENERIC) as plan:
        mean, _ = plan.row_stats(plane)
        sw = plan.width_sigma(plane, mean)
        sw2 = plan.width_sigma(plane, mean)
        torch.cuda.synchronize()
    ref = oracle_lib.width_sigma(x, widths)
    got = sw.cpu().numpy().astype(np.float64)
    assert np.allclose(got, ref, rtol=2e-5, atol=0), np.abs(got / ref - 1).max()
    assert torch.equal(sw, sw2)                                            # fixed-order reduction
    if n_t >= 8192 * 4:
        white = ref[1 if n_dm > 1 else 0] if n_dm > 1 else None
        if white is not None:
            L = np.asarray(widths, dtype=np.float64)
            assert np.allclose(white[L <= 64], np.sqrt(L[L <= 64]), rtol=0.05)   # eq. (5) on the white row
        assert ref[0][-1] > 0 and not np.allclose(ref[0], ref[0][0] * np.sqrt(np.asarray(widths) / widths[0]), rtol=0.05)


def _plane_for_sigma_w(n_dm, n_t, seed):
    rng = np.random.default_rng(seed)
    x = rng.standard_normal((n_dm, n_t))
    x[1] = np.convolve(x[1], np.ones(5) / 2.0, mode="same")      # correlated: sigma_L is not sqrt(L) sigma
    x[2, n_t // 2: n_t // 2 + 40] += 1.5
    return (x + 2.0).astype(np.float32)


def test_run_with_measured_sigma_per_width(spd, oracle_lib):
    """spd_run_sigma_w on the any-width-set path against direct summation with the same table (oracle A,
    every sample); a uint8-index plan refuses; misaligned buffers are an error, not a fault."""
    n_dm, n_t = 3, 20000
    x = _plane_for_sigma_w(n_dm, n_t, 31)
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    widths = spd.spd_width_set_generate("IGRID", 1, 128)
    with spd.Plan(n_dm, n_t, widths, 128, flags=spd.SPD_FLAG_FORCE_GENERIC) as plan:
        mean, _ = plan.row_stats(plane)
        sw = plan.width_sigma(plane, mean)
        snr, idx = plan.run_sigma_w(plane, mean, sw)
        torch.cuda.synchronize()
        big = torch.empty(n_dm * n_t + 4, dtype=torch.float32, device=dev)
        with pytest.raises(spd.SpdError) as e:   # an offset view: 4-byte aligned only
            spd.binding._check(spd.load().spd_run_sigma_w(
                plan.handle, plane.data_ptr(), mean.data_ptr(), sw.data_ptr(), big.data_ptr() + 4,
                idx.data_ptr(), 0))
        assert e.value.status == -1
    mu64 = mean.cpu().numpy().astype(np.float64)
    sw64 = sw.cpu().numpy().astype(np.float64)
    ref = oracle_lib.spd_direct_sw(x, mu64, sw64, widths)
    parity.assert_parity_table(oracle_lib, x, mu64, sw64, widths, None, snr.cpu().numpy(), idx.cpu().numpy(), *ref,
                               what="sigma_w generic")
    with spd.Plan(n_dm, n_t, [1, 2, 4, 8], 8, flags=spd.SPD_FLAG_WIDTH_U8) as plan:
        with pytest.raises(spd.SpdError):
            plan.run_sigma_w(plane, mean, sw[:, :4].contiguous())


@pytest.mark.parametrize("wkind,wparam,M,gkind,gparam", [("BOXDIT", 8, 120, "BOXDIT", 8), ("IGRID", 1, 128, "IGRID", 4),
                                                          ("POW2", 0, 256, "DIT", 0), ("POW2", 0, 4096, "IGRID", 4),
                                                          ("IGRID", 2, 512, "EVERY_SAMPLE", 0)])
def test_grid_plans_with_measured_sigma_per_width(spd, oracle_lib, wkind, wparam, M, gkind, gparam):
    """spd_run_sigma_w on SPD_PATH_GRID plans (rows f1 + f2 together), every sample against
    oracle_spd_grid_sw with the table the device measured: BoxDIT, IGRID and DIT grids, and a {2^k} set that
    also has a tree plan (K = 13: spd_run takes the tree kernel, spd_run_sigma_w the grid tile kernel)."""
    n_dm, n_t = 3, 12000 + 4 * 13
    x = _plane_for_sigma_w(n_dm, n_t, 77 + M)
    widths = spd.spd_width_set_generate(wkind, wparam, M)
    seps = spd.spd_separation_generate(gkind, gparam, widths)
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    with spd.Plan(n_dm, n_t, widths, M, separations=seps) as plan:
        assert plan.info["path"] == spd.SPD_PATH_GRID
        mean, _ = plan.row_stats(plane)
        sw = plan.width_sigma(plane, mean)
        snr, idx = plan.run_sigma_w(plane, mean, sw)
        torch.cuda.synchronize()
    mu64 = mean.cpu().numpy().astype(np.float64)
    sw64 = sw.cpu().numpy().astype(np.float64)
    ref = oracle_lib.spd_grid_sw(x, mu64, sw64, widths, seps)
    st = parity.assert_parity_table(oracle_lib, x, mu64, sw64, widths, seps, snr.cpu().numpy(), idx.cpu().numpy(),
                                    *ref, what=f"sigma_w grid {wkind}/{gkind}")
    assert st.n == n_dm * n_t


@pytest.mark.parametrize("K", [3, 8, 15, 16])
def test_block_kernel_with_measured_sigma_per_width(spd, oracle_lib, K):
    """spd_run_sigma_w on the block-per-stream kernel (K <= 8 and configs 4 / 5: K = 16 / 15), PAPER.md:728:
    parity with direct summation using the same table; the table sqrt(L) sigma reproduces spd_run."""
    M = 1 << (K - 1)
    n_dm, n_t = 3, max(2048 * 7 + 8, 2 * M + 2048 + 20)
    x = _plane_for_sigma_w(n_dm, n_t, 500 + K)
    x[0, n_t // 3: n_t // 3 + max(1, M // 2)] += np.float32(9.0 / np.sqrt(max(1, M // 2)))
    widths = [1 << k for k in range(K)]
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    with spd.Plan(n_dm, n_t, widths, M) as plan:
        assert plan.info["tree_kernel"] == 1
        plan.set_option(spd.SPD_OPT_SEGMENTS_PER_ROW, 2)
        mean, sigma = plan.row_stats(plane)
        sw = plan.width_sigma(plane, mean)
        snr, idx = plan.run_sigma_w(plane, mean, sw)
        white = (sigma[:, None] * torch.sqrt(torch.tensor(widths, dtype=torch.float32, device=dev))[None, :]).contiguous()
        snr_w, idx_w = plan.run_sigma_w(plane, mean, white)
        snr_0, idx_0 = plan.run(plane, mean, sigma)
        torch.cuda.synchronize()
    mu64 = mean.cpu().numpy().astype(np.float64)
    sw64 = sw.cpu().numpy().astype(np.float64)
    # oracle A on windows (direct summation of 2^15-sample boxcars over whole rows is minutes): the pulse,
    # a segment boundary, the row tail
    got_snr, got_idx = snr.cpu().numpy(), idx.cpu().numpy()
    for t0, t1 in [(n_t // 3 - 300, n_t // 3 + 300), (n_t // 2 - 200, n_t // 2 + 200), (n_t - 500, n_t), (0, 300)]:
        ref = oracle_lib.spd_direct_sw(x, mu64, sw64, widths, t0, t1)
        tol = parity.snr_tolerance(ref[0])
        fit = ref[1] >= 0
        assert np.all(np.abs(got_snr[:, t0:t1] - ref[0])[fit] <= tol[fit]), (K, t0)
        decisive = fit & ((ref[0] - ref[2]) > tol)
        assert np.array_equal(got_idx[:, t0:t1][decisive], ref[1][decisive]), (K, t0)
    a, b = snr_w.cpu().numpy(), snr_0.cpu().numpy()
    fin = np.isfinite(b)
    assert np.all(np.abs(a - b)[fin] <= 1e-5 * np.maximum(1.0, np.abs(b[fin])))
    assert np.mean(idx_w.cpu().numpy() == idx_0.cpu().numpy()) > 0.999


@pytest.mark.parametrize("K", [9, 12, 14])
def test_warp_stream_kernel_with_measured_sigma_per_width(spd, oracle_lib, K):
    """spd_run_sigma_w on the tuned dyadic path: the warp-per-stream kernel takes 1 / sigma_{d, 2^k} per level
    at run time.  White, correlated and offset rows; parity with direct summation using the same table;
    with the table sqrt(L) sigma it reproduces spd_run to the last few ulp."""
    M = 1 << (K - 1)
    rng = np.random.default_rng(900 + K)
    n_dm, n_t = 4, max(512 * 21 + 8, 3 * M + 516)
    x = rng.standard_normal((n_dm, n_t))
    x[1] = np.convolve(x[1], np.ones(7) / 2.5, mode="same")
    x[2, n_t // 2: n_t // 2 + M // 4] += 10.0 / np.sqrt(M // 4)
    x = (x + np.array([0.0, 3.0, -1.0, 0.5])[:, None]).astype(np.float32)
    widths = [1 << k for k in range(K)]
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    with spd.Plan(n_dm, n_t, widths, M) as plan:
        assert plan.info["tree_kernel"] == 2
        mean, sigma = plan.row_stats(plane)
        sw = plan.width_sigma(plane, mean)
        snr, idx = plan.run_sigma_w(plane, mean, sw)
        white = (sigma[:, None] * torch.sqrt(torch.tensor(widths, dtype=torch.float32, device=dev))[None, :]).contiguous()
        snr_w, idx_w = plan.run_sigma_w(plane, mean, white)
        snr_0, idx_0 = plan.run(plane, mean, sigma)
        torch.cuda.synchronize()
    mu64 = mean.cpu().numpy().astype(np.float64)
    ref = oracle_lib.spd_direct_sw(x, mu64, sw.cpu().numpy().astype(np.float64), widths)
    got_snr, got_idx = snr.cpu().numpy(), idx.cpu().numpy()
    tol = parity.snr_tolerance(ref[0])
    assert np.all(np.abs(got_snr - ref[0]) <= tol), float(np.max(np.abs(got_snr - ref[0]) / tol))
    decisive = (ref[0] - ref[2]) > tol
    assert np.array_equal(got_idx[decisive], ref[1][decisive])
    a, b = snr_w.cpu().numpy(), snr_0.cpu().numpy()
    assert np.all(np.abs(a - b) <= 1e-5 * np.maximum(1.0, np.abs(b)))
    assert np.mean(idx_w.cpu().numpy() == idx_0.cpu().numpy()) > 0.999


@pytest.mark.parametrize("K,gkind,gparam", [(14, "DIT", 0), (12, "IGRID", 4), (9, "IGRID", 16), (13, "EVERY_SAMPLE", 0)])
def test_grid_plans_with_dyadic_widths_run_on_the_tree_kernel(spd, oracle_lib, K, gkind, gparam):
    """Widths {2^k} on a grid (Alg. 3's DIT, or the same widths on P layers) take the
    warp-per-stream tree kernel with each level counted only on its grid; against oracle_spd_grid on every
    sample, pieces stopping inside rows, a ragged tail; off-grid samples never win."""
    M = 1 << (K - 1)
    widths = [1 << k for k in range(K)]
    seps = spd.spd_separation_generate(gkind, gparam, widths)
    rng = np.random.default_rng(600 + K)
    n_dm, n_t = 5, max(512 * 19 + 12, 3 * M + 520)
    x = rng.standard_normal((n_dm, n_t)).astype(np.float32)
    x[1, 3 * 512 + 77: 3 * 512 + 77 + M // 2] += np.float32(11.0 / np.sqrt(M // 2))
    x[4, n_t - M // 3:] += np.float32(0.8)
    got_snr, got_idx, info = run_gpu_grid(spd, x, 0.0, 1.0, widths, seps, M)
    assert info["tree_kernel"] == 2
    ref_snr, ref_idx, ref_sec = oracle_lib.spd_grid(x, 0.0, 1.0, widths, seps)
    parity.assert_parity(oracle_lib, x, 0.0, 1.0, widths, got_snr, got_idx, ref_snr, ref_idx, ref_sec,
                         what=f"grid tree K={K} {gkind}:{gparam}")
    n = np.arange(n_t)[None, :]
    assert np.all(n % np.asarray(seps)[got_idx] == 0)


def test_grid_tree_plan_flagged_candidates(spd, oracle_lib):
    """A grid plan over widths 2^k fuses the threshold test like the tree plans: flagged run = plain run,
    flagged candidates = the rule on the plane."""
    rng = np.random.default_rng(61)
    K, n_dm, n_t = 11, 3, 512 * 40 + 16
    widths = [1 << k for k in range(K)]
    seps = spd.spd_separation_generate("DIT", 0, widths)
    x = rng.standard_normal((n_dm, n_t)).astype(np.float32)
    x[2, 7000:7000 + 256] += np.float32(0.9)
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    mean, sigma = torch.zeros(n_dm, device=dev), torch.ones(n_dm, device=dev)
    with spd.Plan(n_dm, n_t, widths, 1 << (K - 1), separations=seps) as plan:
        assert plan.info["tree_kernel"] == 2 and plan.info["activity_block"] == 2048
        snr0, idx0 = plan.run(plane, mean, sigma)
        snr, idx, act = plan.run_flagged(plane, mean, sigma, 5.0)
        lst, n_found = plan.find_candidates_flagged(snr, idx, act, 5.0, 1 << 14)
        torch.cuda.synchronize()
        count, cands = spd.candidates_to_numpy(lst, n_found, 1 << 14)
    assert torch.equal(snr, snr0) and torch.equal(idx, idx0)
    ref_count, c_dm, c_t, c_snr, c_w = oracle_lib.find_candidates(snr.cpu().numpy(), idx.cpu().numpy(), 5.0)
    assert count == ref_count and count > 0
    assert np.array_equal(cands["dm"], c_dm) and np.array_equal(cands["t"], c_t)
    assert 0 < int(act.sum().item()) < act.numel()


@pytest.mark.parametrize("B,M,thr", [(8, 1016, 5.0), (16, 2000, 6.0), (4, 124, -1.0)])
def test_boxdit_plan_flagged_candidates(spd, oracle_lib, B, M, thr):
    """The BoxDIT streaming kernel fuses the threshold test of row a8 like the tree kernels (one flag per
    4096-sample chunk): the flagged run writes the same planes, the flagged candidate kernel returns exactly
    the rule's candidates on them (also through the row-block path of spd_run_host_candidates), and only
    some chunks are marked."""
    rng = np.random.default_rng(300 + B)
    n_dm, n_t = 5, 4096 * 9 + 4 * 33
    widths = spd.spd_width_set_generate("BOXDIT", B, M)
    seps = spd.spd_separation_generate("BOXDIT", B, widths)
    x = rng.standard_normal((n_dm, n_t)).astype(np.float32)
    x[1, 4096 * 3 - 40: 4096 * 3 - 40 + M // 2] += np.float32(9.0 / np.sqrt(M // 2))   # across a chunk boundary
    x[4, n_t - 300:] += np.float32(0.8)                                                 # at the row's end
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    mean, sigma = torch.zeros(n_dm, device=dev), torch.full((n_dm,), 1.1, device=dev)
    with spd.Plan(n_dm, n_t, widths, M, separations=seps) as plan:
        assert plan.info["path"] == spd.SPD_PATH_GRID and plan.info["threads_per_block"] == 256
        assert plan.info["activity_block"] == 4096
        snr0, idx0 = plan.run(plane, mean, sigma)
        snr, idx, act = plan.run_flagged(plane, mean, sigma, thr)
        lst, n_found = plan.find_candidates_flagged(snr, idx, act, thr, 1 << 18)
        lst_all, n_all = plan.find_candidates(snr, idx, thr, 1 << 18)
        torch.cuda.synchronize()
        count, cands = spd.candidates_to_numpy(lst, n_found, 1 << 18)
        count_all, cands_all = spd.candidates_to_numpy(lst_all, n_all, 1 << 18)
        plan.set_option(spd.SPD_OPT_HOST_ROWS_PER_BLOCK, 2)
        host_found, host_1d, host_arr = plan.run_host_candidates(
            torch.from_numpy(x).pin_memory(), mean.cpu().pin_memory(), sigma.cpu().pin_memory(), thr, 0, 1 << 18)
    assert torch.equal(snr, snr0) and torch.equal(idx, idx0)
    ref_count, c_dm, c_t, _, _ = oracle_lib.find_candidates(snr.cpu().numpy(), idx.cpu().numpy(), thr)
    assert count == ref_count == count_all and count > 0
    order = np.lexsort((cands["t"], cands["dm"]))
    assert np.array_equal(cands["dm"][order], c_dm) and np.array_equal(cands["t"][order], c_t)
    assert host_1d == ref_count
    marked = int(act[: n_dm * ((n_t + 4095) // 4096)].sum().item())
    if thr > 0:
        assert 0 < marked < n_dm * ((n_t + 4095) // 4096)
    else:
        assert marked == n_dm * ((n_t + 4095) // 4096)     # a negative threshold marks every chunk
