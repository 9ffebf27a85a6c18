"""Output separated by iteration (eq. 12) on the GPU: spd_run_iterations against
oracle_spd_grid_iter (direct summation) on every point of every iteration, for the paper's grids."""
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


CASES = [
    # width set, max width, grid, n_dm, n_t
    ("BOXDIT", 4, 124, "BOXDIT", 4, 3, 4096 * 2 + 4 * 37),
    ("BOXDIT", 8, 2040, "BOXDIT", 8, 2, 4096 * 3 + 4 * 5),
    ("BOXDIT", 16, 1008, "BOXDIT", 16, 2, 10007),          # n_t not a multiple of 4: the tile kernel only
    ("BOXDIT", 32, 2000, "BOXDIT", 32, 2, 4096 * 2 + 8),   # the last iteration cut by max_width
    ("POW2", 0, 1024, "DIT", 0, 3, 9000),                  # one width per iteration
    ("IGRID", 1, 512, "IGRID", 4, 2, 8192 + 12),           # the widths of a step on four layers
    ("IGRID", 1, 256, "EVERY_SAMPLE", 0, 2, 3000),         # a single iteration = the every-sample plane
    ("BOXDIT", 4, 28, "BOXDIT", 4, 1, 28),                 # a row no longer than the widest boxcar, one DM trial
    ("BOXDIT", 8, 56, "BOXDIT", 8, 3, 4096),               # exactly one chunk of the streaming kernel
    ("POW2", 0, 8, "DIT", 0, 2, 9),                        # nine samples
]


@pytest.mark.parametrize("wkind,wparam,M,gkind,gparam,n_dm,n_t", CASES)
def test_run_iterations_matches_the_oracle(spd, oracle_lib, wkind, wparam, M, gkind, gparam, n_dm, n_t):
    rng = np.random.default_rng(4242 + M + n_t)
    x = (rng.standard_normal((n_dm, n_t)) * 1.3 + 0.25).astype(np.float32)
    S = max(1, M // 3)
    t_p = (n_t // 3) // 64 * 64
    x[n_dm - 1, t_p: t_p + S] += np.float32(12.0 * 1.3 / np.sqrt(S))
    x[0, n_t - M // 2:] += np.float32(0.7)                 # a step near the row's end: windows that do not fit
    mu = np.array([0.25, 0.2, 0.3][:n_dm])
    sg = np.array([1.3, 1.25, 1.35][:n_dm])
    widths = spd.spd_width_set_generate(wkind, wparam, M)
    seps = spd.spd_separation_generate(gkind, gparam, widths)
    dev = torch.device("cuda:0")
    plane = torch.from_numpy(x).to(dev)
    mean = torch.from_numpy(mu.astype(np.float32)).to(dev)
    sigma = torch.from_numpy(sg.astype(np.float32)).to(dev)
    mu64, sg64 = mean.cpu().numpy().astype(np.float64), sigma.cpu().numpy().astype(np.float64)
    with spd.Plan(n_dm, n_t, widths, M, separations=seps) as plan:
        its = plan.iterations()
        planes, buf_snr, buf_idx = plan.run_iterations(plane, mean, sigma)
        merged_snr, merged_idx = plan.run(plane, mean, sigma)
        torch.cuda.synchronize()
    want = oracle_lib.grid_iterations(seps)
    assert [(it["first_width"], it["first_width"] + it["n_widths"]) for it in its] == want
    assert buf_snr.numel() == n_dm * sum(it["n_points"] for it in its)
    merged = np.full((n_dm, n_t), -np.inf, dtype=np.float32)
    for it, (kb, ke), (y, w) in zip(its, want, planes):
        s = it["separation"]
        assert s == seps[kb] and it["n_points"] == (n_t + s - 1) // s
        ref = oracle_lib.spd_grid_iter(x, mu64, sg64, widths, seps, kb, ke)
        got_snr, got_idx = y.cpu().numpy(), w.cpu().numpy()
        st = parity.assert_parity(oracle_lib, x, mu64, sg64, widths, got_snr, got_idx, *ref, stride=s,
                                  what=f"iteration [{kb}, {ke}) of {wkind}:{wparam} on {gkind}:{gparam}")
        assert st.n == n_dm * it["n_points"]
        fit = got_idx >= 0
        assert np.all((got_idx[fit] >= kb) & (got_idx[fit] < ke))     # an iteration reports its own widths only
        merged[:, ::s] = np.maximum(merged[:, ::s], got_snr)
    # reading A16: spd_run's merged plane is the maximum over the iterations (to the tag perturbation of the
    # kernels that tag their keys)
    ms = merged_snr.cpu().numpy()
    both = np.isfinite(ms)
    assert np.array_equal(both, np.isfinite(merged))
    assert np.all(np.abs(ms[both] - merged[both]) <= 1e-4 * np.maximum(1.0, np.abs(merged[both])))


def test_run_iterations_needs_a_grid_plan(spd):
    dev = torch.device("cuda:0")
    with spd.Plan(2, 4096, [1, 2, 4, 8]) as plan:
        with pytest.raises(spd.SpdError):
            plan.iterations()
        with pytest.raises(spd.SpdError):
            plan.run_iterations(torch.zeros((2, 4096), device=dev), torch.zeros(2, device=dev),
                                torch.ones(2, device=dev))
