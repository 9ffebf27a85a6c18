"""spd_row_stats_static (include/spd.h): the per-DM mean / sigma kernels of row f1 with their scratch in a static
device array, for callers that may not allocate.  Checked against the existing path (spd_row_stats with a plan
workspace) on two calls in a row; the file is named so that pytest collects it last (the suite runs with -x)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def spd():
    import paper_1910_08324_b200 as spd
    spd.build()
    spd.load()
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    return spd


def _plane(n_dm, n_t, seed):
    rng = np.random.default_rng(seed)
    x = (rng.standard_normal((n_dm, n_t)) * 2.5 + 11.0).astype(np.float32)
    x[0, n_t // 4: n_t // 4 + max(4, n_t // 50)] += np.float32(40.0)  # a strong wide pulse
    x[n_dm - 1, ::97] -= np.float32(25.0)                             # scattered outliers
    return x


def _existing_path(spd, plane, clip, passes):
    n_dm, n_t = plane.shape
    widths = [1, 2, 4] if n_t % 4 == 0 else [1, 3]
    with spd.Plan(n_dm, n_t, widths) as plan:
        mean, sigma = plan.row_stats(plane, clip, passes)
        torch.cuda.synchronize()
    return mean, sigma


def _assert_close(got, ref, sigma_ref, what):
    # the tolerance of tests/test_gpu_parity.py::_assert_stats_close for rows without border-line samples
    tol = 2e-6 * sigma_ref.double() + 1e-7 * ref.double().abs()
    err = (got.double() - ref.double()).abs()
    assert bool(torch.all(err <= tol)), (what, float((err / tol).max()))


def test_static_scratch_row_stats_equals_the_plan_path_on_two_calls_in_a_row(spd):
    dev = torch.device("cuda:0")
    # (n_dm, n_t, clip, passes): the second call is smaller and ragged, so that it runs over the first call's
    # left-overs in the shared scratch; the third repeats the first (contents of the second in the scratch)
    cases = [(300, 4096 + 4, 2.5, 4), (7, 30001, 2.0, 3), (300, 4096 + 4, 2.5, 4), (16, 1 << 18, 3.0, 0)]
    first = None
    for i, (n_dm, n_t, clip, passes) in enumerate(cases):
        plane = torch.from_numpy(_plane(n_dm, n_t, 9100 + n_dm)).to(dev)
        mean = torch.full((n_dm,), float("nan"), device=dev)
        sigma = torch.full((n_dm,), float("nan"), device=dev)
        out = spd.spd_row_stats_static(plane, mean, sigma, clip, passes)
        torch.cuda.synchronize()
        assert out[0] is mean and out[1] is sigma                      # the caller's buffers, nothing allocated
        ref_mean, ref_sigma = _existing_path(spd, plane, clip, passes)
        assert bool(torch.isfinite(mean).all()) and bool(torch.isfinite(sigma).all())
        _assert_close(mean, ref_mean, ref_sigma, f"mean, call {i}")
        _assert_close(sigma, ref_sigma, ref_sigma, f"sigma, call {i}")
        if i == 0:
            first = (mean.clone(), sigma.clone())
        if i == 2:   # same input as call 0, other contents in the scratch: bit-identical
            assert torch.equal(mean, first[0]) and torch.equal(sigma, first[1])


def test_static_scratch_row_stats_back_to_back_on_one_stream(spd):
    """Two calls enqueued without a synchronisation in between, on one stream (ordered, so no race): each
    result equals the plan path's."""
    dev = torch.device("cuda:0")
    a = torch.from_numpy(_plane(64, 8192, 77)).to(dev)
    b = torch.from_numpy(_plane(5, 10007, 78)).to(dev)
    ma, sa = torch.empty(64, device=dev), torch.empty(64, device=dev)
    mb, sb = torch.empty(5, device=dev), torch.empty(5, device=dev)
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        spd.spd_row_stats_static(a, ma, sa, 2.0, 2, stream=s)
        spd.spd_row_stats_static(b, mb, sb, 2.0, 2, stream=s)
    s.synchronize()
    for plane, m, sg, name in ((a, ma, sa, "a"), (b, mb, sb, "b")):
        rm, rs = _existing_path(spd, plane, 2.0, 2)
        _assert_close(m, rm, rs, f"mean {name}")
        _assert_close(sg, rs, rs, f"sigma {name}")


def test_static_scratch_row_stats_rejects_sizes_beyond_its_maximum(spd):
    dev = torch.device("cuda:0")
    n_dm = spd.SPD_STATIC_MAX_ROWS + 1
    plane = torch.zeros((n_dm, 8), device=dev)
    mean, sigma = torch.empty(n_dm, device=dev), torch.empty(n_dm, device=dev)
    with pytest.raises(spd.SpdError) as err:
        spd.spd_row_stats_static(plane, mean, sigma)
    assert "SPD_STATIC_MAX_ROWS" in str(err.value)
    with pytest.raises(spd.SpdError):
        spd.spd_row_stats_static(plane[:4], mean[:4], sigma[:4], 0.0, 3)   # rejection needs clip_sigma > 0
    # the maximum itself works (rows cut into at most SPD_STATIC_MAX_PARTIALS / n_dm parts)
    n_dm = spd.SPD_STATIC_MAX_ROWS
    plane = torch.from_numpy(_plane(n_dm, 2048, 5)).to(dev)
    mean, sigma = torch.empty(n_dm, device=dev), torch.empty(n_dm, device=dev)
    spd.spd_row_stats_static(plane, mean, sigma, 2.5, 1)
    torch.cuda.synchronize()
    rm, rs = _existing_path(spd, plane, 2.5, 1)
    _assert_close(mean, rm, rs, "mean at the maximum")
    _assert_close(sigma, rs, rs, "sigma at the maximum")
