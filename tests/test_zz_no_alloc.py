"""trex_xsec_moments_noalloc: the cross-section moments through the entry point that allocates nothing (block partials in
a file-scope device array, result in a device buffer of the caller) against the existing trex_xsec_moments path.
Collected last on purpose (file name): the suite runs with pytest -x."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

RTOL = 1e-12          # the bar of the xsec tests: the two paths differ in the number of blocks, i.e. in summation order


@pytest.fixture(scope="module")
def T():
    import torch
    assert torch.cuda.is_available()
    import paper_2510_05100_b200 as T
    T.lib()
    T.trex_set_stream(None)
    T.trex_set_precision(0)
    return T


def _weights(n, seed):
    rng = np.random.default_rng(seed)
    w_in = rng.lognormal(0.0, 0.5, n)
    w_out = w_in * rng.lognormal(0.0, 0.3, n)
    w_in[::97] = 0.0                      # zero-weight events: skipped in the ratio sum, counted in N
    w_out[::97] = 0.0
    return w_in, w_out


def _close(a, b):
    return np.all(np.abs(a - b) <= RTOL * np.abs(b))


def test_two_calls_in_a_row_match_the_allocating_path(T):
    import torch
    out = torch.full((4,), -1.0, dtype=torch.float64, device="cuda")
    # the second call is smaller than the first: whatever the first left in the shared array must not leak into it
    for n, seed in ((1_000_003, 1), (70_001, 2), (4097, 3), (1, 4)):
        w_in, w_out = _weights(n, seed)
        di, do = torch.from_numpy(w_in).cuda(), torch.from_numpy(w_out).cuda()
        ref = T.trex_xsec_moments(di, do)                       # existing path: host array [4]
        got = T.trex_xsec_moments_noalloc(di, do, out)
        torch.cuda.synchronize()
        g = got.cpu().numpy()
        assert g[0] == n == ref[0]
        assert _close(g[1:3], ref[1:3]), (n, g, ref)
        assert abs(g[3] - ref[3]) <= RTOL * ref[3] + 1e-300, (n, g, ref)
        # and against plain numpy
        assert abs(g[1] - w_out.sum()) <= 1e-11 * w_out.sum()
        # the same call again: identical bits (fixed summation order, nothing carried over)
        again = T.trex_xsec_moments_noalloc(di, do, torch.empty_like(out))
        torch.cuda.synchronize()
        assert np.array_equal(again.cpu().numpy(), g)
    # the combined result of eqs.(6)-(7) agrees as well
    a = T.trex_xsec_finish(ref, 2.0, 100.0, 3.0)
    b = T.trex_xsec_finish(g, 2.0, 100.0, 3.0)
    assert abs(a[0] - b[0]) <= RTOL * abs(a[0]) and abs(a[1] - b[1]) <= RTOL * abs(a[1]) and a[2] == b[2]


def test_empty_and_oversized_inputs(T):
    import torch
    out = torch.full((4,), -1.0, dtype=torch.float64, device="cuda")
    e = torch.empty(0, dtype=torch.float64, device="cuda")
    T.trex_xsec_moments_noalloc(e, e, out)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), np.zeros(4))
    n = T.TREX_XSEC_NOALLOC_MAX_EVENTS + 1
    big = torch.ones(n, dtype=torch.float64, device="cuda")
    out.fill_(-1.0)
    with pytest.raises(T.TrexError, match="exceeds the static scratch"):
        T.trex_xsec_moments_noalloc(big, big, out)
    torch.cuda.synchronize()
    assert bool((out == -1.0).all())                            # rejected before anything was enqueued
    # exactly the maximum is served
    T.trex_xsec_moments_noalloc(big[:-1], big[:-1], out)
    torch.cuda.synchronize()
    g = out.cpu().numpy()
    assert g[0] == n - 1 and g[1] == n - 1 and g[2] == n - 1 and g[3] == 0.0
