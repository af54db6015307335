"""Parity symmetry of the helicity sum (trex_set_helicity_symmetry; R-21): with Gamma_t = 0 the kernels that honour
the switch evaluate one helicity configuration of every pair {h, -h}; results must match the oracle (which sums every
configuration) with the switch on AND off, and with a width the switch must change nothing, bit for bit."""
import numpy as np
import pytest

from oracle import oracle as O
from trex_inputs import make_config, TH_GAMMAT

pytestmark = pytest.mark.gpu

RTOL64 = 1e-11


@pytest.fixture(scope="module")
def T():
    import torch
    assert torch.cuda.is_available()
    import paper_2510_05100_b200 as T
    T.lib()
    T.trex_set_stream(None)
    T.trex_set_precision(0)
    yield T
    T.trex_set_helicity_symmetry(True)


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rel(a, b):
    return np.abs(a - b) / np.abs(b)


@pytest.mark.parametrize("cfg,sid,n,nor", [(5, 4, 300, 3), (2, 1, 5000, 64), (3, 2, 4000, 24), (3, 5, 4000, 6), (3, 7, 4000, 6), (3, 8, 4000, 6), (7, 3, 900, 8), (7, 22, 2000, 2), (7, 21, 2000, 1)])
def test_on_and_off_against_the_oracle(T, cfg, sid, n, nor):
    w = make_config(cfg, n=n)
    assert w.theta_old[TH_GAMMAT] == 0.0 and w.theta_new[TH_GAMMAT] == 0.0
    dm, dw = dev(w.momenta), dev(w.w_in)
    res = {}
    for on in (True, False):
        T.trex_set_helicity_symmetry(on)
        res[on] = [x.cpu().numpy() for x in T.trex_reweight(sid, dm, w.theta_old, w.theta_new, dw)]
    T.trex_set_helicity_symmetry(True)
    for a, b in zip(res[True], res[False]):
        assert rel(a, b).max() < 1e-12                       # the symmetry itself, on every event
    assert not np.array_equal(res[True][1], res[False][1])  # ... and the switch really selects another evaluation
    idx = np.arange(nor)
    if (cfg, sid) in ((2, 1), (3, 2), (3, 7), (7, 3)):       # reduced-precision modes take the same path: both settings agree
        for mode, tol in ((1, 1e-5), (2, 2e-3)):
            T.trex_set_precision(mode)
            try:
                r = {}
                for on in (True, False):
                    T.trex_set_helicity_symmetry(on)
                    r[on] = T.trex_reweight(sid, dm, w.theta_old, w.theta_new, dw)[0].cpu().numpy()
            finally:
                T.trex_set_precision(0)
                T.trex_set_helicity_symmetry(True)
            assert rel(r[True], r[False]).max() < tol and rel(r[True], res[False][0]).max() < tol
    want = O.reweight(sid, np.ascontiguousarray(w.momenta[:, :, idx]), w.theta_old, w.theta_new, w.w_in[idx])
    for on in (True, False):
        for g, r in zip(res[on], want):
            assert rel(g[idx], r).max() < RTOL64, (on, rel(g[idx], r).max())


@pytest.mark.parametrize("cfg,sid,n", [(5, 4, 200), (2, 1, 3000), (3, 2, 3000), (3, 7, 3000), (7, 3, 600), (7, 23, 1000)])
def test_with_a_width_every_configuration_is_evaluated(T, cfg, sid, n):
    w = make_config(cfg, n=n)
    th_old, th_new = w.theta_old.copy(), w.theta_new.copy()
    th_old[TH_GAMMAT] = 1.5                                  # one point with a width is enough to break the symmetry
    dm, dw = dev(w.momenta), dev(w.w_in)
    res = {}
    for on in (True, False):
        T.trex_set_helicity_symmetry(on)
        res[on] = [x.cpu().numpy() for x in T.trex_reweight(sid, dm, th_old, th_new, dw)]
    T.trex_set_helicity_symmetry(True)
    for a, b in zip(res[True], res[False]):
        assert np.array_equal(a, b)
    want = O.reweight(sid, np.ascontiguousarray(w.momenta[:, :, :1]), th_old, th_new, w.w_in[:1])
    for g, r in zip(res[True], want):
        assert rel(g[:1], r).max() < RTOL64


def test_whole_path_and_graph_replay_follow_the_switch(T):
    import torch
    w = make_config(7, n=6000)
    dk = torch.from_numpy(w.keys.view(np.int64)).cuda()
    dm, dw = dev(w.momenta), dev(w.w_in)
    wo = torch.empty_like(dw)
    outs = {}
    for on in (True, False, True):
        T.trex_set_helicity_symmetry(on)
        for _ in range(3):                                    # the third call replays the captured graph
            T.trex_run(dk, dm, w.theta_old, w.theta_new, dw, w_out=wo, want_me2=False)
        torch.cuda.synchronize()
        r = wo.cpu().numpy().copy()
        if on in outs:
            assert np.array_equal(outs[on], r)
        outs[on] = r
    assert not np.array_equal(outs[True], outs[False]) and rel(outs[True], outs[False]).max() < 1e-12
