"""trex_run_alphas (per-event strong coupling) against the oracle's definition (-m gpu)."""
import numpy as np
import pytest

from oracle import oracle as O
from trex_inputs import make_config, REX_NPOS, TH_ALPHA_S, TH_GAMMAT, TH_MT

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
    return T


def dev(a):
    import torch
    a = np.ascontiguousarray(a)
    if a.dtype == np.uint64:
        a = a.view(np.int64)
    return torch.from_numpy(a).cuda()


def rel(a, b):
    return np.abs(a - b) / np.abs(b)


def _alphas(n, seed):
    return np.random.default_rng(seed).uniform(0.085, 0.16, n)


@pytest.mark.parametrize("cfg,n,per_class", [(2, 3000, 48), (3, 6000, 6), (4, 700, 12)])
def test_against_the_oracle_definition(T, cfg, n, per_class):
    """cfg 4 has different top widths at the two parameter points (two top-line passes), cfg 3 five classes."""
    w = make_config(cfg, n=n)
    th_old, th_new = w.theta_old.copy(), w.theta_new.copy()
    if cfg == 2:
        th_old[7] = -0.4                                   # kappa_old != 0 as well
    al = _alphas(n, 40 + cfg)
    out = T.trex_run_alphas(dev(w.keys), dev(w.momenta), th_old, th_new, dev(al), dev(w.w_in))
    got = [x.cpu().numpy() for x in out[:3]]
    assert out[3] == len(w.classes)
    for sp in w.classes:
        sel = np.where(w.keys == sp.key)[0]
        sel = sel[:per_class if sp.sid <= 4 else max(2, per_class // 3)]
        want = O.reweight_alphas(sp.sid, np.ascontiguousarray(w.momenta[:, :, sel]), th_old, th_new, al[sel], w.w_in[sel])
        for g, r in zip(got, want):
            assert rel(g[sel], r).max() < RTOL64, (sp.name, rel(g[sel], r).max())


@pytest.mark.parametrize("cfg,n", [(1, 4096), (2, 5000), (3, 20000), (5, 300), (7, 3000)])
def test_constant_alpha_s_equals_the_plain_path(T, cfg, n):
    w = make_config(cfg, n=n)
    keys = w.keys.copy()
    if cfg == 3:
        keys[3::97] = np.uint64(REX_NPOS)
    dk, dm, dw = dev(keys), dev(w.momenta), dev(w.w_in)
    ref = T.trex_run(dk, dm, w.theta_old, w.theta_new, dw)
    al = np.full(n, w.theta_old[TH_ALPHA_S])
    out = T.trex_run_alphas(dk, dm, w.theta_old, w.theta_new, dev(al), dw)
    assert out[3] == ref[3]
    known = keys != np.uint64(REX_NPOS)
    for a, b in zip(out[:3], ref[:3]):
        a, b = a.cpu().numpy(), b.cpu().numpy()
        if cfg == 1:
            assert np.array_equal(a, b)                    # no alpha_s in e- e+ > mu- mu+: the same kernel result
        else:
            assert rel(a[known], b[known]).max() < 2e-13
        assert np.all(a[~known] == 0) and np.all(b[~known] == 0)


def test_mass_shift_and_zero_coupling(T):
    """m_t differs between the points (the quadratic is fitted per parameter point); an event with alpha_s = 0 gets weight 0."""
    w = make_config(3, n=4000)
    th_old, th_new = w.theta_old.copy(), w.theta_new.copy()
    th_old[TH_GAMMAT], th_new[TH_GAMMAT] = 1.4, 1.6
    th_new[TH_MT] = 172.0
    al = _alphas(w.n, 3)
    al[5] = 0.0
    out = [x.cpu().numpy() for x in T.trex_run_alphas(dev(w.keys), dev(w.momenta), th_old, th_new, dev(al), dev(w.w_in))[:3]]
    assert out[0][5] == 0 and out[1][5] == 0 and out[2][5] == 0
    sp = w.classes[0]
    sel = np.where(w.keys == sp.key)[0][10:26]
    want = O.reweight_alphas(sp.sid, np.ascontiguousarray(w.momenta[:, :, sel]), th_old, th_new, al[sel], w.w_in[sel])
    for g, r in zip(out, want):
        assert rel(g[sel], r).max() < RTOL64
    with pytest.raises(T.TrexError):
        T.trex_run_alphas(dev(w.keys), dev(w.momenta), th_old, th_new, dev(al[:100]), dev(w.w_in))
