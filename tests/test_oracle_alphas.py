"""Pins for the per-event strong coupling: how alpha_s enters the oracle's |M|^2.
With nv strong vertices (nv = number of legs - 2 for every QCD subprocess here) and at most one dimension-6 insertion,
|M|^2 = A + kappa B + kappa^2 D with A ~ alpha_s^nv, B ~ alpha_s^(nv - 1/2), D ~ alpha_s^(nv - 1): the insertion replaces a
g_s vertex by kappa (closed form of B for g g > t t~: SURVEY.md F-3, ~ alpha_s g_s)."""
import numpy as np
import pytest

from oracle import oracle as O
from trex_inputs import default_theta, make_config, TH_ALPHA_S, TH_CTG


@pytest.mark.parametrize("sid,cfg,engine", [(1, 2, 1), (2, 3, 1), (3, 4, 1), (5, 3, 2), (7, 3, 2)])
def test_power_laws_in_alpha_s(sid, cfg, engine):
    w = make_config(cfg, n=8)
    mom = np.ascontiguousarray(w.momenta[:, :, :2])
    nv = mom.shape[0] - 2
    th1, th2 = default_theta(), default_theta()
    th1[TH_ALPHA_S], th2[TH_ALPHA_S] = 0.118, 0.09
    r = 0.09 / 0.118
    a, b = O.abd(sid, mom, th1, engine=engine), O.abd(sid, mom, th2, engine=engine)
    assert np.allclose(b[:, 0] / a[:, 0], r ** nv, rtol=1e-13, atol=0)
    assert np.allclose(b[:, 1] / a[:, 1], r ** (nv - 0.5), rtol=1e-13, atol=0)
    assert np.allclose(b[:, 2] / a[:, 2], r ** (nv - 1), rtol=1e-13, atol=0)


def test_electroweak_process_does_not_see_alpha_s():
    w = make_config(1, n=8)
    th = w.theta_new.copy()
    a = O.me2(0, w.momenta, th)
    th[TH_ALPHA_S] = 0.3
    assert np.array_equal(a, O.me2(0, w.momenta, th))


def test_per_event_alpha_s_is_the_definition():
    w = make_config(3, n=64)
    sp = w.classes[0]
    sel = np.where(w.keys == sp.key)[0][:6]
    mom = np.ascontiguousarray(w.momenta[:, :, sel])
    # a constant vector equal to theta's value changes nothing
    const = np.full(len(sel), w.theta_old[TH_ALPHA_S])
    a = O.reweight_alphas(sp.sid, mom, w.theta_old, w.theta_new, const, w.w_in[sel])
    b = O.reweight(sp.sid, mom, w.theta_old, w.theta_new, w.w_in[sel])
    for x, y in zip(a, b):
        assert np.array_equal(x, y)
    # varying alpha_s: the weight ratio moves (the kappa term scales differently from the alpha_s^nv term) and follows
    # the power laws: w'/w = (A + kappa B r^-1/2 + kappa^2 D r^-1) / A with r = alpha_s / alpha_s(theta) when kappa_old = 0
    al = np.linspace(0.08, 0.16, len(sel))
    got = O.reweight_alphas(sp.sid, mom, w.theta_old, w.theta_new, al, w.w_in[sel])
    abd = O.abd(sp.sid, mom, w.theta_old)
    k = O.kappa(w.theta_new)
    r = al / w.theta_old[TH_ALPHA_S]
    want = w.w_in[sel] * (abd[:, 0] + k * abd[:, 1] / np.sqrt(r) + k * k * abd[:, 2] / r) / abd[:, 0]
    assert np.allclose(got[0], want, rtol=1e-12, atol=0)
    assert not np.allclose(got[0], b[0], rtol=1e-4, atol=0)
    assert np.allclose(got[1], abd[:, 0] * r ** 3, rtol=1e-12, atol=0)
