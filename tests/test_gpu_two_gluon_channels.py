"""Parity of the one-light-line + two-gluon kernels (k_qq2; ids 21..26) with the oracle (-m gpu).

The oracle's explicit-colour evaluator needs about half a minute per event and thread for these channels, so the direct
comparisons use a handful of events: (A, B, D) of |M|^2 = A + kappa B + kappa^2 D from ONE oracle evaluation per event are
compared with the CUDA path at three values of c_tG; a further case has different top masses and widths at theta_old and
theta_new (the kernel then walks the top line once per parameter point). Everything else (the family launch inside
trex_run, flavours, reduced precision) is checked against those oracle-checked fp64 results at larger sizes."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from trex_inputs import SUBPROCESSES, default_theta, make_config, TH_CTG, TH_GAMMAT, TH_MT

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


def _events(n, first=0):
    w = make_config(7, n=64)
    return np.ascontiguousarray(w.momenta[:, :, first:first + n])


@pytest.mark.parametrize("sid", [21, 22, 23, 25])
def test_abd_against_oracle(T, sid):
    mom = _events(4, first=sid - 21)
    th0 = default_theta()
    abd = O.abd(sid, mom, th0, engine=2)                   # [n, 3]
    dm, dw = dev(mom), dev(np.ones(mom.shape[2]))
    for c in (1.7, -2.3):
        th1 = th0.copy()
        th1[TH_CTG] = c
        k = O.kappa(th1)
        want_new = abd[:, 0] + k * abd[:, 1] + k * k * abd[:, 2]
        w_out, mo, mn = (x.cpu().numpy() for x in T.trex_reweight(sid, dm, th0, th1, dw))
        assert rel(mo, abd[:, 0]).max() < RTOL64, rel(mo, abd[:, 0])
        assert rel(mn, want_new).max() < RTOL64, rel(mn, want_new)
        assert rel(w_out, want_new / abd[:, 0]).max() < RTOL64
    # the three coefficients separately: B and D from three parameter points
    th_p, th_m = th0.copy(), th0.copy()
    th_p[TH_CTG], th_m[TH_CTG] = 1.0, -1.0
    k = O.kappa(th_p)
    mp = T.trex_reweight(sid, dm, th0, th_p, dw)[2].cpu().numpy()
    mm = T.trex_reweight(sid, dm, th0, th_m, dw)[2].cpu().numpy()
    B = (mp - mm) / (2 * k)
    D = ((mp + mm) / 2 - abd[:, 0]) / (k * k)
    assert rel(B, abd[:, 1]).max() < 1e-9 and rel(D, abd[:, 2]).max() < 1e-7      # D k^2 is 1e-4 of A here: cancellation


def test_top_mass_and_width_differ_between_the_parameter_points(T):
    mom = _events(2, first=9)
    th0, th1 = default_theta(), default_theta()
    th0[TH_GAMMAT], th1[TH_GAMMAT] = 1.5, 1.3
    th1[TH_MT] = 171.0
    th1[TH_CTG] = 0.9
    # on-shell momenta belong to m_t = 173: the new point evaluates the same momenta with another mass parameter in the
    # propagators and spinors, exactly as the oracle does
    w_in = np.array([0.7, 1.9])
    want = O.reweight(22, mom, th0, th1, w_in)
    got = [x.cpu().numpy() for x in T.trex_reweight(22, dev(mom), th0, th1, dev(w_in))]
    for g, r in zip(got, want):
        assert rel(g, r).max() < RTOL64, (g, r)


def test_flavour_of_the_light_line_is_a_label(T):
    mom = _events(64)
    th0, th1 = default_theta(), default_theta()
    th1[TH_CTG] = 1.1
    dm, dw = dev(mom), dev(np.ones(64))
    for u in (21, 22, 23):
        a = T.trex_reweight(u, dm, th0, th1, dw)
        for d in (u + 3, u + 6, u + 9, u + 12):               # d, s, c, b
            b = T.trex_reweight(d, dm, th0, th1, dw)
            for x, y in zip(a, b):
                assert np.array_equal(x.cpu().numpy(), y.cpu().numpy())
    # the oracle agrees that it is a label (single helicity: the full sum takes minutes)
    m1 = np.ascontiguousarray(mom[:, :, :1])
    for u, d in ((21, 24), (22, 31), (23, 35)):
        assert np.array_equal(O.abd(u, m1, th1, engine=2, hel_only=0b010110 if u == 21 else 0b010111 if u == 23 else 0b010011),
                              O.abd(d, m1, th1, engine=2, hel_only=0b010110 if u == 21 else 0b010111 if u == 23 else 0b010011))


@pytest.mark.parametrize("n", [7, 1000, 30011])
def test_cfg7_whole_path_equals_per_class_calls(T, n):
    """trex_run on the seven-class 2 -> t t~ + 2 partons sample: categorisation (bit-exact against the oracle's bucketing),
    one launch of the g g kernel + ONE family launch for the six quark classes, results equal to per-class trex_reweight
    calls on the gathered events (which test_abd_against_oracle pins to the oracle)."""
    import torch
    w = make_config(7, n=n)
    dk, dm, dw = dev(w.keys), dev(w.momenta), dev(w.w_in)
    l0 = T.trex_launch_count()
    w_out, mo, mn, nb = T.trex_run(dk, dm, w.theta_old, w.theta_new, dw)
    torch.cuda.synchronize()
    launches = T.trex_launch_count() - l0
    present = [sp for sp in w.classes if np.any(w.keys == sp.key)]
    assert nb == len(present)
    assert launches <= 12, launches                        # bucketing passes + gather + TWO |M|^2 launches + scatter
    w_out, mo, mn = w_out.cpu().numpy(), mo.cpu().numpy(), mn.cpu().numpy()
    assert np.all(np.isfinite(w_out)) and np.all(mo > 0)
    perm, off, _ = O.bucket(w.keys)
    gperm, goff, _ = T.rex_bucket(dk)
    assert np.array_equal(gperm.cpu().numpy(), perm) and np.array_equal(goff, off)
    for sp in present:
        sel = np.where(w.keys == sp.key)[0]
        r = T.trex_reweight(sp.sid, dev(np.ascontiguousarray(w.momenta[:, :, sel])), w.theta_old, w.theta_new, dev(w.w_in[sel]))
        assert np.array_equal(w_out[sel], r[0].cpu().numpy()), sp.name
        assert np.array_equal(mo[sel], r[1].cpu().numpy()) and np.array_equal(mn[sel], r[2].cpu().numpy()), sp.name


def test_cfg7_sampled_events_against_oracle(T):
    """Two events of the mixed sample straight against the oracle, through the whole path (one q g and one g q~ event)."""
    import torch
    w = make_config(7, n=4096)
    dk, dm, dw = dev(w.keys), dev(w.momenta), dev(w.w_in)
    w_out = T.trex_run(dk, dm, w.theta_old, w.theta_new, dw)[0].cpu().numpy()
    for sid in (25, 23):
        sp = [s for s in SUBPROCESSES if s.sid == sid][0]
        i = np.where(w.keys == sp.key)[0][-1:]
        want = O.reweight(sid, np.ascontiguousarray(w.momenta[:, :, i]), w.theta_old, w.theta_new, w.w_in[i])[0]
        assert rel(w_out[i], want).max() < RTOL64, (sid, w_out[i], want)


def test_reduced_precision_modes(T):
    """mixed (fp64 amplitudes, fp32 colour sum) and fp32 against the oracle-checked fp64 kernel on 4096 events per class:
    median 5e-5, maximum 1e-3 of the weight ratio (the bars of the other channels)."""
    w = make_config(7, n=8192)
    th0, th1 = w.theta_old, w.theta_new
    for sid in (21, 22, 23):
        dm, dw = dev(w.momenta), dev(w.w_in)
        T.trex_set_precision(0)
        ref = T.trex_reweight(sid, dm, th0, th1, dw)[0].cpu().numpy()
        try:
            for mode, med, mx in ((1, 1e-6, 1e-4), (2, 5e-5, 1e-3)):
                T.trex_set_precision(mode)
                got = T.trex_reweight(sid, dm, th0, th1, dw)[0].cpu().numpy()
                r = rel(got, ref)
                assert np.median(r) < med and r.max() < mx, (sid, mode, np.median(r), r.max())
        finally:
            T.trex_set_precision(0)


def test_cfg7_events_in_arbitrary_parton_order(T):
    """trex_run_pdg on the seven-class sample with shuffled legs: keys and leg maps bit-exact against
    the oracle's, weights equal to those of the canonical sample (the order of the identical gluons does not matter), one
    q q~ > t t~ g g event straight against the oracle on its re-indexed momenta, unknown classes zero."""
    import torch
    from trex_inputs import shuffled_legs
    w = make_config(7, n=12007)
    pdg, mom, n_in = shuffled_legs(w, 77, unknown_every=61)
    keys, lm = T.rex_keys(torch.from_numpy(pdg).cuda(), n_in)
    rk, rl = O.keys_and_legmap(pdg, n_in, [sp.pdg for sp in SUBPROCESSES])
    assert np.array_equal(keys.cpu().numpy().view(np.uint64), rk) and np.array_equal(lm.cpu().numpy(), rl)
    wo, mo, mn, nb = T.trex_run_pdg(torch.from_numpy(pdg).cuda(), dev(mom), n_in, w.theta_old, w.theta_new, dev(w.w_in))
    wo = wo.cpu().numpy()
    known = np.isin(rk, np.array([sp.key for sp in w.classes], dtype=np.uint64))
    assert (~known).sum() > 0 and np.all(wo[~known] == 0) and np.all(wo[known] > 0)
    assert nb == len(np.unique(rk))
    w0 = T.trex_run(dev(w.keys), dev(w.momenta), w.theta_old, w.theta_new, dev(w.w_in))[0].cpu().numpy()
    assert rel(wo[known], w0[known]).max() < 1e-12
    sp = [s for s in SUBPROCESSES if s.sid == 21][0]
    i = np.where(rk == sp.key)[0][:1]
    canon = np.ascontiguousarray(mom[rl[:, i], :, i].transpose(0, 2, 1))
    want = O.reweight(21, canon, w.theta_old, w.theta_new, w.w_in[i])[0]
    assert rel(wo[i], want).max() < RTOL64


def test_all_fifteen_two_gluon_classes_through_the_whole_path(T):
    """A 16-class sample (g g > t t~ g g + the fifteen one-light-line + two-gluon classes, all five flavours): ONE family launch
    serves the fifteen; per-class results equal per-class trex_reweight calls, bucketing bit-exact."""
    import torch
    rng = np.random.default_rng(21)
    w = make_config(7, n=9000)
    classes = [sp for sp in SUBPROCESSES if sp.npar == 6]
    assert len(classes) == 16
    keys = np.array([sp.key for sp in classes], dtype=np.uint64)[rng.integers(0, 16, w.n)]
    dk, dm, dw = dev(keys), dev(w.momenta), dev(w.w_in)
    l0 = T.trex_launch_count()
    w_out, mo, mn, nb = T.trex_run(dk, dm, w.theta_old, w.theta_new, dw)
    torch.cuda.synchronize()
    assert nb == 16 and T.trex_launch_count() - l0 <= 12
    perm, off, _ = O.bucket(keys)
    gperm, goff, _ = T.rex_bucket(dk)
    assert np.array_equal(gperm.cpu().numpy(), perm) and np.array_equal(goff, off)
    w_out = w_out.cpu().numpy()
    for sp in classes:
        sel = np.where(keys == sp.key)[0]
        r = T.trex_reweight(sp.sid, dev(np.ascontiguousarray(w.momenta[:, :, sel])), w.theta_old, w.theta_new, dev(w.w_in[sel]))
        assert np.array_equal(w_out[sel], r[0].cpu().numpy()), sp.name


def test_cfg7_many_parameter_points(T):
    """trex_run_multi on the seven-class sample: the direct path equals trex_run row by row (bit for bit), the polynomial
    path (exact quadratic in kappa) agrees with it to 1e-12."""
    w = make_config(7, n=5000)
    dk, dm, dw = dev(w.keys), dev(w.momenta), dev(w.w_in)
    thetas = np.tile(w.theta_new, (6, 1))
    thetas[:, TH_CTG] = np.linspace(-2.0, 3.0, 6)
    T.trex_set_poly_multi(False)
    try:
        direct = T.trex_run_multi(dk, dm, w.theta_old, thetas, dw)
    finally:
        T.trex_set_poly_multi(True)
    for k in (0, 3, 5):
        one = T.trex_run(dk, dm, w.theta_old, thetas[k], dw)
        assert np.array_equal(direct[0][k].cpu().numpy(), one[0].cpu().numpy())
        assert np.array_equal(direct[2][k].cpu().numpy(), one[2].cpu().numpy())
    poly = T.trex_run_multi(dk, dm, w.theta_old, thetas, dw)
    assert rel(poly[0].cpu().numpy(), direct[0].cpu().numpy()).max() < 1e-12


@pytest.mark.parametrize("sid", [5, 7, 8, 21, 22, 23])
def test_every_helicity_of_the_production_kernels_against_the_oracle(T, sid):
    """Per-helicity parity (SURVEY.md I-4 for the quark channels): the colour-summed |M_h|^2 of EVERY helicity configuration
    as the production kernels (k_qq, k_qq2) form it, before their helicity sum, against the oracle's explicit-colour
    evaluation of that one helicity. Compensating errors between helicities cannot hide here; forbidden helicities of the
    massless line must be exact zeros on both sides."""
    npar = T.trex_npar(sid)
    w = make_config(7 if npar == 6 else 3, n=64)
    mom1 = np.ascontiguousarray(w.momenta[:, :, 11:12])
    th0, th1 = default_theta(), default_theta()
    th1[TH_CTG] = 1.4
    got = T.trex_debug_helicity_me2(sid, mom1[:, :, 0], th0, th1)          # [nhel, 2]
    nhel = 1 << npar
    assert got.shape == (nhel, 2)
    k = O.kappa(th1)
    hs = range(nhel) if npar == 5 else list(range(0, nhel, 3)) + [1, 2, 62]      # E2 at 6 legs: 0.4 s per helicity
    nz = 0
    for h in hs:
        abd = O.abd(sid, mom1, th0, engine=2, hel_only=h)[0]
        want = np.array([abd[0], abd[0] + k * abd[1] + k * k * abd[2]])
        if abd[0] == 0.0:
            assert np.all(got[h] == 0.0), (sid, bin(h), got[h])
        else:
            nz += 1
            assert rel(got[h], want).max() < RTOL64, (sid, bin(h), got[h], want)
    assert nz >= len(list(hs)) // 3
    # and the helicity sum is what the kernel returns
    r = T.trex_reweight(sid, dev(mom1), th0, th1, dev(np.ones(1)))
    assert rel(got[:, 0].sum(), r[1].cpu().numpy()[0]) < 1e-13 and rel(got[:, 1].sum(), r[2].cpu().numpy()[0]) < 1e-13
