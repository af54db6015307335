"""Invariance pins of the oracle: Ward identity, Lorentz invariance,
exact quadratic c_tG dependence, unit ratio at theta_new = theta_old, zero guard."""
import numpy as np
import pytest

from oracle import oracle as O
from trex_inputs import default_theta, make_config, TH_CTG, TH_GAMMAT

from helpers import random_lorentz, apply_lorentz, relclose

# (sid, config to take momenta from, events)
TTNG = [(1, 2, 4), (2, 3, 3), (3, 4, 2), (4, 5, 1)]
QCH = [(5, 3, 2), (7, 3, 2), (8, 3, 2)]


@pytest.mark.parametrize("sid,cfg,nev", TTNG)
def test_ward_identity_colour_ordered(sid, cfg, nev):
    """eps_k -> K_k kills every order in kappa (Gamma_t = 0; with a fixed width it is violated, R-9)."""
    w = make_config(cfg, n=8)
    th = default_theta()
    mom = w.momenta[:, :, :nev]
    full = O.abd(sid, mom, th)
    ngl = mom.shape[0] - 2
    for g in range(ngl):                        # every gluon, also at n = 5
        z = O.abd(sid, mom, th, gauge_gluon=g)
        assert np.all(np.abs(z) < 1e-20 * np.abs(full)), (g, z / full)
    # fixed-width scheme: violated (not a bug), so the probe really is sensitive
    th_w = th.copy()
    th_w[TH_GAMMAT] = 1.5
    z = O.abd(sid, mom, th_w, gauge_gluon=0)
    assert np.all(np.abs(z[:, 0]) > 1e-16 * np.abs(full[:, 0]))


@pytest.mark.parametrize("sid,cfg,nev", QCH)
def test_ward_identity_quark_channels_explicit_colour(sid, cfg, nev):
    w = make_config(cfg, n=8)
    th = default_theta()
    mom = w.momenta[:, :, :nev]
    full = O.abd(sid, mom, th, engine=2)
    z = O.abd(sid, mom, th, engine=2, gauge_gluon=0)
    assert np.all(np.abs(z) < 1e-20 * np.abs(full))


@pytest.mark.parametrize("sid,cfg,nev", [(0, 1, 8)] + TTNG[:3] + QCH)
def test_lorentz_invariance(sid, cfg, nev):
    rng = np.random.default_rng(5)
    w = make_config(cfg, n=8)
    mom = w.momenta[:, :, :nev]
    th = w.theta_new.copy()
    # a fixed top width breaks the Ward identity (R-9) and with it the frame independence of the polarisation
    # sum at the 1e-6 level; the invariance is a property of the Gamma_t = 0 amplitude
    th[TH_GAMMAT] = 0.0
    ref = O.me2(sid, mom, th)
    for _ in range(2):
        L = random_lorentz(rng)
        got = O.me2(sid, apply_lorentz(L, mom), th)
        assert relclose(got, ref, rtol=5e-12), got / ref - 1


@pytest.mark.parametrize("sid,cfg,nev", TTNG[:3] + QCH[:1])
def test_me2_is_exactly_quadratic_in_ctg(sid, cfg, nev):
    """At most one dim-6 insertion per amplitude (R-4): a cubic through 4 points has no cubic term, and the
    public me2 entry agrees with A + kappa B + kappa^2 D."""
    w = make_config(cfg, n=8)
    mom = w.momenta[:, :, :nev]
    cs = np.array([0.0, 0.7, 1.9, -2.6, 4.0])
    vals = []
    for c in cs:
        th = default_theta()
        th[TH_CTG] = c
        vals.append(O.me2(sid, mom, th))
    vals = np.array(vals)                       # [5, nev]
    for e in range(nev):
        coef = np.polyfit(cs, vals[:, e], 4)    # exact interpolation through 5 points
        assert abs(coef[0]) < 1e-11 * abs(vals[0, e]) and abs(coef[1]) < 1e-11 * abs(vals[0, e])
    th = default_theta()
    abd = O.abd(sid, mom, th, engine=1 if sid <= 4 else 2)
    th[TH_CTG] = 1.9
    k = O.kappa(th)
    assert relclose(vals[2], abd[:, 0] + k * abd[:, 1] + k * k * abd[:, 2], rtol=1e-13)
    assert np.all(abd[:, 0] > 0) and np.all(abd[:, 2] > 0)
    assert np.all(abd[:, 1] ** 2 <= 4 * abd[:, 0] * abd[:, 2] * (1 + 1e-12))   # |M|^2 >= 0 for every kappa


def test_reweight_definition_unit_ratio_and_zero_guard():
    w = make_config(2, n=64)
    w_out, mo, mn = O.reweight(1, w.momenta, w.theta_old, w.theta_new, w.w_in)
    assert relclose(w_out, w.w_in * O.me2(1, w.momenta, w.theta_new) / O.me2(1, w.momenta, w.theta_old), rtol=1e-15)
    same, _, _ = O.reweight(1, w.momenta, w.theta_old, w.theta_old, w.w_in)
    assert np.allclose(same, w.w_in, rtol=4e-16, atol=0)
    # zero guard: alpha_s = 0 makes me2_old exactly 0 -> weight 0, not NaN/Inf
    th0 = w.theta_old.copy()
    th0[0] = 0.0
    z, mo0, _ = O.reweight(1, w.momenta[:, :, :4], th0, w.theta_new, w.w_in[:4])
    assert np.all(mo0 == 0) and np.all(z == 0)


def test_top_width_enters_continuously_and_double_matches_long_double():
    w = make_config(4, n=4)
    th = w.theta_old.copy()
    a = O.me2(3, w.momenta, th)
    b = O.me2(3, w.momenta, th, long_double=True)
    assert np.allclose(a, b, rtol=1e-12, atol=0)
    th0 = th.copy(); th0[TH_GAMMAT] = 0.0
    th1 = th.copy(); th1[TH_GAMMAT] = 1e-6
    assert np.allclose(O.me2(3, w.momenta, th0), O.me2(3, w.momenta, th1), rtol=1e-6, atol=0)
    assert not np.allclose(a, O.me2(3, w.momenta, th0), rtol=1e-9, atol=0)     # Gamma_t = 1.5 really changes the value


def test_flop_counter_counts_the_same_evaluation():
    """The counting scalar runs the very same templated evaluator: counts are deterministic, grow with the multiplicity,
    and the 2 -> 2 count has the size the plain algorithm implies (16 helicities x 2 orderings x 2 parameter points of
    4 x 4 complex matrix-vector chains: 1e5 - 1e7 operations)."""
    from trex_inputs import make_config
    counts = []
    for cfg, sid in ((2, 1), (3, 2), (4, 3)):
        w = make_config(cfg, n=64)
        i = int(np.where(w.keys == w.classes[0].key)[0][0])
        c1 = O.count_flops(sid, w.momenta[:, :, i], w.theta_old, w.theta_new)
        c2 = O.count_flops(sid, w.momenta[:, :, i], w.theta_old, w.theta_new)
        assert c1 == c2 and c1["flop"] == c1["add"] + c1["mul"] + c1["div"] + c1["sqrt"]
        counts.append(c1["flop"])
    assert 1e5 < counts[0] < 1e7 and counts[0] * 5 < counts[1] and counts[1] * 5 < counts[2]


# ---------------------------------------------------------------- the other massless flavours (ids 10..20)
def test_flavour_of_the_light_line_does_not_change_the_matrix_element():
    """QCD does not see the flavour of a massless quark: ids 10..20 are ids 5, 7, 8 under another label."""
    from trex_inputs import SUBPROCESSES
    w = make_config(3, n=8)
    mom = np.ascontiguousarray(w.momenta[:, :, :2])
    th = w.theta_new.copy()
    ref = {False: None}
    want = {"qq": O.me2(5, mom, th), "qg": O.me2(7, mom, th), "gqb": O.me2(8, mom, th)}
    seen = 0
    for sp in SUBPROCESSES:
        if not 10 <= sp.sid <= 20:
            continue
        kind = "qq" if 21 not in sp.pdg[:2] else ("qg" if sp.pdg[1] == 21 else "gqb")
        assert np.array_equal(O.me2(sp.sid, mom, th), want[kind]), sp.name
        seen += 1
    assert seen == 11


# ---------------------------------------------------------------- parity of the helicity sum (R-21)
@pytest.mark.parametrize("sid,cfg,engine", [(1, 2, 1), (2, 3, 1), (3, 4, 1), (5, 3, 2), (7, 3, 2), (8, 3, 2)])
def test_flipping_every_helicity_is_a_symmetry_only_without_a_width(sid, cfg, engine):
    """QCD and the chromomagnetic operator with a real coefficient conserve parity: flipping every helicity conjugates the
    spinor products, so the three coefficients (A, B, D) of |M_h|^2 equal those of |M_{-h}|^2 -- as long as no propagator
    carries a width (the width keeps its sign under the conjugation). The CUDA kernels use this when Gamma_t = 0; the oracle
    never does, and this test pins both halves of the statement on single helicity configurations."""
    w = make_config(cfg, n=8)
    mom = np.ascontiguousarray(w.momenta[:, :, :2])
    npar = mom.shape[0]
    full = (1 << npar) - 1
    th = default_theta()
    th[TH_CTG] = 0.9
    scale = O.abd(sid, mom, th, engine=engine)              # helicity-summed, for an absolute yardstick
    checked = broken = 0
    for h in list(range(0, full, 3))[:8]:
        a = O.abd(sid, mom, th, engine=engine, hel_only=h)
        b = O.abd(sid, mom, th, engine=engine, hel_only=full ^ h)
        assert np.all(np.abs(a - b) <= 1e-12 * np.abs(scale)), (sid, bin(h), a, b)
        if np.any(a != 0):
            checked += 1
        th_w = th.copy()
        th_w[TH_GAMMAT] = 1.5
        aw = O.abd(sid, mom, th_w, engine=engine, hel_only=h)
        bw = O.abd(sid, mom, th_w, engine=engine, hel_only=full ^ h)
        if np.any(np.abs(aw - bw) > 1e-6 * np.abs(scale)):
            broken += 1
    # the symmetry was tested on non-zero amplitudes, and a width breaks it (not visibly in the 2 -> 2 process, where the
    # top propagators are far off shell in the t / u channels)
    assert checked >= 2 and (broken >= 1 or npar == 4)
