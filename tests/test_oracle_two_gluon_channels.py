"""Pins of the oracle for the one-light-line channels with TWO gluons (ids 21, 22, 23: u u~ > t t~ g g, u g > t t~ u g,
g u~ > t t~ u~ g). The explicit-colour evaluator E2 is generic in the number of gluon
sources; what is new for these ids is the list of gluon legs, the identical-particle factor and the average. Pinned by
  - the Ward identity on BOTH gluons, helicity by helicity,
  - Lorentz invariance of the top-spin sum at fixed massless helicities,
  - Bose symmetry of the two final gluons (id 21),
  - the collinear limits: |M(.. g g)|^2 -> (1/2!) 8 pi alpha_s / s_45 P_gg(z) |M(.. g)|^2 (azimuthal average) and
    |M(.. q g)|^2 -> 8 pi alpha_s / s_45 P_qq(z) |M(.. q)|^2 against the one-gluon channels (ids 5, 7, 8), which fixes the
    overall normalisation: coupling power, colour factors C_A and C_F, the 1/2! of id 21 and the averages.
The full helicity and colour sum of one event takes E2 about half a minute, so every pin works on single helicity
configurations (`hel_only`; bit `leg` of the index = helicity of that leg)."""
import numpy as np
import pytest

from oracle import oracle as O
from trex_inputs import default_theta, make_config
from trex_inputs.configs import _two_to_n

from helpers import random_lorentz, apply_lorentz

MT = 173.0
SIDS = (21, 22, 23)
# helicity indices with a non-vanishing amplitude: the massless line needs opposite chiralities at its two ends
# (legs 0, 1 for id 21: h0 != h1; legs 0, 4 for id 22 and 1, 4 for id 23: equal helicities, one end is crossed)
HELS = {21: (0b000001, 0b010110, 0b101010, 0b111101), 22: (0b000000, 0b010011, 0b100110, 0b111111),
        23: (0b000000, 0b010111, 0b101000, 0b111111)}


def _events(nev):
    w = make_config(4, n=8)                        # 2 -> t t~ + two massless partons at sqrt(s) = 1500
    return np.ascontiguousarray(w.momenta[:, :, :nev])


def _sum_over(sid, mom, th, fixed, free):
    tot = 0.0
    for c in range(1 << len(free)):
        h = fixed
        for i, b in enumerate(free):
            h |= ((c >> i) & 1) << b
        tot = tot + O.abd(sid, mom, th, engine=2, hel_only=h)
    return tot


@pytest.mark.parametrize("sid", SIDS)
def test_ward_identity_on_both_gluons(sid):
    mom = _events(2)
    th = default_theta()
    seen = 0
    for h in HELS[sid]:
        full = O.abd(sid, mom, th, engine=2, hel_only=h)
        assert np.all(full[:, 0] > 0) and np.all(full[:, 2] > 0), (sid, bin(h))
        for g in range(2):
            z = O.abd(sid, mom, th, engine=2, gauge_gluon=g, hel_only=h)
            assert np.all(np.abs(z) < 1e-20 * np.abs(full)), (sid, bin(h), g, z / full)
            seen += 1
    assert seen == 8


@pytest.mark.parametrize("sid", SIDS)
def test_helicity_selection_of_the_massless_line(sid):
    mom = _events(1)
    th = default_theta()
    ends = {21: (0, 1), 22: (0, 4), 23: (1, 4)}[sid]
    for h in range(0, 64, 5):
        a = O.abd(sid, mom, th, engine=2, hel_only=h)[0]
        h0, h1 = (h >> ends[0]) & 1, (h >> ends[1]) & 1
        allowed = (h0 != h1) if sid == 21 else (h0 == h1)
        assert (a[0] > 0) == allowed and (allowed or np.all(a == 0)), (sid, bin(h), a)


@pytest.mark.parametrize("sid", SIDS)
def test_lorentz_invariance_of_the_top_spin_sum(sid):
    rng = np.random.default_rng(17)
    mom = _events(2)
    th = default_theta()
    th[7] = 1.3                                    # (A, B, D) are each invariant
    L = random_lorentz(rng)
    for h in HELS[sid][1:2]:
        fixed = h & ~0b001100
        ref = _sum_over(sid, mom, th, fixed, [2, 3])
        got = _sum_over(sid, apply_lorentz(L, mom), th, fixed, [2, 3])
        assert np.allclose(got, ref, rtol=5e-11, atol=0), (sid, bin(h), got / ref - 1)


def test_bose_symmetry_of_the_final_gluons():
    mom = _events(2)
    th = default_theta()
    th[7] = 0.7
    sw = mom.copy()
    sw[4], sw[5] = mom[5].copy(), mom[4].copy()
    for h in (0b010110, 0b100001, 0b011010):
        hs = (h & 0b001111) | (((h >> 4) & 1) << 5) | (((h >> 5) & 1) << 4)
        a = O.abd(21, mom, th, engine=2, hel_only=h)
        b = O.abd(21, sw, th, engine=2, hel_only=hs)
        assert np.allclose(a, b, rtol=1e-11, atol=0), (bin(h), a / b - 1)
    # and the other two ids are NOT symmetric under the exchange of their gluons (one is incoming): the check can fail
    sw2 = mom.copy()
    sw2[1], sw2[5] = mom[5].copy(), mom[1].copy()
    assert not np.allclose(O.abd(22, mom, th, engine=2, hel_only=0), O.abd(22, sw2, th, engine=2, hel_only=0), rtol=1e-3, atol=0)


def _split(P, m, cth, phi):
    """two massless momenta summing to P (P^2 = m^2): decay angles (cth, phi) in the rest frame w.r.t. the flight direction"""
    E, p = P[0], P[1:]
    pm = np.linalg.norm(p)
    n = p / pm
    a = np.array([1.0, 0.0, 0.0]) if abs(n[0]) < 0.9 else np.array([0.0, 1.0, 0.0])
    e1 = np.cross(n, a)
    e1 /= np.linalg.norm(e1)
    e2 = np.cross(n, e1)
    sth = np.sqrt(1.0 - cth * cth)
    d = sth * np.cos(phi) * e1 + sth * np.sin(phi) * e2 + cth * n
    k = 0.5 * m * np.concatenate([[1.0], d])
    g, bg = E / m, pm / m
    kl = k[1:] @ n
    k1 = np.concatenate([[g * k[0] + bg * kl], k[1:] + ((g - 1.0) * kl + bg * k[0]) * n])
    return k1, P - k1


@pytest.mark.parametrize("sid,parent_sid", [(21, 5), (22, 7), (23, 8)])
def test_collinear_limit_reproduces_the_one_gluon_channel(sid, parent_sid):
    """Final-state collinear factorisation at fixed helicities of the other legs, summed over the helicities of the two
    daughters (legs 4, 5) and of the parent (leg 4 of the one-gluon channel). The 5-leg event and the 6-leg event come from
    the same phase-space draws with a pair mass of 0 and m45 = 0.01 GeV; corrections are O(m45 / Q) (measured: 3e-7 for
    g -> g g after the azimuthal average, 1e-5..2e-4 for q -> q g)."""
    th = default_theta()
    m45, cth = 1e-2, 0.3
    z = 0.5 * (1.0 + cth)                          # energy fraction of the first daughter
    m6 = _two_to_n(np.random.default_rng(11), 1, 1200.0, [MT, MT, m45], False)
    m5 = _two_to_n(np.random.default_rng(11), 1, 1200.0, [MT, MT, 0.0], False)
    P = m6[4, :, 0]
    if sid == 21:
        split_fn = 2.0 * 3.0 * (z / (1.0 - z) + (1.0 - z) / z + z * (1.0 - z))      # P_gg, C_A = 3
        phis, sym, tol = [0.4 + k * np.pi / 2 for k in range(4)], 0.5, 2e-6      # cos(2 phi) spin correlation averages out
    else:
        split_fn = 4.0 / 3.0 * (1.0 + z * z) / (1.0 - z)                            # P_qq, C_F = 4/3, z = quark fraction
        phis, sym, tol = [0.4], 1.0, 1e-3
    for fixed in HELS[sid][:3]:
        fixed &= 0b001111
        acc = 0.0
        for phi in phis:
            k1, k2 = _split(P, m45, cth, phi)
            mom = np.zeros((6, 4, 1))
            mom[:4] = m6[:4]
            mom[4, :, 0], mom[5, :, 0] = k1, k2
            acc = acc + _sum_over(sid, mom, th, fixed, [4, 5])[:, 0] / len(phis)
        ref = _sum_over(parent_sid, m5, th, fixed, [4])[:, 0]
        pred = sym * 8.0 * np.pi * th[0] / m45 ** 2 * split_fn * ref
        assert ref[0] > 0 and abs(acc[0] / pred[0] - 1.0) < tol, (sid, bin(fixed), acc / pred - 1)


def test_flavour_labels_of_the_two_gluon_channels():
    """ids 24..35 are ids 21, 22, 23 under another flavour label (d, s, c, b)."""
    mom = _events(1)
    th = default_theta()
    th[7] = 0.5
    for base, h in ((21, 0b010110), (22, 0b010011), (23, 0b010111)):
        ref = O.abd(base, mom, th, engine=2, hel_only=h)
        for k in (1, 2, 3, 4):
            assert np.array_equal(O.abd(base + 3 * k, mom, th, engine=2, hel_only=h), ref)
    assert O.lib().oracle_npar(35) == 6 and O.lib().oracle_npar(36) == -1
