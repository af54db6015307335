"""Closed-form pins of the oracle: textbook 2->2 results retyped in tests/helpers.py."""
import math
import os

import numpy as np

from oracle import oracle as O
from trex_inputs import default_theta, make_config

from helpers import eemumu_closed, ggtt_sm_closed, ggtt_linear_closed, qqtt_sm_closed, relclose

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_eemumu_matches_gamma_z_closed_form_both_parameter_points():
    w = make_config(1, n=512)
    for th in (w.theta_old, w.theta_new):
        got = O.me2(0, w.momenta, th)
        assert np.allclose(got, eemumu_closed(w.momenta, th), rtol=2e-14, atol=0)
    # ratio is exactly alpha_em independent (|M|^2 ~ alpha^2), R-5
    th_o, th_n = w.theta_old.copy(), w.theta_new.copy()
    r1 = O.me2(0, w.momenta, th_n) / O.me2(0, w.momenta, th_o)
    th_o[1] = th_n[1] = 1 / 128.0
    r2 = O.me2(0, w.momenta, th_n) / O.me2(0, w.momenta, th_o)
    assert relclose(r1, r2, rtol=1e-14)


def test_eemumu_survey_spot_values():
    th_o, th_n = default_theta(), default_theta()
    th_n[2] = 0.2400
    e = 91.1876 / 2
    for line in open(os.path.join(GOLD, "survey_points.txt")):
        if not line.startswith("ee "):
            continue
        c = float(line.split()[1])
        vals = [float(x) for x in line.split("|")[1].split()]
        s = math.sqrt(1 - c * c)
        mom = np.array([[e, 0, 0, e], [e, 0, 0, -e], [e, e * s, 0, e * c], [e, -e * s, 0, -e * c]])[:, :, None]
        assert abs(O.me2(0, mom, th_o)[0] / vals[0] - 1) < 1e-12
        assert abs(O.me2(0, mom, th_n)[0] / vals[1] - 1) < 1e-12


def test_ggtt_sm_and_linear_ctg_closed_forms():
    w = make_config(2, n=256)
    th = w.theta_old
    abd = O.abd(1, w.momenta, th)
    assert relclose(abd[:, 0], ggtt_sm_closed(w.momenta, th), rtol=1e-12)
    kappa_per_c = th[9] / (math.sqrt(2) * th[8] ** 2)
    assert relclose(abd[:, 1] * kappa_per_c, ggtt_linear_closed(w.momenta, th), rtol=1e-12)
    # and through the public me2 entry at c_tG = 0
    assert relclose(O.me2(1, w.momenta, th), ggtt_sm_closed(w.momenta, th), rtol=1e-12)


def test_qqtt_sm_closed_form_pins_light_quark_line_and_its_colour():
    w = make_config(2, n=16)
    got = O.me2(9, w.momenta, w.theta_old)
    assert relclose(got, qqtt_sm_closed(w.momenta, w.theta_old), rtol=1e-12)


def test_survey_appendix_points_cross_check():
    th = default_theta()
    for line in open(os.path.join(GOLD, "survey_points.txt")):
        if line.startswith("#") or line.startswith("ee") or not line.strip():
            continue
        n_s, mom_s, abd_s = line.split("|")
        n = int(n_s)
        mom = np.array([[float(x) for x in leg.split()] for leg in mom_s.split(";")])[:, :, None]
        want = np.array([float(x) for x in abd_s.split()])
        got = O.abd(n - 1, mom, th)[0]
        assert relclose(got, want, rtol=2e-12), (n, got, want)
