"""Pins of the oracle's reweighted cross section / error propagation (eqs.(6)-(7)) against closed
forms that do not come from the oracle itself."""
import math

import numpy as np

from oracle import oracle as O


def test_identity_reweighting_keeps_cross_section_and_error():
    # w' = w = const: sigma' = C N w, mean ratio 1, std 0  =>  Delta sigma' = Delta sigma exactly
    n, c = 1000, 0.25
    w = np.full(n, 2.0)
    s, d, fb = O.xsec(w, w, c, sigma=c * n * 2.0, dsigma=3.5)
    assert s == c * n * 2.0 and d == 3.5 and not fb


def test_arithmetic_series_has_textbook_standard_deviation():
    # w' = 1..N on unit weights: sum = N(N+1)/2, population variance = (N^2 - 1)/12, mean ratio = (N+1)/2
    n = 2001
    w_in = np.ones(n)
    w_out = np.arange(1, n + 1, dtype=np.float64)
    s, d, fb = O.xsec(w_in, w_out, 2.0, sigma=7.0, dsigma=0.5)
    assert s == 2.0 * n * (n + 1) / 2 and not fb
    expect = 0.5 * (n + 1) / 2 + 7.0 * math.sqrt((n * n - 1) / 12.0)
    assert abs(d / expect - 1) < 1e-15


def test_uniform_rescaling_scales_the_statistical_term_only_through_the_ratio():
    # w' = k w: sigma' = k sigma, ratio = k, std(w') = k std(w)
    rng = np.random.default_rng(5)
    w = rng.lognormal(0, 0.5, 500)
    k, c = 1.7, 0.01
    sigma = c * w.sum()
    s, d, fb = O.xsec(w, k * w, c, sigma, dsigma=0.3)
    assert abs(s / (k * sigma) - 1) < 1e-14 and not fb
    assert abs(d / (0.3 * k + sigma * k * w.std()) - 1) < 1e-13


def test_zero_weights_are_skipped_in_the_ratio_but_counted_in_n():
    w_in = np.array([1.0, 0.0, 2.0, 0.0])
    w_out = np.array([2.0, 0.0, 2.0, 0.0])
    s, d, fb = O.xsec(w_in, w_out, 1.0, sigma=3.0, dsigma=1.0)
    # ratio = (2 + 1)/4, mean 1, variance 1
    assert s == 4.0 and abs(d - (0.75 + 3.0 * 1.0)) < 1e-15 and not fb


def test_fallback_rule_takes_the_ratio_greater_than_one():
    w_in = np.ones(4)
    w_out = np.array([1.0, float("inf"), 1.0, 1.0])          # error propagation fails (inf - inf -> nan)
    s, d, fb = O.xsec(w_in, w_out, 1.0, sigma=4.0, dsigma=0.2)
    assert fb and d == 0.2                                     # sigma' itself is unusable: Delta sigma kept
    w_out = -np.ones(4)                                        # negative weights: non-positive error
    s, d, fb = O.xsec(w_in, w_out, 1.0, sigma=4.0, dsigma=0.2)
    assert fb and s == -4.0 and d == 0.2
    # positive sigma' but a non-positive propagated error (negative original error): ratio rule, both directions
    s, d, fb = O.xsec(np.ones(3), np.full(3, 0.5), 1.0, sigma=3.0, dsigma=-0.1)
    assert fb and s == 1.5 and abs(d - (-0.1) * 2.0) < 1e-16
    s, d, fb = O.xsec(np.ones(3), np.full(3, 4.0), 1.0, sigma=3.0, dsigma=-0.1)
    assert fb and abs(d - (-0.1) * 4.0) < 1e-16
