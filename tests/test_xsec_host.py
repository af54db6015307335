"""Host half of the reweighted cross section (trex_xsec_finish: combination of shard moments + eqs.(6)-(7) + fallback
rule) against the oracle; no GPU needed (the moments are formed with numpy here)."""
import numpy as np
import pytest

import paper_2510_05100_b200 as T
from oracle import oracle as O


def _moments(w_in, w_out):
    n = len(w_out)
    if n == 0:
        return [0.0, 0.0, 0.0, 0.0]
    nz = w_in != 0
    return [float(n), float(w_out.sum()), float((w_out[nz] / w_in[nz]).sum()), float(((w_out - w_out.mean()) ** 2).sum())]


@pytest.mark.parametrize("cuts", [(), (1,), (300, 301), (0, 10, 10, 999)])
def test_shard_combination_matches_the_unsharded_definition(cuts):
    rng = np.random.default_rng(11)
    w = rng.lognormal(0, 0.5, 1000)
    w[::13] = 0.0
    wo = w * rng.uniform(0.5, 2.0, 1000)
    edges = [0, *cuts, 1000]
    parts = [_moments(w[a:b], wo[a:b]) for a, b in zip(edges[:-1], edges[1:])]
    got = T.trex_xsec_finish(parts, 0.1, 5.0, 0.2)
    ref = O.xsec(w, wo, 0.1, 5.0, 0.2)
    assert abs(got[0] / ref[0] - 1) < 1e-13 and abs(got[1] / ref[1] - 1) < 1e-12 and got[2] == ref[2] is False


def test_fallback_rule():
    w = np.ones(3)
    for wo, sigma, ds in ((np.full(3, 0.5), 3.0, -0.1), (np.full(3, 4.0), 3.0, -0.1), (-np.ones(3), 3.0, 0.2)):
        got = T.trex_xsec_finish(_moments(w, wo), 1.0, sigma, ds)
        ref = O.xsec(w, wo, 1.0, sigma, ds)
        assert got[2] and ref[2] and got[0] == ref[0] and abs(got[1] - ref[1]) < 1e-15
    assert T.trex_xsec_finish(np.zeros((2, 4)), 1.0, 2.0, 0.3) == (0.0, 0.3, True)     # empty sample
