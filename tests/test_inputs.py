"""Seeded workload generators: kinematic sanity of the recipe in DESIGN.md section 4."""
import numpy as np
import pytest

from trex_inputs import make_config, subprocess_by_key


@pytest.mark.parametrize("cfg,n", [(1, 512), (2, 2048), (3, 4096), (4, 1024), (5, 512)])
def test_momentum_conservation_and_mass_shell(cfg, n):
    w = make_config(cfg, n=n)
    mom = w.momenta
    assert mom.shape == (w.npar, 4, n) and mom.flags["C_CONTIGUOUS"]
    sqrt_s = mom[0, 0] + mom[1, 0]
    tot = mom[0] + mom[1] - mom[2:].sum(axis=0)
    assert np.abs(tot).max() < 1e-11 * sqrt_s.max()
    m2 = mom[:, 0] ** 2 - (mom[:, 1:] ** 2).sum(axis=1)
    masses = np.zeros(w.npar)
    if cfg > 1:
        masses[2] = masses[3] = 173.0
    assert np.abs(m2 - masses[:, None] ** 2).max() < 1e-9 * (sqrt_s.max() ** 2)
    assert np.all(mom[2:, 0] > 0)


def test_config_shapes_and_statistics():
    w2 = make_config(2, n=20000)
    s = w2.momenta[0, 0] * 2
    assert 400 <= s.min() and s.max() <= 2000 and abs(s.mean() - 1200) < 20
    lw = np.log(w2.w_in)
    assert abs(lw.mean()) < 0.02 and abs(lw.std() - 0.5) < 0.02
    w3 = make_config(3, n=10000)
    keys, counts = np.unique(w3.keys, return_counts=True)
    got = {subprocess_by_key(k).name: c for k, c in zip(keys, counts)}
    assert got == {"g g > t t~ g": 6000, "u u~ > t t~ g": 1000, "d d~ > t t~ g": 500,
                   "u g > t t~ u": 1500, "g u~ > t t~ u~": 1000}
    # shuffled, not sorted
    assert len(np.unique(w3.keys[:50])) > 1
    # determinism
    assert np.array_equal(make_config(3, n=10000).momenta, w3.momenta)
    w4 = make_config(4, n=16)
    assert w4.theta_old[6] == 1.50 and w4.theta_new[6] == 1.35 and w4.theta_new[7] == 0.3
    assert make_config(5, n=4).npar == 7 and make_config(1).n == 4096
