"""Colour pins: colour matrices vs. their group-theory values, relabelling shortcut vs. direct brute force,
and the colour-ordered engine E1 against the explicit-colour brute force E2."""
import itertools
import os

import numpy as np
import pytest

from oracle import oracle as O
from trex_inputs import default_theta, make_config

from helpers import relclose

GOLD = {}
for line in open(os.path.join(os.path.dirname(__file__), "golden", "colour_matrices.txt")):
    if line.startswith("#") or ":" not in line:
        continue
    k, v = line.split(":")
    GOLD[k.strip()] = [int(x) for x in v.split()]


def test_colour_matrix_values():
    assert np.allclose(O.colour_matrix(2) * 3, np.array(GOLD["n2_times3"]).reshape(2, 2), atol=1e-12)
    assert np.allclose(O.colour_matrix(3)[0] * 9, GOLD["n3_row_times9"], atol=1e-12)
    c4 = O.colour_matrix(4) * 54
    assert np.allclose(c4, np.round(c4), atol=1e-9)
    assert sorted(set(np.round(c4).astype(int).ravel().tolist())) == sorted(GOLD["n4_values_times54"])
    c5 = O.colour_matrix(5) * 324
    assert np.allclose(c5, np.round(c5), atol=1e-8)
    k5 = np.round(c5).astype(int)
    assert np.all(np.diag(k5) == GOLD["n5_diag_times324"][0])
    assert len(set(k5.ravel().tolist())) == GOLD["n5_distinct"][0]
    off = k5[~np.eye(120, dtype=bool)]
    assert np.abs(off).max() == GOLD["n5_offdiag_maxabs_times324"][0]


@pytest.mark.parametrize("n", [2, 3, 4, 5])
def test_colour_matrix_structure(n):
    c = O.colour_matrix(n)
    assert np.allclose(c, c.T, atol=1e-12)
    ev = np.linalg.eigvalsh(c)
    assert ev.min() > 0
    # diagonal: tr over a closed string = C_F^n N_c
    assert relclose(np.diag(c), np.full(len(c), (4.0 / 3.0) ** n * 3.0), rtol=1e-12)
    # total colour sum is permutation invariant: every row has the same multiset of entries
    r0 = np.sort(c[0])
    for r in c[1:: max(1, len(c) // 7)]:
        assert np.allclose(np.sort(r), r0, atol=1e-12)


def test_relabelling_shortcut_against_direct_entries():
    rng = np.random.default_rng(3)
    for n in (3, 4):
        perms = list(itertools.permutations(range(n)))
        c = O.colour_matrix(n)
        for _ in range(6):
            i, j = rng.integers(len(perms), size=2)
            assert abs(O.colour_entry(perms[i], perms[j]) - c[i, j]) < 1e-12


def test_colour_ordered_engine_equals_explicit_colour_brute_force():
    th = default_theta()
    w = make_config(2, n=4)
    a = O.abd(1, w.momenta[:, :, :2], th, engine=1)
    b = O.abd(1, w.momenta[:, :, :2], th, engine=2)
    assert relclose(a, b, rtol=1e-12)
    w = make_config(3, n=4)
    for h in (6, 19, 31):        # single helicities of gg -> tt~g (all 8^3 x 9 colour assignments each)
        a = O.abd(2, w.momenta[:, :, :1], th, engine=1, hel_only=h)
        b = O.abd(2, w.momenta[:, :, :1], th, engine=2, hel_only=h)
        assert relclose(a, b, rtol=1e-11), (h, a, b)


def test_colour_ordered_engine_equals_brute_force_with_four_gluon_vertex():
    """gg -> tt~gg, one helicity: 8^4 x 9 colour assignments; exercises the 4-gluon vertex's three colour
    structures and the ttgg contact term against their colour-ordered forms."""
    th = default_theta()
    w = make_config(4, n=2)
    a = O.abd(3, w.momenta[:, :, :1], th, engine=1, hel_only=37)
    b = O.abd(3, w.momenta[:, :, :1], th, engine=2, hel_only=37)
    assert relclose(a, b, rtol=1e-11), (a, b)


def test_colour_ordered_engine_equals_brute_force_at_five_gluons():
    """gg -> tt~ggg, one helicity: the explicit-colour engine E2 needs 8^5 x 9 colour assignments (five minutes on one
    core), so its (A, B, D) are stored by tests/golden/make_e2_n5.py (a committed script that calls only oracle/). E1 is
    the engine every n = 5 parity test uses; this is its only pin that is neither a symmetry nor E1 itself."""
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "e2_n5_single_helicity.txt")
    ref = np.array([float(x) for x in [l for l in open(path) if not l.startswith("#")][0].split()])
    w = make_config(5, n=8)
    a = O.abd(4, w.momenta[:, :, :1], default_theta(), engine=1, hel_only=77)[0]
    assert relclose(a, ref, rtol=1e-11), (a, ref)
    assert np.all(ref > 0) and ref[1] ** 2 <= 4 * ref[0] * ref[2]


def test_helicity_sum_is_sum_of_single_helicities():
    th = default_theta()
    w = make_config(2, n=2)
    tot = sum(O.abd(1, w.momenta[:, :, :1], th, hel_only=h) for h in range(16))
    assert relclose(tot, O.abd(1, w.momenta[:, :, :1], th), rtol=1e-13)
