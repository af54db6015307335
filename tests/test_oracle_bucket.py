"""Bucketing oracle pins."""
import itertools

import numpy as np

from oracle import oracle as O
from trex_inputs import pack_key, REX_NPOS


def brute(keys):
    """Tiny-input definition, written independently: walk the input, open a bucket at first sight."""
    buckets, order = {}, []
    for i, k in enumerate(keys):
        if k not in buckets:
            buckets[k] = []
            order.append(k)
        buckets[k].append(i)
    npos = int(REX_NPOS)
    if npos in order:
        order.remove(npos)
        order.append(npos)
    perm = [i for k in order for i in buckets[k]]
    offs = np.cumsum([0] + [len(buckets[k]) for k in order])
    return perm, offs, order


def test_all_small_inputs_brute_force():
    alphabet = [7, 3, int(REX_NPOS), 11]
    for n in range(0, 7):
        for keys in itertools.product(alphabet, repeat=n):
            perm, offs, bk = O.bucket(np.array(keys, dtype=np.uint64))
            bp, bo, border = brute(list(keys))
            assert perm.tolist() == bp and offs.tolist() == bo.tolist() and bk.tolist() == border


def test_first_appearance_order_npos_last_and_stability():
    keys = np.array([5, int(REX_NPOS), 9, 5, 2, 9, int(REX_NPOS), 2, 5], dtype=np.uint64)
    perm, offs, bk = O.bucket(keys)
    assert bk.tolist() == [5, 9, 2, int(REX_NPOS)]
    assert perm.tolist() == [0, 3, 8, 2, 5, 4, 7, 1, 6]
    assert offs.tolist() == [0, 3, 5, 7, 9]
    assert perm.dtype == np.int32 and offs.dtype == np.int64


def test_keys_follow_alg1_example():
    """PAPER.md:419-444 (Alg.1): {21,21,6,-6} vs {2,-2,6,-6} differ when all external legs are compared;
    legs are unordered within initial / final state."""
    st = (-1, -1, 1, 1)
    assert pack_key((21, 21, 6, -6), st) != pack_key((2, -2, 6, -6), st)
    assert pack_key((2, 21, 6, -6, 2), (-1, -1, 1, 1, 1)) == pack_key((21, 2, 2, -6, 6), (-1, -1, 1, 1, 1))
    # initial and final state are kept apart: g g -> t t~ g  !=  g (g) with the third gluon incoming
    assert pack_key((21, 21, 6, -6, 21), (-1, -1, 1, 1, 1)) != pack_key((21, 21, 6, -6, 21), (-1, -1, 1, 1, -1))
    assert pack_key((2, -2, 6, -6, 21), (-1, -1, 1, 1, 1)) != pack_key((1, -1, 6, -6, 21), (-1, -1, 1, 1, 1))


def test_gather_is_the_soa_transpose():
    rng = np.random.default_rng(0)
    src = rng.normal(size=(5, 4, 37))
    keys = rng.integers(0, 4, size=37).astype(np.uint64)
    perm, offs, _ = O.bucket(keys)
    dst = O.gather(src, perm)
    for j in range(37):
        assert np.array_equal(dst[:, :, j], src[:, :, perm[j]])
    assert sorted(perm.tolist()) == list(range(37))


# ---------------------------------------------------------------- comparators with a status filter (Alg.1)
def test_alg1_example_both_halves():
    """Alg.1: g g > t t~ and u u~ > t t~ DIFFER under the comparator over all external legs and are
    EQUAL under the comparator over final-state particles only."""
    ev1 = ([21, 21, 6, -6], [-1, -1, 1, 1])
    ev2 = ([2, -2, 6, -6], [-1, -1, 1, 1])
    assert not O.comparator_equal(*ev1, *ev2, status_filter=(-1, 1))
    assert O.comparator_equal(*ev1, *ev2, status_filter=(1,))
    assert O.flavour_key_filtered(*ev1, status_filter=(-1, 1)) != O.flavour_key_filtered(*ev2, status_filter=(-1, 1))
    assert O.flavour_key_filtered(*ev1, status_filter=(1,)) == O.flavour_key_filtered(*ev2, status_filter=(1,))
    # with the external-leg filter and no intermediate partons the key is the default one
    assert O.flavour_key_filtered(*ev1) == O.flavour_key(ev1[0], 2)


def test_filtered_key_equality_is_exactly_the_comparator():
    """Brute force: for random small events (statuses -1, 1, 2; a few flavours) and every filter, two keys are equal iff
    the comparator -- written out as the paper's definition -- calls the events equal."""
    rng = np.random.default_rng(12)
    flav = [21, 2, -2, 6, -6, 23]
    evs = []
    for _ in range(60):
        n = int(rng.integers(3, 7))
        st = [-1, -1] + [int(x) for x in rng.choice([1, 1, 1, 2], size=n - 2)]
        evs.append(([int(x) for x in rng.choice(flav, size=n)], st))
    for filt in ((-1, 1), (1,), (-1,), (), (1, 2), (-1, 1, 2)):
        keys = [int(O.flavour_key_filtered(p, s, status_filter=filt)) for p, s in evs]
        assert all(k != 0xFFFFFFFFFFFFFFFF for k in keys)
        for i in range(len(evs)):
            for j in range(i):
                assert (keys[i] == keys[j]) == O.comparator_equal(*evs[i], *evs[j], status_filter=filt), (filt, evs[i], evs[j])
    # what the key cannot hold is "no class"
    assert int(O.flavour_key_filtered([21] * 9, [-1, -1] + [1] * 7)) == 0xFFFFFFFFFFFFFFFF
    assert int(O.flavour_key_filtered([21, 21, 1000022], [-1, -1, 1])) == 0xFFFFFFFFFFFFFFFF
    assert int(O.flavour_key_filtered([21, 21, 6], [-1, -1, -2], status_filter=())) == 0xFFFFFFFFFFFFFFFF
