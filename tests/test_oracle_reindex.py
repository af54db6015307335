"""Pins of the oracle's flavour keys / parton re-indexing by brute force and by the
defining properties, none of which come from the oracle itself."""
import itertools

import numpy as np

from oracle import oracle as O
from trex_inputs import SUBPROCESSES, make_config, shuffled_legs, pack_key

STRINGS = [sp.pdg for sp in SUBPROCESSES]


def test_key_is_invariant_under_every_permutation_inside_initial_and_final_state():
    for sp in SUBPROCESSES:
        ref = pack_key(sp.pdg, sp.status)                       # generator-side packing (include/rex_trex.h layout)
        seen = set()
        for pi in itertools.permutations(range(2)):
            for pf in itertools.permutations(range(2, sp.npar)):
                ev = [sp.pdg[i] for i in pi + pf]
                seen.add(int(O.flavour_key(ev, 2)))
        assert seen == {int(ref)}
    # initial and final state are kept apart: u g > t t~ u  is not  g g > t t~ ... nor u u~ -> with swapped sides
    assert O.flavour_key([2, 21, 6, -6, 2], 2) != O.flavour_key([2, 2, 6, -6, 21], 2)
    assert int(O.flavour_key([2, 21, 6, -6, 300], 2)) == 0xFFFFFFFFFFFFFFFF


def test_legmap_restores_the_process_string_for_every_permutation():
    for sp in SUBPROCESSES:
        for pi in itertools.permutations(range(2)):
            for pf in itertools.permutations(range(2, sp.npar)):
                perm = pi + pf
                ev = np.array([[sp.pdg[i]] for i in perm], dtype=np.int32)
                keys, lm = O.keys_and_legmap(ev, 2, STRINGS)
                assert keys[0] == sp.key
                assert tuple(int(ev[lm[pos, 0], 0]) for pos in range(sp.npar)) == sp.pdg      # the defining property
                assert sorted(lm[:, 0]) == list(range(sp.npar))                               # a permutation
                assert all(lm[pos, 0] < 2 for pos in range(2))                                # sides are kept apart


def test_identical_particles_keep_their_event_order_and_unknown_events_map_to_identity():
    ev = np.array([[21], [21], [21], [-6], [6], [21]], dtype=np.int32)          # g g > g t~ t g
    _, lm = O.keys_and_legmap(ev, 2, STRINGS)
    assert list(lm[:, 0]) == [0, 1, 4, 3, 2, 5]                                 # g g > t t~ g g: gluons 2 and 5 in event order
    ev = np.array([[3], [-4], [6], [-6], [21]], dtype=np.int32)             # s c~ > ...: no such class
    keys, lm = O.keys_and_legmap(ev, 2, STRINGS)
    assert list(lm[:, 0]) == [0, 1, 2, 3, 4] and all(keys[0] != sp.key for sp in SUBPROCESSES)


def test_shuffled_sample_maps_back_to_the_canonical_sample():
    w = make_config(3, n=500)
    pdg, mom, n_in = shuffled_legs(w, 3)
    keys, lm = O.keys_and_legmap(pdg, n_in, STRINGS)
    assert np.array_equal(keys, w.keys)
    back = mom[lm, :, np.arange(w.n)].transpose(0, 2, 1)
    # only identical gluons in the initial state may come back swapped; everything else is the canonical sample again
    same = np.all(back == w.momenta, axis=(0, 1))
    gg = w.keys == SUBPROCESSES[2].key
    assert np.all(same[~gg]) and same[gg].mean() > 0.3
    assert np.allclose(np.sort(back[:2], axis=0), np.sort(w.momenta[:2], axis=0))
