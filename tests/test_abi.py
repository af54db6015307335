"""The C-ABI library builds, loads, and exports every symbol include/rex_trex.h declares (no compute calls: no GPU here).
Host-only entry points (keys, registry, colour matrices) are exercised against independent expectations."""
import ctypes
import math
import os
import re

import numpy as np
import pytest

import paper_2510_05100_b200 as T
from paper_2510_05100_b200 import build as B
from trex_inputs import SUBPROCESSES, pack_key

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    B.build()
    return T.lib()


def declared_functions(headers=("rex_trex.h", "rex_trex_diag.h")):
    names = set()
    for h in headers:
        text = open(os.path.join(ROOT, "include", h)).read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        names |= set(re.findall(r"\b((?:rex|trex)_[a-z0-9_]+)\s*\(", text))
    return sorted(names)


def test_every_declared_symbol_is_exported_and_bound(lib):
    names = declared_functions()
    assert len(names) >= 20
    for name in names:
        assert hasattr(lib, name), name
    assert set(names) == set(T.exported_symbols())


def test_no_torch_types_in_signatures():
    for h in ("rex_trex.h", "rex_trex_diag.h"):
        text = open(os.path.join(ROOT, "include", h)).read()
        assert "torch" not in text and "at::" not in text and 'extern "C"' in text


def test_product_header_carries_no_diagnostics():
    """Probes, counters, debug dumps and kernel-selection knobs live in rex_trex_diag.h, not in the boundary."""
    prod = declared_functions(("rex_trex.h",))
    for name in ("trex_debug_flow_amps", "trex_probe_fma", "trex_launch_count", "trex_set_algorithm", "trex_graph_replays"):
        assert name not in prod and name in declared_functions(("rex_trex_diag.h",))
    for name in ("rex_bucket", "rex_gather", "trex_reweight", "trex_run", "trex_subproc_id", "rex_pack_key"):
        assert name in prod


def test_pack_key_matches_input_generator_and_alg1_semantics(lib):
    for sp in SUBPROCESSES:
        assert T.rex_pack_key(sp.pdg, sp.status) == int(pack_key(sp.pdg, sp.status))
        assert T.trex_subproc_id(int(sp.key)) == sp.sid
        assert T.trex_npar(sp.sid) == sp.npar
    # unordered legs, initial and final state kept apart (Alg.1 :419-444)
    a = T.rex_pack_key([21, 2, 6, -6, 2], [-1, -1, 1, 1, 1])
    b = T.rex_pack_key([2, 21, 2, -6, 6], [-1, -1, 1, 1, 1])
    assert a == b
    assert T.rex_pack_key([21, 21, 6, -6], [-1, -1, 1, 1]) != T.rex_pack_key([2, -2, 6, -6], [-1, -1, 1, 1])
    assert T.rex_pack_key([21, 6, 21, -6], [-1, -1, 1, 1]) != T.rex_pack_key([21, 21, 6, -6], [-1, -1, 1, 1])
    # intermediate (status 2) legs are ignored; too many legs / unknown codes give REX_NPOS
    assert T.rex_pack_key([21, 21, 23, 6, -6], [-1, -1, 2, 1, 1]) == T.rex_pack_key([21, 21, 6, -6], [-1, -1, 1, 1])
    assert T.rex_pack_key([1] * 8, [-1, -1, 1, 1, 1, 1, 1, 1]) == T.REX_NPOS
    assert T.rex_pack_key([1000022, 21, 6, -6], [-1, -1, 1, 1]) == T.REX_NPOS
    assert T.trex_subproc_id(T.REX_NPOS) == -2 and T.trex_npar(99) == -2


def test_registry_counts_match_baseline_configs(lib):
    # BASELINE.json configs: ncolor 2 / 6 / 24 / 120 and 16 / 32 / 64 / 128 helicities for g g > t t~ + 0..3 g
    for sid, nc, nh in [(0, 1, 16), (1, 2, 16), (2, 6, 32), (3, 24, 64), (4, 120, 128), (5, 4, 32), (7, 4, 32), (8, 4, 32)]:
        assert T.trex_ncolor(sid) == nc and T.trex_nhel(sid) == nh


def test_colour_matrices_against_group_theory(lib):
    """Independent of the oracle: values quoted in tests/golden/colour_matrices.txt and SU(3) sum rules."""
    c2 = T.trex_colour_matrix(1)
    assert np.allclose(c2 * 3, [[16, -2], [-2, 16]], atol=1e-12)
    c6 = T.trex_colour_matrix(2)
    assert np.allclose(c6[0] * 9, [64, -8, -8, 1, 1, 10], atol=1e-12)
    c24 = T.trex_colour_matrix(3)
    k = np.round(c24 * 54).astype(int)
    assert np.allclose(c24 * 54, k, atol=1e-9) and set(np.unique(k)) == {512, 80, 71, 62, 8, -1, -10, -28, -64}
    c120 = T.trex_colour_matrix(4)
    k = np.round(c120 * 324).astype(int)
    assert np.allclose(c120 * 324, k, atol=1e-8) and k[0, 0] == 4096 and len(np.unique(k)) == 24
    for n, c in ((2, c2), (3, c6), (4, c24), (5, c120)):
        assert np.allclose(c, c.T) and np.all(np.linalg.eigvalsh(c) > 0)
        # diagonal = C_F^n N ; each row sums to the same value (the matrix is a group convolution)
        assert np.allclose(np.diag(c), (4.0 / 3.0) ** n * 3)
        assert np.allclose(c.sum(axis=1), c.sum(axis=1)[0])
        assert c.shape == (math.factorial(n),) * 2
    cq = T.trex_colour_matrix(5)
    assert np.array_equal(cq, [[12, 0, 4, 4], [0, 12, 4, 4], [4, 4, 12, 0], [4, 4, 0, 12]])


def test_colour_matrix_of_the_two_gluon_channels(lib):
    """The 12 x 12 matrix the kernel sums with, against explicit Gell-Mann matrices (flows as in trex_qq2.cuh)."""
    C = T.trex_colour_matrix(21)
    assert C.shape == (12, 12) and np.array_equal(C, C.T)
    lam = np.zeros((8, 3, 3), dtype=complex)
    lam[0][0, 1] = lam[0][1, 0] = 1
    lam[1][0, 1], lam[1][1, 0] = -1j, 1j
    lam[2][0, 0], lam[2][1, 1] = 1, -1
    lam[3][0, 2] = lam[3][2, 0] = 1
    lam[4][0, 2], lam[4][2, 0] = -1j, 1j
    lam[5][1, 2] = lam[5][2, 1] = 1
    lam[6][1, 2], lam[6][2, 1] = -1j, 1j
    lam[7] = np.diag([1, 1, -2]) / math.sqrt(3)
    Tm = lam / 2
    one = np.eye(3)
    flows = []
    for typ in (1, 2):
        for s1, s2 in (("ab", ""), ("ba", ""), ("a", "b"), ("b", "a"), ("", "ab"), ("", "ba")):
            f = np.zeros((8, 8, 3, 3, 3, 3), dtype=complex)          # [a, b, t, tb, r, k]
            for a in range(8):
                for b in range(8):
                    def string(s):
                        m = one
                        for ch in s:
                            m = m @ Tm[a if ch == "a" else b]
                        return m
                    m1, m2 = string(s1), string(s2)
                    if typ == 1:
                        f[a, b] = np.einsum("tk,rq->tqrk", m1, m2)    # (S1)_{t k} (S2)_{r tb}
                    else:
                        f[a, b] = np.einsum("tq,rk->tqrk", m1, m2)    # (S1)_{t tb} (S2)_{r k}
            flows.append(f.reshape(-1))
    F = np.array(flows)
    want = (F.conj() @ F.T).real
    assert np.allclose(C, want, rtol=0, atol=1e-12)
    assert T.trex_ncolor(22) == 12 and T.trex_nhel(23) == 64 and T.trex_npar(26) == 6 and T.trex_npar(35) == 6 and T.trex_npar(36) == -2


def test_compute_calls_fail_loudly_without_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(T.TrexError):
        T.trex_reweight(1, None, np.zeros(16), np.zeros(16), None)


def test_argument_errors_do_not_crash(lib):
    th = (ctypes.c_double * 16)()
    assert lib.trex_reweight(99, None, 4, th, th, None, None, None, None) == -2
    assert lib.trex_reweight(1, None, -1, th, th, None, None, None, None) == -1
    assert lib.trex_reweight(1, None, 4, th, th, None, None, None, None) == -1
    assert b"null" in lib.trex_last_error()
    assert lib.trex_reweight(1, None, 0, th, th, None, None, None, None) == 0      # n == 0 is a no-op
    assert lib.trex_set_precision(7) == -1 and lib.trex_set_precision(0) == 0
    off = (ctypes.c_int64 * 257)()
    assert lib.rex_bucket(None, 0, None, off) == 0 and off[0] == 0
    assert lib.rex_bucket(None, 5, None, off) == -1


def test_filtered_key_host_helper_matches_the_oracle_comparator(lib):
    """rex_pack_key_filtered against the oracle's key AND against the comparator definition (Alg.1)."""
    from oracle import oracle as O
    rng = np.random.default_rng(4)
    flav = [21, 2, -2, 1, 6, -6, 23, 25]
    evs = []
    for _ in range(80):
        n = int(rng.integers(3, 9))
        st = [-1, -1] + [int(x) for x in rng.choice([1, 1, 1, 2], size=n - 2)]
        evs.append(([int(x) for x in rng.choice(flav, size=n)], st))
    for filt in ((-1, 1), (1,), (), (1, 2), (-1,)):
        keys = []
        for p, s in evs:
            k = T.rex_pack_key_filtered(p, s, filt)
            assert k == int(O.flavour_key_filtered(p, s, status_filter=filt))
            keys.append(k)
        for i in range(len(evs)):
            for j in range(i):
                if keys[i] != T.REX_NPOS and keys[j] != T.REX_NPOS:
                    assert (keys[i] == keys[j]) == O.comparator_equal(*evs[i], *evs[j], status_filter=filt)
    # Alg.1: the two events differ under the external-leg comparator and are equal under the final-state one
    a, b = ([21, 21, 6, -6], [-1, -1, 1, 1]), ([2, -2, 6, -6], [-1, -1, 1, 1])
    assert T.rex_pack_key_filtered(*a, (-1, 1)) != T.rex_pack_key_filtered(*b, (-1, 1))
    assert T.rex_pack_key_filtered(*a, (1,)) == T.rex_pack_key_filtered(*b, (1,))
    assert T.rex_pack_key_filtered(*a, (-1, 1)) == T.rex_pack_key(*a)
    assert T.rex_pack_key_filtered(*a, (7,)) == T.REX_NPOS                      # a status the filter cannot hold
