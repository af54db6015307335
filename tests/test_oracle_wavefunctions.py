"""Pins for the oracle's external wavefunctions and Dirac algebra (R-1, R-2).
Textbook identities, written out here independently of the oracle source."""
import numpy as np
import pytest

from oracle import oracle as O

G = [O.gamma(mu) for mu in range(4)]
G5 = O.gamma(4)
METRIC = np.diag([1.0, -1.0, -1.0, -1.0])


def slash(p):
    return G[0] * p[0] - G[1] * p[1] - G[2] * p[2] - G[3] * p[3]


def momenta():
    rng = np.random.default_rng(11)
    out = []
    for m in (0.0, 173.0):
        for _ in range(6):
            p3 = rng.normal(size=3) * 300
            out.append((np.array([np.sqrt(m * m + p3 @ p3), *p3]), m))
    out.append((np.array([100.0, 0, 0, 100.0]), 0.0))
    out.append((np.array([100.0, 0, 0, -100.0]), 0.0))
    out.append((np.array([np.hypot(173.0, 50.0), 0, 0, -50.0]), 173.0))
    out.append((np.array([173.0, 0, 0, 0.0]), 173.0))
    return out


def test_clifford_algebra_and_gamma5():
    for mu in range(4):
        for nu in range(4):
            ac = G[mu] @ G[nu] + G[nu] @ G[mu]
            assert np.allclose(ac, 2 * METRIC[mu, nu] * np.eye(4), atol=1e-15)
    assert np.allclose(G5, 1j * G[0] @ G[1] @ G[2] @ G[3], atol=1e-15)
    assert np.allclose(G[0].conj().T, G[0]) and all(np.allclose(G[i].conj().T, -G[i]) for i in (1, 2, 3))


@pytest.mark.parametrize("p,m", momenta())
def test_spin_sums_and_dirac_equation(p, m):
    scale = p[0]
    su = np.zeros((4, 4), complex)
    sv = np.zeros((4, 4), complex)
    for lam in (-1, 1):
        u, v = O.wavefunction("u", p, lam, m == 0), O.wavefunction("v", p, lam, m == 0)
        ub, vb = O.wavefunction("ubar", p, lam, m == 0), O.wavefunction("vbar", p, lam, m == 0)
        assert np.allclose(ub, u.conj() @ G[0], atol=1e-13 * scale)
        assert np.allclose(vb, v.conj() @ G[0], atol=1e-13 * scale)
        su += np.outer(u, ub)
        sv += np.outer(v, vb)
        assert np.allclose((slash(p) - m * np.eye(4)) @ u, 0, atol=1e-12 * scale ** 1.5)
        assert np.allclose((slash(p) + m * np.eye(4)) @ v, 0, atol=1e-12 * scale ** 1.5)
        # normalisation ubar u = 2m, vbar v = -2m
        assert abs(ub @ u - 2 * m) < 1e-12 * scale and abs(vb @ v + 2 * m) < 1e-12 * scale
    assert np.allclose(su, slash(p) + m * np.eye(4), atol=1e-12 * scale)
    assert np.allclose(sv, slash(p) - m * np.eye(4), atol=1e-12 * scale)


@pytest.mark.parametrize("p,m", [pm for pm in momenta() if np.linalg.norm(pm[0][1:]) > 0])
def test_u_is_helicity_eigenstate(p, m):
    # helicity operator (Sigma . p)/|p| with Sigma^i = (i/2) eps_ijk gamma^j gamma^k = gamma5 gamma0 gamma^i
    sig = [G5 @ G[0] @ G[i] for i in (1, 2, 3)]
    n = p[1:] / np.linalg.norm(p[1:])
    h = sum(n[i] * sig[i] for i in range(3))
    for lam in (-1, 1):
        u = O.wavefunction("u", p, lam, m == 0)
        v = O.wavefunction("v", p, lam, m == 0)
        assert np.allclose(h @ u, lam * u, atol=1e-12 * p[0] ** 0.5)
        assert np.allclose(h @ v, -lam * v, atol=1e-12 * p[0] ** 0.5)     # v(p,lam) has spin projection -lam


@pytest.mark.parametrize("p,m", [pm for pm in momenta() if pm[1] == 0.0])
def test_polarisation_vectors(p, m):
    def md(a, b):
        return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]
    for lam in (-1, 1):
        e = O.wavefunction("eps", p, lam)
        assert abs(md(e, p)) < 1e-13 * p[0]
        assert abs(md(e, e.conj()) + 1) < 1e-14
        assert abs(md(e, e)) < 1e-14
        assert e[0] == 0
    ep, em = O.wavefunction("eps", p, 1), O.wavefunction("eps", p, -1)
    assert abs(md(ep, em.conj())) < 1e-14
    # circular polarisation of helicity lam: rotating by angle a about p multiplies eps by exp(-i lam a)
    n = p[1:] / np.linalg.norm(p[1:])
    assert np.allclose(np.cross(n, ep[1:]), -1j * ep[1:], atol=1e-14)
    assert np.allclose(np.cross(n, em[1:]), +1j * em[1:], atol=1e-14)
