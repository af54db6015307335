"""Flat massive RAMBO phase space (Kleiss, Stirling, Ellis), numpy, vectorised over events.

Input generator only: stands in for the paper's MG5aMC LHE samples,
which are not available. Recipe: DESIGN.md section 4 / SURVEY.md 8(d).
"""
import numpy as np


def massive_rambo(r, sqrt_s, masses):
    """Final-state momenta for n events.

    r       : float64 [n, nf, 4] uniform(0,1) numbers, r[:, i, :] = (r1, r2, r3, r4) of particle i
    sqrt_s  : float64 [n] centre-of-mass energies
    masses  : sequence of nf masses
    returns : float64 [n, nf, 4] momenta (E, px, py, pz) in the centre-of-mass frame
    """
    r = np.asarray(r, dtype=np.float64)
    n, nf, _ = r.shape
    sqrt_s = np.broadcast_to(np.asarray(sqrt_s, dtype=np.float64), (n,))
    m = np.asarray(masses, dtype=np.float64)[None, :]

    c = 2.0 * r[:, :, 0] - 1.0
    phi = 2.0 * np.pi * r[:, :, 1]
    q0 = -np.log(r[:, :, 2] * r[:, :, 3])
    st = np.sqrt(np.maximum(0.0, 1.0 - c * c))
    q = np.stack([q0, q0 * st * np.cos(phi), q0 * st * np.sin(phi), q0 * c], axis=-1)

    Q = q.sum(axis=1)                                    # [n,4]
    M = np.sqrt(Q[:, 0] ** 2 - Q[:, 1] ** 2 - Q[:, 2] ** 2 - Q[:, 3] ** 2)
    b = -Q[:, 1:] / M[:, None]                           # [n,3]
    x = sqrt_s / M
    gamma = Q[:, 0] / M
    a = 1.0 / (1.0 + gamma)

    bq = np.einsum("nk,nik->ni", b, q[:, :, 1:])         # [n,nf]
    p0 = x[:, None] * (gamma[:, None] * q[:, :, 0] + bq)
    pv = x[:, None, None] * (q[:, :, 1:] + b[:, None, :] * q[:, :, 0:1]
                             + (a[:, None] * bq)[:, :, None] * b[:, None, :])

    # massive rescaling: solve sum_i sqrt(m_i^2 + xi^2 p0_i^2) = sqrt_s by Newton
    xi = np.sqrt(np.maximum(0.0, 1.0 - (m.sum(axis=1) / sqrt_s) ** 2))
    if np.any(m != 0.0):
        for _ in range(60):
            e = np.sqrt(m * m + (xi[:, None] * p0) ** 2)
            f = e.sum(axis=1) - sqrt_s
            if np.all(np.abs(f) < 1e-14 * sqrt_s):
                break
            df = (xi[:, None] * p0 * p0 / e).sum(axis=1)
            xi = xi - f / df
    else:
        xi = np.ones(n)
    out = np.empty((n, nf, 4), dtype=np.float64)
    out[:, :, 1:] = xi[:, None, None] * pv
    out[:, :, 0] = np.sqrt(m * m + (xi[:, None] * p0) ** 2)
    return out
