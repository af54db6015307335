"""Shared test helpers: Lorentz transformations and textbook closed forms (retyped here on purpose,
independent of oracle/ and of the CUDA path)."""
import math

import numpy as np


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


def random_lorentz(rng, max_beta=0.6):
    """A proper orthochronous Lorentz matrix: random rotation times random boost."""
    a = rng.normal(size=(3, 3))
    q, _ = np.linalg.qr(a)
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    rot = np.eye(4)
    rot[1:, 1:] = q
    d = rng.normal(size=3)
    d /= np.linalg.norm(d)
    beta = max_beta * rng.random()
    g = 1.0 / math.sqrt(1.0 - beta * beta)
    b = np.eye(4)
    b[0, 0] = g
    b[0, 1:] = b[1:, 0] = g * beta * d
    b[1:, 1:] += (g - 1.0) * np.outer(d, d)
    return b @ rot


def apply_lorentz(L, momenta):
    """momenta [npar,4,n] -> transformed."""
    return np.einsum("uv,pvn->pun", L, momenta)


# ---- closed forms (textbook results)
def eemumu_closed(mom, th):
    """F-1: me2 = 1/4 sum_{a,b in L,R} s^2 (1 + eta_a eta_b cos)^2 |e^2/s + g_a g_b / D|^2."""
    s = mdot(mom[0] + mom[1], mom[0] + mom[1])
    c = (mom[0, 1:] * mom[2, 1:]).sum(0) / np.sqrt((mom[0, 1:] ** 2).sum(0) * (mom[2, 1:] ** 2).sum(0))
    e2 = 4 * math.pi * th[1]
    sw2 = th[2]
    cw2 = 1 - sw2
    e = math.sqrt(e2)
    gl = e / math.sqrt(sw2 * cw2) * (-0.5 + sw2)
    gr = e / math.sqrt(sw2 * cw2) * sw2
    D = s - th[3] ** 2 + 1j * th[3] * th[4]
    tot = 0
    for ga, ea in ((gl, -1), (gr, 1)):
        for gb, eb in ((gl, -1), (gr, 1)):
            tot = tot + s ** 2 * (1 + ea * eb * c) ** 2 * np.abs(e2 / s + ga * gb / D) ** 2
    return tot / 4


def tau_rho(mom, mt):
    s = mdot(mom[0] + mom[1], mom[0] + mom[1])
    t = mdot(mom[0] - mom[2], mom[0] - mom[2])
    u = mdot(mom[0] - mom[3], mom[0] - mom[3])
    return (mt ** 2 - t) / s, (mt ** 2 - u) / s, 4 * mt ** 2 / s


def ggtt_sm_closed(mom, th):
    """F-2: LO gg -> tt~ averaged |M|^2."""
    t1, t2, rho = tau_rho(mom, th[5])
    gs4 = (4 * math.pi * th[0]) ** 2
    return gs4 * (1 / (6 * t1 * t2) - 3 / 8) * (t1 ** 2 + t2 ** 2 + rho - rho ** 2 / (4 * t1 * t2))


def ggtt_linear_closed(mom, th):
    """F-3: coefficient of c_tG^1 in gg -> tt~ (SM x chromomagnetic interference), per unit c_tG."""
    t1, t2, _ = tau_rho(mom, th[5])
    gs = math.sqrt(4 * math.pi * th[0])
    return 16 * math.sqrt(2) * math.pi * th[0] * gs * th[9] * th[5] / th[8] ** 2 * (1 / (6 * t1 * t2) - 3 / 8)


def qqtt_sm_closed(mom, th):
    """F-4: LO q q~ -> t t~ averaged |M|^2."""
    t1, t2, rho = tau_rho(mom, th[5])
    gs4 = (4 * math.pi * th[0]) ** 2
    return (4.0 / 9.0) * gs4 * (t1 ** 2 + t2 ** 2 + rho / 2)


def relclose(a, b, rtol):
    """Pure relative comparison (numpy's default atol=1e-8 would swallow |M|^2 values of 1e-7)."""
    a, b = np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)
    return bool(np.all(np.abs(a - b) <= rtol * np.abs(b)))
