"""The five seeded workloads of BASELINE.json `configs` (recipe: DESIGN.md section 4).

Only input generation lives here: flavour labels, keys, phase-space points, weights and
parameter vectors. No amplitude or bucketing arithmetic.
"""
from dataclasses import dataclass, field

import numpy as np

from .rambo import massive_rambo

# theta[] layout (include/rex_trex.h; replaces the SLHA `BLOCK ID VALUE` cards of PAPER.md:996-1002)
NTHETA = 16
TH_ALPHA_S, TH_ALPHA_EM, TH_SIN2W, TH_MZ, TH_GAMMAZ = 0, 1, 2, 3, 4
TH_MT, TH_GAMMAT, TH_CTG, TH_LAMBDA, TH_VEV = 5, 6, 7, 8, 9

REX_NPOS = np.uint64(0xFFFFFFFFFFFFFFFF)


def default_theta():
    th = np.zeros(NTHETA, dtype=np.float64)
    th[TH_ALPHA_S] = 0.118
    th[TH_ALPHA_EM] = 1.0 / 132.507
    th[TH_SIN2W] = 0.2312
    th[TH_MZ] = 91.1876
    th[TH_GAMMAZ] = 2.4952
    th[TH_MT] = 173.0
    th[TH_GAMMAT] = 0.0
    th[TH_CTG] = 0.0
    th[TH_LAMBDA] = 1000.0
    th[TH_VEV] = 246.22
    return th


def pack_key(pdg, status):
    """Canonical flavour signature (include/rex_trex.h `rex_pack_key`):
    initial-state (status -1) PDG codes sorted ascending, then final-state (status +1) codes
    sorted ascending, one byte each ((pdg & 0x7F) | 0x80 if negative), byte 7 = (n_in<<4)|n_out."""
    ini = sorted(int(p) for p, s in zip(pdg, status) if s == -1)
    fin = sorted(int(p) for p, s in zip(pdg, status) if s == 1)
    legs = ini + fin
    assert len(legs) <= 7
    key = 0
    for i, p in enumerate(legs):
        b = (abs(p) & 0x7F) | (0x80 if p < 0 else 0)
        key |= b << (8 * i)
    key |= ((len(ini) << 4) | len(fin)) << 56
    return np.uint64(key)


@dataclass(frozen=True)
class Subprocess:
    sid: int            # compiled-in subprocess id (include/rex_trex.h)
    name: str
    pdg: tuple          # process-string order
    status: tuple       # -1 incoming, +1 outgoing
    top_legs: tuple     # indices of massive (top) legs

    @property
    def npar(self):
        return len(self.pdg)

    @property
    def key(self):
        return pack_key(self.pdg, self.status)


SUBPROCESSES = (
    Subprocess(0, "e- e+ > mu- mu+", (11, -11, 13, -13), (-1, -1, 1, 1), ()),
    Subprocess(1, "g g > t t~", (21, 21, 6, -6), (-1, -1, 1, 1), (2, 3)),
    Subprocess(2, "g g > t t~ g", (21, 21, 6, -6, 21), (-1, -1, 1, 1, 1), (2, 3)),
    Subprocess(3, "g g > t t~ g g", (21, 21, 6, -6, 21, 21), (-1, -1, 1, 1, 1, 1), (2, 3)),
    Subprocess(4, "g g > t t~ g g g", (21, 21, 6, -6, 21, 21, 21), (-1, -1, 1, 1, 1, 1, 1), (2, 3)),
    Subprocess(5, "u u~ > t t~ g", (2, -2, 6, -6, 21), (-1, -1, 1, 1, 1), (2, 3)),
    Subprocess(6, "d d~ > t t~ g", (1, -1, 6, -6, 21), (-1, -1, 1, 1, 1), (2, 3)),
    Subprocess(7, "u g > t t~ u", (2, 21, 6, -6, 2), (-1, -1, 1, 1, 1), (2, 3)),
    Subprocess(8, "g u~ > t t~ u~", (21, -2, 6, -6, -2), (-1, -1, 1, 1, 1), (2, 3)),
)


def _light_line_channels():
    """The one-light-line channels for the other massless flavours (labels only; QCD does not see the flavour): ids
    10, 11, 12 = s s~, c c~, b b~ > t t~ g; 13..16 = d g, s g, c g, b g > t t~ q; 17..20 = g d~, g s~, g c~, g b~ > t t~ q~.
    (The two beam orders of a channel share one flavour key -- legs are compared unordered, PAPER.md:334 -- and are
    brought to the order of the process string by the parton re-indexing of trex_run_pdg.)"""
    name = {1: "d", 2: "u", 3: "s", 4: "c", 5: "b"}
    out, sid = [], 10
    for f in (3, 4, 5):
        out.append(Subprocess(sid, "%s %s~ > t t~ g" % (name[f], name[f]), (f, -f, 6, -6, 21), (-1, -1, 1, 1, 1), (2, 3))); sid += 1
    for f in (1, 3, 4, 5):
        out.append(Subprocess(sid, "%s g > t t~ %s" % (name[f], name[f]), (f, 21, 6, -6, f), (-1, -1, 1, 1, 1), (2, 3))); sid += 1
    for f in (1, 3, 4, 5):
        out.append(Subprocess(sid, "g %s~ > t t~ %s~" % (name[f], name[f]), (21, -f, 6, -6, -f), (-1, -1, 1, 1, 1), (2, 3))); sid += 1
    return tuple(out)


def _two_gluon_channels():
    """One light line + two gluons (ids 21..35): u u~ > t t~ g g, u g > t t~ u g, g u~ > t t~ u~ g and the
    same three for d, s, c, b (labels only: QCD does not see the flavour of a massless quark)."""
    name = {1: "d", 2: "u", 3: "s", 4: "c", 5: "b"}
    out, sid = [], 21
    for f in (2, 1, 3, 4, 5):
        q = name[f]
        out.append(Subprocess(sid, "%s %s~ > t t~ g g" % (q, q), (f, -f, 6, -6, 21, 21), (-1, -1, 1, 1, 1, 1), (2, 3))); sid += 1
        out.append(Subprocess(sid, "%s g > t t~ %s g" % (q, q), (f, 21, 6, -6, f, 21), (-1, -1, 1, 1, 1, 1), (2, 3))); sid += 1
        out.append(Subprocess(sid, "g %s~ > t t~ %s~ g" % (q, q), (21, -f, 6, -6, -f, 21), (-1, -1, 1, 1, 1, 1), (2, 3))); sid += 1
    return tuple(out)


SUBPROCESSES = SUBPROCESSES + _light_line_channels() + _two_gluon_channels()


def subprocess_by_name(name):
    for sp in SUBPROCESSES:
        if sp.name == name:
            return sp
    raise KeyError(name)


def subprocess_by_key(key):
    for sp in SUBPROCESSES:
        if sp.key == np.uint64(key):
            return sp
    return None


@dataclass
class Workload:
    cfg: int
    name: str
    n: int
    npar: int
    keys: np.ndarray          # uint64 [n] flavour signature per event, input order
    momenta: np.ndarray       # float64 [npar, 4, n] SoA, (E,px,py,pz), GeV, input order
    w_in: np.ndarray          # float64 [n]
    theta_old: np.ndarray     # float64 [NTHETA]
    theta_new: np.ndarray     # float64 [NTHETA]
    classes: tuple = field(default_factory=tuple)   # Subprocess objects present


def _two_to_n(rng, n, sqrt_s_range, masses, draw_sqrt_s):
    """Draw per event: [sqrt_s if random], then (r1..r4) for each final particle in order."""
    nf = len(masses)
    if draw_sqrt_s:
        u = rng.random((n, 1 + 4 * nf))
        lo, hi = sqrt_s_range
        sqrt_s = lo + (hi - lo) * u[:, 0]
        r = u[:, 1:].reshape(n, nf, 4)
    else:
        sqrt_s = np.full(n, float(sqrt_s_range))
        r = rng.random((n, 4 * nf)).reshape(n, nf, 4)
    fin = massive_rambo(r, sqrt_s, masses)               # [n,nf,4]
    mom = np.empty((2 + nf, 4, n), dtype=np.float64)
    mom[0] = np.stack([sqrt_s / 2, np.zeros(n), np.zeros(n), sqrt_s / 2])
    mom[1] = np.stack([sqrt_s / 2, np.zeros(n), np.zeros(n), -sqrt_s / 2])
    mom[2:] = np.transpose(fin, (1, 2, 0))
    return np.ascontiguousarray(mom)


def largest_remainder(fracs, n):
    raw = np.asarray(fracs, dtype=np.float64) * n
    base = np.floor(raw).astype(np.int64)
    rem = n - int(base.sum())
    order = np.argsort(-(raw - base), kind="stable")
    base[order[:rem]] += 1
    return base


def make_config(cfg, n=None):
    """Build workload `cfg` in 1..5 (BASELINE.json configs[cfg-1]); `n` overrides the event count
    (a seeded prefix-equivalent smaller sample drawn with the same recipe)."""
    th_old, th_new = default_theta(), default_theta()
    mt = th_old[TH_MT]
    if cfg == 1:
        n = 4096 if n is None else n
        rng = np.random.default_rng(0)
        u = rng.random((n, 2))
        c = 2.0 * u[:, 0] - 1.0
        phi = 2.0 * np.pi * u[:, 1]
        e = 91.1876 / 2.0
        s = np.sqrt(1.0 - c * c)
        z = np.zeros(n)
        mom = np.empty((4, 4, n))
        mom[0] = np.stack([np.full(n, e), z, z, np.full(n, e)])
        mom[1] = np.stack([np.full(n, e), z, z, np.full(n, -e)])
        mom[2] = np.stack([np.full(n, e), e * s * np.cos(phi), e * s * np.sin(phi), e * c])
        mom[3] = np.stack([np.full(n, e), -mom[2][1], -mom[2][2], -mom[2][3]])
        th_new[TH_SIN2W] = 0.2400
        sp = SUBPROCESSES[0]
        return Workload(1, "cfg1 e+e- -> mu+mu- (gamma+Z)", n, 4, np.full(n, sp.key, dtype=np.uint64),
                        mom, np.ones(n), th_old, th_new, (sp,))
    if cfg == 2:
        n = 65536 if n is None else n
        rng = np.random.default_rng(1)
        mom = _two_to_n(rng, n, (400.0, 2000.0), [mt, mt], True)
        w = rng.lognormal(0.0, 0.5, n)
        th_new[TH_CTG] = 0.5
        sp = SUBPROCESSES[1]
        return Workload(2, "cfg2 gg -> tt~ (+c_tG)", n, 4, np.full(n, sp.key, dtype=np.uint64),
                        mom, w, th_old, th_new, (sp,))
    if cfg == 3:
        n = 1048576 if n is None else n
        rng = np.random.default_rng(2)
        classes = (SUBPROCESSES[2], SUBPROCESSES[5], SUBPROCESSES[6], SUBPROCESSES[7], SUBPROCESSES[8])
        counts = largest_remainder([0.60, 0.10, 0.05, 0.15, 0.10], n)
        labels = np.concatenate([np.full(int(c), i, dtype=np.int64) for i, c in enumerate(counts)])
        labels = rng.permutation(labels)
        class_keys = np.array([sp.key for sp in classes], dtype=np.uint64)
        keys = class_keys[labels]
        mom = _two_to_n(rng, n, (500.0, 3000.0), [mt, mt, 0.0], True)
        w = rng.lognormal(0.0, 0.5, n)
        th_new[TH_CTG] = 1.0
        return Workload(3, "cfg3 mixed pp -> tt~ + 1 parton", n, 5, keys, mom, w, th_old, th_new, classes)
    if cfg == 4:
        n = 1048576 if n is None else n
        rng = np.random.default_rng(3)
        mom = _two_to_n(rng, n, 1500.0, [mt, mt, 0.0, 0.0], False)
        th_old[TH_GAMMAT] = 1.50
        th_new[TH_GAMMAT] = 1.35
        th_new[TH_CTG] = 0.3
        sp = SUBPROCESSES[3]
        return Workload(4, "cfg4 gg -> tt~gg", n, 6, np.full(n, sp.key, dtype=np.uint64),
                        mom, np.ones(n), th_old, th_new, (sp,))
    if cfg == 5:
        n = 262144 if n is None else n
        rng = np.random.default_rng(4)
        mom = _two_to_n(rng, n, 2000.0, [mt, mt, 0.0, 0.0, 0.0], False)
        th_new[TH_CTG] = 0.5
        sp = SUBPROCESSES[4]
        return Workload(5, "cfg5 gg -> tt~ggg", n, 7, np.full(n, sp.key, dtype=np.uint64),
                        mom, np.ones(n), th_old, th_new, (sp,))
    if cfg == 6:
        # multi-channel p p -> t t~ + 1 parton sample with every one-light-line channel (16 classes; the paper's QCD sample has
        # 65 distinct parton configurations): g g > t t~ g 45 %, the rest shared among the quark channels with
        # parton-density-like weights (u : d : s : c : b = 8 : 4 : 2 : 1 : 1; q g twice as likely as q q~; antiquark-initiated
        # channels half as likely as quark-initiated ones). Same recipe as cfg 3 otherwise.
        n = 1048576 if n is None else n
        rng = np.random.default_rng(6)
        classes = tuple(sp for sp in SUBPROCESSES if sp.npar == 5)
        fw = {1: 4.0, 2: 8.0, 3: 2.0, 4: 1.0, 5: 1.0}
        wts = []
        for sp in classes:
            ini = sp.pdg[:2]
            if ini == (21, 21):
                wts.append(0.0)
                continue
            f = [abs(x) for x in ini if x != 21][0]
            kind_w = 2.0 if 21 in ini else 1.0
            anti_w = 0.5 if (21 in ini and min(ini) < 0) else 1.0
            wts.append(fw[f] * kind_w * anti_w)
        wts = np.array(wts)
        fr = 0.55 * wts / wts.sum()
        fr[[i for i, sp in enumerate(classes) if sp.pdg[:2] == (21, 21)][0]] = 0.45
        counts = largest_remainder(fr, n)
        labels = np.concatenate([np.full(int(c), i, dtype=np.int64) for i, c in enumerate(counts)])
        labels = rng.permutation(labels)
        class_keys = np.array([sp.key for sp in classes], dtype=np.uint64)
        keys = class_keys[labels]
        mom = _two_to_n(rng, n, (500.0, 3000.0), [mt, mt, 0.0], True)
        w = rng.lognormal(0.0, 0.5, n)
        th_new[TH_CTG] = 1.0
        present = tuple(sp for sp, c in zip(classes, counts) if c > 0)
        return Workload(6, "cfg6 multi-channel pp -> tt~ + 1 parton, 16 classes", n, 5, keys, mom, w, th_old, th_new, present)
    if cfg == 7:
        # multi-channel p p -> t t~ + 2 partons sample: g g > t t~ g g 50 %, q g 24 % (u : d = 2 : 1), g q~ 8 %, q q~ 18 %
        # (the multi-jet samples of PAPER.md:1279-1284 mix the gluonic channel with quark-line channels). Same phase space as
        # cfg 4 (sqrt(s) = 1500, RAMBO), theta as cfg 3.
        n = 262144 if n is None else n
        rng = np.random.default_rng(7)
        classes = tuple(sp for sp in SUBPROCESSES if sp.npar == 6 and sp.sid <= 26)
        fr = {3: 0.50, 21: 0.12, 22: 0.16, 23: 0.05, 24: 0.06, 25: 0.08, 26: 0.03}
        counts = largest_remainder([fr[sp.sid] for sp in classes], n)
        labels = np.concatenate([np.full(int(c), i, dtype=np.int64) for i, c in enumerate(counts)])
        labels = rng.permutation(labels)
        class_keys = np.array([sp.key for sp in classes], dtype=np.uint64)
        keys = class_keys[labels]
        mom = _two_to_n(rng, n, 1500.0, [mt, mt, 0.0, 0.0], False)
        w = rng.lognormal(0.0, 0.5, n)
        th_new[TH_CTG] = 1.0
        present = tuple(sp for sp, c in zip(classes, counts) if c > 0)
        return Workload(7, "cfg7 multi-channel pp -> tt~ + 2 partons, 7 classes", n, 6, keys, mom, w, th_old, th_new, present)
    raise ValueError(f"unknown config {cfg}")


def shuffled_legs(w, seed, unknown_every=0):
    """LHE-like view of a workload: per-event PDG codes [npar, n] (int32) and momenta whose legs were shuffled inside
    the initial state and inside the final state with a seeded permutation per event (an LHE file does not promise the
    parton order of the process string: PAPER.md:227-242). Returns (pdg, momenta, n_in). `unknown_every` > 0 turns
    every k-th event into a class no subprocess claims (s c~ > ...). No method arithmetic here: only labels move."""
    rng = np.random.default_rng(seed)
    npar, n = w.npar, w.n
    n_in = 2
    pdg = np.zeros((npar, n), dtype=np.int32)
    for sp in (w.classes if w.classes else ()):
        sel = w.keys == sp.key
        for leg in range(npar):
            pdg[leg, sel] = sp.pdg[leg]
    mom = w.momenta.copy()
    order = np.tile(np.arange(npar)[:, None], (1, n))
    swap = rng.random(n) < 0.5
    order[0, swap], order[1, swap] = 1, 0
    fin = np.argsort(rng.random((npar - n_in, n)), axis=0) + n_in
    order[n_in:, :] = fin
    cols = np.arange(n)
    pdg = pdg[order, cols]
    mom = np.ascontiguousarray(mom[order, :, cols].transpose(0, 2, 1))     # [npar, n, 4] -> [npar, 4, n]
    if unknown_every:
        pdg[0, ::unknown_every] = 3
        pdg[1, ::unknown_every] = -4
    return pdg, mom, n_in
