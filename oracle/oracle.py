"""ctypes front end of the CPU oracle (TEST INFRASTRUCTURE ONLY).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import this.
The product package never does. Array conventions as in include/rex_trex.h: momenta SoA [npar][4][n].
"""
import ctypes
import math

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(_build.build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        L.oracle_npar.argtypes = [ctypes.c_int]
        L.oracle_me2.argtypes = [ctypes.c_int, dp, ctypes.c_long, dp, dp, ctypes.c_int]
        L.oracle_abd.argtypes = [ctypes.c_int, ctypes.c_int, dp, ctypes.c_long, dp, ctypes.c_int, ctypes.c_int, dp, ctypes.c_int]
        L.oracle_reweight.argtypes = [ctypes.c_int, dp, ctypes.c_long, dp, dp, dp, dp, dp, dp, ctypes.c_int]
        L.oracle_ttng_amps.argtypes = [ctypes.c_int, dp, dp, ctypes.c_int, ctypes.c_int, dp]
        L.oracle_colour_matrix.argtypes = [ctypes.c_int, dp]
        L.oracle_colour_entry.argtypes = [ctypes.c_int, ip, ip]
        L.oracle_colour_entry.restype = ctypes.c_double
        L.oracle_wavefunction.argtypes = [ctypes.c_int, dp, ctypes.c_int, ctypes.c_int, dp]
        L.oracle_gamma.argtypes = [ctypes.c_int, dp]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _mom(sid, momenta):
    npar = lib().oracle_npar(sid)
    m = np.ascontiguousarray(momenta, dtype=np.float64)
    assert m.ndim == 3 and m.shape[0] == npar and m.shape[1] == 4, (m.shape, npar)
    return m, m.shape[2]


def me2(sid, momenta, theta, long_double=False):
    """Helicity/colour-summed, averaged |M|^2 per event at parameters theta."""
    m, n = _mom(sid, momenta)
    th = np.ascontiguousarray(theta, dtype=np.float64)
    out = np.empty(n)
    rc = lib().oracle_me2(sid, _dp(m), n, _dp(th), _dp(out), int(long_double))
    assert rc == 0, rc
    return out


def abd(sid, momenta, theta, engine=1, gauge_gluon=-1, hel_only=-1, long_double=False):
    """(A,B,D) with me2 = A + kappa B + kappa^2 D; engine 1 = colour-ordered E1, 2 = explicit-colour E2."""
    m, n = _mom(sid, momenta)
    th = np.ascontiguousarray(theta, dtype=np.float64)
    out = np.empty((n, 3))
    rc = lib().oracle_abd(sid, engine, _dp(m), n, _dp(th), gauge_gluon, hel_only, _dp(out), int(long_double))
    assert rc == 0, rc
    return out


def count_flops(sid, momenta_one, theta_old, theta_new):
    """Real additions/subtractions, multiplications, divisions and square roots the plain evaluator performs for ONE
    reweighted event (old + new |M|^2 and the weight): the evaluator instantiated on a counting scalar type
    (SURVEY.md 8(d) count (iii); BASELINE.json: "FLOPs per event counted from the oracle"). Returns a dict."""
    mom = np.ascontiguousarray(np.asarray(momenta_one, dtype=np.float64).reshape(-1, 4, 1))
    out = (ctypes.c_longlong * 4)()
    f = lib().oracle_count_flops
    f.argtypes = [ctypes.c_int, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double),
                  ctypes.POINTER(ctypes.c_longlong)]
    tho = np.ascontiguousarray(theta_old, dtype=np.float64)
    thn = np.ascontiguousarray(theta_new, dtype=np.float64)
    rc = f(int(sid), _dp(mom), _dp(tho), _dp(thn), out)
    if rc != 0:
        raise RuntimeError("oracle_count_flops failed (%d)" % rc)
    return {"add": int(out[0]), "mul": int(out[1]), "div": int(out[2]), "sqrt": int(out[3]), "flop": int(sum(out))}


def kappa(theta):
    return theta[7] * theta[9] / (math.sqrt(2.0) * theta[8] ** 2)


def reweight(sid, momenta, theta_old, theta_new, w_in, long_double=False):
    """Returns (w_out, me2_old, me2_new): eq.(5) PAPER.md:714 with the zero guard of PAPER.md:789-799."""
    m, n = _mom(sid, momenta)
    to = np.ascontiguousarray(theta_old, dtype=np.float64)
    tn = np.ascontiguousarray(theta_new, dtype=np.float64)
    w = np.ascontiguousarray(w_in, dtype=np.float64)
    w_out, mo, mn = np.empty(n), np.empty(n), np.empty(n)
    rc = lib().oracle_reweight(sid, _dp(m), n, _dp(to), _dp(tn), _dp(w), _dp(w_out), _dp(mo), _dp(mn), int(long_double))
    assert rc == 0, rc
    return w_out, mo, mn


def reweight_alphas(sid, momenta, theta_old, theta_new, alpha_s, w_in):
    """Reweighting with a per-event strong coupling (an LHE event carries its own alpha_s; g_S per event: PAPER.md:66-67,
    104): for event i both parameter points are evaluated with theta[0] = alpha_s[i]. Written as its definition: one plain
    `reweight` call per event with the two parameter vectors changed in that one entry."""
    m, n = _mom(sid, momenta)
    w_out, mo, mn = np.empty(n), np.empty(n), np.empty(n)
    for i in range(n):
        to = np.array(theta_old, dtype=np.float64)
        tn = np.array(theta_new, dtype=np.float64)
        to[0] = tn[0] = alpha_s[i]
        w_out[i:i + 1], mo[i:i + 1], mn[i:i + 1] = reweight(sid, np.ascontiguousarray(m[:, :, i:i + 1]), to, tn, w_in[i:i + 1])
    return w_out, mo, mn


def ttng_amps(sid, momenta_one, theta, hel, gauge_gluon=-1):
    """Colour-flow amplitudes A_sigma (order 0 and order 1 in kappa) of one event and one helicity index.
    Returns complex array [n!, 2]; orderings lexicographic."""
    m, n = _mom(sid, momenta_one)
    assert n == 1
    npar = m.shape[0]
    nperm = math.factorial(npar - 2)
    out = np.empty((nperm, 4))
    th = np.ascontiguousarray(theta, dtype=np.float64)
    rc = lib().oracle_ttng_amps(sid, _dp(m), _dp(th), hel, gauge_gluon, _dp(out))
    assert rc == 0, rc
    return out[:, 0::2] + 1j * out[:, 1::2]


def colour_matrix(n):
    k = math.factorial(n)
    out = np.empty((k, k))
    assert lib().oracle_colour_matrix(n, _dp(out)) == 0
    return out


def colour_entry(sigma, sigma_p):
    n = len(sigma)
    a = (ctypes.c_int * n)(*sigma)
    b = (ctypes.c_int * n)(*sigma_p)
    return lib().oracle_colour_entry(n, a, b)


def wavefunction(kind, p, lam, massless=False):
    """kind: 'u','v','ubar','vbar','eps' -> complex[4]. massless=True: E := |p| (R-2)."""
    k = {"u": 0, "v": 1, "ubar": 2, "vbar": 3, "eps": 4}[kind]
    pp = np.ascontiguousarray(p, dtype=np.float64)
    out = np.empty(8)
    assert lib().oracle_wavefunction(k, _dp(pp), lam, int(massless), _dp(out)) == 0
    return out[0::2] + 1j * out[1::2]


def gamma(mu):
    out = np.empty(32)
    assert lib().oracle_gamma(mu, _dp(out)) == 0
    return (out[0::2] + 1j * out[1::2]).reshape(4, 4)


# ---------------------------------------------------------------- bucketing oracle (R-10)
def bucket(keys):
    """Stable categorisation: buckets ordered by first appearance of their key, REX_NPOS forced last.
    Returns (perm int32[n], offsets int64[nb+1], bucket_keys uint64[nb])."""
    keys = np.asarray(keys, dtype=np.uint64)
    npos = np.uint64(0xFFFFFFFFFFFFFFFF)
    order = []
    seen = {}
    for k in keys.tolist():
        if k not in seen and k != int(npos):
            seen[k] = len(order)
            order.append(k)
    has_npos = bool(np.any(keys == npos))
    if has_npos:
        seen[int(npos)] = len(order)
        order.append(int(npos))
    bid = np.array([seen[k] for k in keys.tolist()], dtype=np.int64)
    perm = np.argsort(bid, kind="stable").astype(np.int32)
    counts = np.bincount(bid, minlength=len(order)) if len(order) else np.zeros(0, dtype=np.int64)
    offsets = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    return perm, offsets, np.array(order, dtype=np.uint64)


def gather(src, perm):
    """dst[r, j] = src[r, perm[j]] (the SoA 'transpose' of PAPER.md:100, 691)."""
    src = np.asarray(src)
    return np.ascontiguousarray(src.reshape(-1, src.shape[-1])[:, perm]).reshape(src.shape[:-1] + (len(perm),))


# ---------------------------------------------------------------- reweighted cross section and its error (NEXT-2)
def xsec(w_in, w_out, C, sigma, dsigma):
    """Reweighted cross section and propagated error, written out from PAPER.md:942-948:

        sigma'       = C * sum_i w'_i                                                   eq.(6)
        Delta sigma' = Delta sigma * (1/N) sum_i w'_i / w_i  +  sigma * std(w')         eq.(7)

    std = population standard deviation (divide by N; R-15). Events with w_i = 0 carry w'_i = 0 by the zero
    guard of PAPER.md:789-799 and add nothing to the ratio sum (R-16). If the propagated error is infinite, NaN or not
    positive it is replaced by Delta sigma times whichever of sigma'/sigma, sigma/sigma' is greater than one
    (PAPER.md:948). Returns (sigma', Delta sigma', fallback_used). Plain Python / math.fsum: exact sums.
    """
    w_in = np.asarray(w_in, dtype=np.float64)
    w_out = np.asarray(w_out, dtype=np.float64)
    n = len(w_out)
    if n == 0:
        return 0.0, float(dsigma), True
    s1 = math.fsum(w_out.tolist())
    sigma_p = C * s1
    ratio = math.fsum([wo / wi for wo, wi in zip(w_out.tolist(), w_in.tolist()) if wi != 0.0]) / n
    mean = s1 / n
    var = math.fsum([(x - mean) * (x - mean) for x in w_out.tolist()]) / n
    d = dsigma * ratio + sigma * math.sqrt(var)
    fallback = not (math.isfinite(d) and d > 0.0)
    if fallback:
        r = sigma_p / sigma if sigma != 0.0 else float("nan")
        d = dsigma * max(r, 1.0 / r) if (math.isfinite(r) and r > 0.0) else float(dsigma)
    return sigma_p, d, fallback


# ---------------------------------------------------------------- flavour keys and parton re-indexing (NEXT-3)
def flavour_key(pdg, n_in):
    """Flavour signature of one event from its PDG codes (first n_in legs incoming): initial-state codes sorted
    ascending, then final-state codes sorted ascending -- two events are the same process iff their unordered initial and
    final flavour content agree (default comparator). One byte per leg ((|pdg| & 0x7F) | 0x80 if
    negative), byte 7 = (n_in << 4) | n_out; codes beyond 127 or more than 7 legs give REX_NPOS (all ones)."""
    legs = sorted(int(p) for p in pdg[:n_in]) + sorted(int(p) for p in pdg[n_in:])
    if len(legs) > 7 or any(abs(p) > 127 for p in legs):
        return np.uint64(0xFFFFFFFFFFFFFFFF)
    key = 0
    for i, p in enumerate(legs):
        key |= ((abs(p) & 0x7F) | (0x80 if p < 0 else 0)) << (8 * i)
    key |= ((n_in << 4) | (len(legs) - n_in)) << 56
    return np.uint64(key)


def comparator_equal(pdg1, status1, pdg2, status2, status_filter=(-1, 1)):
    """The event comparison an eventComparatorConfig with set_pdg(true) and the given status_filter defines
    (PAPER.md:227-231): only partons whose status is in status_filter take part (an empty filter means no filtering),
    and two events are equal iff those partons agree as unordered (status, PDG code) collections (the default comparator
    compares unordered external legs; Alg.1). Written out as the definition."""
    def legs(pdg, status):
        return sorted((int(s), int(p)) for p, s in zip(pdg, status) if len(status_filter) == 0 or int(s) in status_filter)
    return legs(pdg1, status1) == legs(pdg2, status2)


def flavour_key_filtered(pdg, status, status_filter=(-1, 1)):
    """Key of one event under the comparator above: the partons the filter keeps, incoming (status < 0) first, then
    final (status 1), then everything else (intermediate: 2, 3, ...), each group sorted ascending by PDG code; one byte
    per parton as in flavour_key; byte 7 = n_other << 6 | n_in << 4 | n_out. More than 7 kept partons, more than 3
    incoming or intermediate ones, statuses outside {-1, 1, 2}, or |pdg| > 127 give REX_NPOS. For events without
    intermediate partons and the filter {-1, 1} this is flavour_key."""
    keep = [(int(s), int(p)) for p, s in zip(pdg, status) if len(status_filter) == 0 or int(s) in status_filter]
    ini = sorted(p for s, p in keep if s == -1)
    fin = sorted(p for s, p in keep if s == 1)
    oth = sorted(p for s, p in keep if s == 2)
    legs = ini + fin + oth
    if (len(legs) != len(keep) or len(legs) > 7 or len(ini) > 3 or len(oth) > 3 or any(abs(p) > 127 for p in legs)):
        return np.uint64(0xFFFFFFFFFFFFFFFF)
    key = 0
    for i, p in enumerate(legs):
        key |= ((abs(p) & 0x7F) | (0x80 if p < 0 else 0)) << (8 * i)
    key |= ((len(oth) << 6) | (len(ini) << 4) | len(fin)) << 56
    return np.uint64(key)


def keys_and_legmap(pdg, n_in, process_strings):
    """pdg int [npar, n]; process_strings: the PDG tuples of the compiled-in subprocesses in process-string order.
    Returns (keys uint64 [n], legmap int8 [npar, n]): legmap[pos, i] = the leg of event i that plays position `pos` of the
    process string of the subprocess with the same flavour key (partons are re-indexed to the
    representative's order) -- for every position, in order, the FIRST not yet used leg on the same side (initial /
    final) with that PDG code, so identical particles keep their event order. Events no subprocess claims map to the
    identity. Plain loops."""
    pdg = np.asarray(pdg)
    npar, n = pdg.shape
    table = {int(flavour_key(np.array(ps), n_in)): ps for ps in process_strings if len(ps) == npar}
    keys = np.zeros(n, dtype=np.uint64)
    legmap = np.zeros((npar, n), dtype=np.int8)
    for i in range(n):
        ev = [int(x) for x in pdg[:, i]]
        k = flavour_key(ev, n_in)
        keys[i] = k
        ps = table.get(int(k))
        if ps is None:
            legmap[:, i] = np.arange(npar)
            continue
        used = [False] * npar
        for pos in range(npar):
            side = range(0, n_in) if pos < n_in else range(n_in, npar)
            for leg in side:
                if not used[leg] and ev[leg] == ps[pos]:
                    used[leg] = True
                    legmap[pos, i] = leg
                    break
    return keys, legmap
