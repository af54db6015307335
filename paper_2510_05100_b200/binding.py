"""ctypes binding of librex_trex.so: same names as include/rex_trex.h, argument marshalling only."""
import ctypes
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(HERE, "librex_trex.so")

REX_MAX_BUCKETS = 256
REX_NPOS = 0xFFFFFFFFFFFFFFFF
TREX_NTHETA = 16
SUBPROCESS_IDS = {
    "e- e+ > mu- mu+": 0, "g g > t t~": 1, "g g > t t~ g": 2, "g g > t t~ g g": 3, "g g > t t~ g g g": 4,
    "u u~ > t t~ g": 5, "d d~ > t t~ g": 6, "u g > t t~ u": 7, "g u~ > t t~ u~": 8,
    "s s~ > t t~ g": 10, "c c~ > t t~ g": 11, "b b~ > t t~ g": 12,
    "d g > t t~ d": 13, "s g > t t~ s": 14, "c g > t t~ c": 15, "b g > t t~ b": 16,
    "g d~ > t t~ d~": 17, "g s~ > t t~ s~": 18, "g c~ > t t~ c~": 19, "g b~ > t t~ b~": 20,
}


class TrexError(RuntimeError):
    pass


_lib = None
_vp, _i64, _i32, _int = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_int
_dp = ctypes.POINTER(ctypes.c_double)
_SIGNATURES = {
    "rex_pack_key": (ctypes.c_uint64, [ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int8), _int]),
    "rex_pack_key_filtered": (ctypes.c_uint64, [ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int8), _int, ctypes.POINTER(ctypes.c_int32), _int]),
    "rex_keys_filtered": (_int, [_vp, _vp, _int, _i64, ctypes.POINTER(ctypes.c_int32), _int, _vp]),
    "rex_bucket": (_int, [_vp, _i64, _vp, ctypes.POINTER(ctypes.c_int64)]),
    "rex_bucket_keys": (_int, [ctypes.POINTER(ctypes.c_uint64)]),
    "rex_gather": (_int, [_vp, _i64, _vp, _i64, _int, _vp]),
    "rex_scatter": (_int, [_vp, _i64, _vp, _i64, _int, _vp]),
    "trex_subproc_id": (_int, [ctypes.c_uint64]),
    "trex_npar": (_int, [_int]),
    "trex_ncolor": (_int, [_int]),
    "trex_nhel": (_int, [_int]),
    "trex_colour_matrix": (_int, [_int, _dp]),
    "trex_reweight": (_int, [_int, _vp, _i64, _dp, _dp, _vp, _vp, _vp, _vp]),
    "trex_run": (_int, [_vp, _vp, _i64, _int, _dp, _dp, _vp, _vp, _vp, _vp]),
    "rex_keys": (_int, [_vp, _int, _int, _i64, _vp, _vp]),
    "trex_run_pdg": (_int, [_vp, _vp, _i64, _int, _int, _dp, _dp, _vp, _vp, _vp, _vp]),
    "trex_run_multi": (_int, [_vp, _vp, _i64, _int, _dp, _dp, _int, _vp, _vp, _vp, _vp]),
    "trex_run_alphas": (_int, [_vp, _vp, _i64, _int, _dp, _dp, _vp, _vp, _vp, _vp, _vp]),
    "trex_run_host": (_int, [_vp, _vp, _i64, _int, _dp, _dp, _vp, _vp, _vp, _vp]),
    "trex_debug_flow_amps": (_int, [_int, _dp, _dp, _dp]),
    "trex_debug_xtile": (_int, [_int, _dp, _dp, _dp, _dp]),
    "trex_debug_helicity_me2": (_int, [_int, _dp, _dp, _dp, _dp]),
    "trex_probe_fma": (ctypes.c_double, [_int, _int, _int]),
    "trex_xsec_moments": (_int, [_vp, _vp, ctypes.c_int64, _vp]),
    "trex_xsec_moments_noalloc": (_int, [_vp, _vp, ctypes.c_int64, _vp]),
    "trex_xsec_finish": (_int, [_vp, _int, ctypes.c_double, ctypes.c_double, ctypes.c_double, _vp]),
    "trex_set_stream": (_int, [_vp]),
    "trex_set_precision": (_int, [_int]),
    "trex_get_precision": (_int, []),
    "trex_set_poly_multi": (_int, [_int]),
    "trex_set_helicity_symmetry": (_int, [_int]),
    "trex_set_algorithm": (_int, [_int]),
    "trex_launch_count": (ctypes.c_int64, []),
    "trex_graph_replays": (ctypes.c_int64, []),
    "trex_kernel_timing": (_int, [_int]),
    "trex_kernel_time": (_int, [_dp, ctypes.POINTER(ctypes.c_int64)]),
    "trex_last_error": (ctypes.c_char_p, []),
    "trex_shutdown": (None, []),
}


def library_path():
    return _LIB_PATH


def exported_symbols():
    """Names the binding expects the library to export (one per declaration in include/rex_trex.h and rex_trex_diag.h)."""
    return sorted(_SIGNATURES)


def lib():
    """Load librex_trex.so. Fails loudly when it has not been built: there is no fallback path."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise TrexError("librex_trex.so is not built: run `python -m paper_2510_05100_b200.build` "
                            "(or __graft_entry__.build()); there is no CPU fallback")
        L = ctypes.CDLL(_LIB_PATH)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def _check(rc, what):
    if rc < 0:
        raise TrexError("%s failed (%d): %s" % (what, rc, lib().trex_last_error().decode()))
    return rc


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise TrexError("no CUDA device: the reweighting path has no CPU fallback")
    return torch


def _dev(t, dtype, what):
    """Device pointer of a contiguous CUDA tensor of the given dtype (None -> NULL)."""
    if t is None:
        return None
    torch = _torch()
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TrexError("%s must be a contiguous CUDA tensor of dtype %s" % (what, dtype))
    return ctypes.c_void_p(t.data_ptr())


def _theta(th):
    a = np.ascontiguousarray(th, dtype=np.float64)
    if a.shape != (TREX_NTHETA,):
        raise TrexError("theta must have %d entries" % TREX_NTHETA)
    return a, a.ctypes.data_as(_dp)


def _shapes(what, n, momenta_soa=None, keys=None, rows=(), mats=(), K=None):
    """Every array of a path call must agree with n (and npar): a mismatch would be an out-of-bounds access on the device."""
    if momenta_soa is not None:
        sh = tuple(momenta_soa.shape)
        if len(sh) != 3 or sh[1] != 4 or sh[2] != n or not 1 <= sh[0] <= 7:
            raise TrexError("%s: momenta_soa must have shape (npar <= 7, 4, %d), got %s" % (what, n, sh))
    if keys is not None and int(np.prod(keys.shape)) != n:
        raise TrexError("%s: pdg_keys must have %d entries, got %s" % (what, n, tuple(keys.shape)))
    for name, t in rows:
        if t is not None and int(np.prod(t.shape)) != n:
            raise TrexError("%s: %s must have %d entries, got %s" % (what, name, n, tuple(t.shape)))
    for name, t in mats:
        if t is not None and tuple(t.shape) != (K, n):
            raise TrexError("%s: %s must have shape (%d, %d), got %s" % (what, name, K, n, tuple(t.shape)))


# ---------------------------------------------------------------- host helpers
def rex_pack_key(pdg, status):
    p = np.ascontiguousarray(pdg, dtype=np.int32)
    s = np.ascontiguousarray(status, dtype=np.int8)
    return int(lib().rex_pack_key(p.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)),
                                  s.ctypes.data_as(ctypes.POINTER(ctypes.c_int8)), len(p)))


def rex_pack_key_filtered(pdg, status, status_filter=(-1, 1)):
    p = np.ascontiguousarray(pdg, dtype=np.int32)
    s = np.ascontiguousarray(status, dtype=np.int8)
    f = np.ascontiguousarray(list(status_filter), dtype=np.int32)
    return int(lib().rex_pack_key_filtered(p.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), s.ctypes.data_as(ctypes.POINTER(ctypes.c_int8)),
                                           len(p), f.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), len(f)))


def trex_subproc_id(key):
    return lib().trex_subproc_id(ctypes.c_uint64(int(key)))


def trex_npar(sid):
    return lib().trex_npar(sid)


def trex_ncolor(sid):
    return lib().trex_ncolor(sid)


def trex_nhel(sid):
    return lib().trex_nhel(sid)


def trex_colour_matrix(sid):
    nc = _check(trex_ncolor(sid), "trex_ncolor")
    out = np.empty((nc, nc))
    _check(lib().trex_colour_matrix(sid, out.ctypes.data_as(_dp)), "trex_colour_matrix")
    return out


def trex_set_stream(stream=None):
    """stream: torch.cuda.Stream, raw cudaStream_t integer, or None for the legacy default stream."""
    h = 0 if stream is None else int(getattr(stream, "cuda_stream", stream))
    return _check(lib().trex_set_stream(ctypes.c_void_p(h)), "trex_set_stream")


def trex_set_precision(mode):
    return _check(lib().trex_set_precision(int(mode)), "trex_set_precision")


def trex_set_algorithm(algo):
    return _check(lib().trex_set_algorithm(int(algo)), "trex_set_algorithm")


def trex_set_helicity_symmetry(on):
    return _check(lib().trex_set_helicity_symmetry(int(bool(on))), "trex_set_helicity_symmetry")


def trex_set_poly_multi(on):
    return _check(lib().trex_set_poly_multi(int(bool(on))), "trex_set_poly_multi")


def trex_get_precision():
    return lib().trex_get_precision()


def trex_launch_count():
    return int(lib().trex_launch_count())


def trex_graph_replays():
    return int(lib().trex_graph_replays())


def trex_kernel_timing(on):
    return _check(lib().trex_kernel_timing(int(bool(on))), "trex_kernel_timing")


def trex_kernel_time():
    """(summed duration [ms], launches) of the |M|^2 launches recorded since the last call (trex_kernel_timing on)."""
    ms, cnt = ctypes.c_double(0.0), ctypes.c_int64(0)
    _check(lib().trex_kernel_time(ctypes.byref(ms), ctypes.byref(cnt)), "trex_kernel_time")
    return ms.value, cnt.value


def trex_last_error():
    return lib().trex_last_error().decode()


def trex_shutdown():
    lib().trex_shutdown()


# ---------------------------------------------------------------- device calls
def rex_bucket(pdg_keys, perm=None):
    """pdg_keys: CUDA tensor [n] (torch.int64 holding the uint64 key bits). Returns (perm int32 CUDA tensor [n],
    offsets numpy int64 [nbuckets+1], bucket_keys numpy uint64 [nbuckets])."""
    torch = _torch()
    n = pdg_keys.numel()
    if perm is None:
        perm = torch.empty(n, dtype=torch.int32, device=pdg_keys.device)
    offsets = (ctypes.c_int64 * (REX_MAX_BUCKETS + 1))()
    nb = _check(lib().rex_bucket(_dev(pdg_keys, torch.int64, "pdg_keys") if n else None, n,
                                 _dev(perm, torch.int32, "perm") if n else None, offsets), "rex_bucket")
    return perm, np.array(offsets[:nb + 1], dtype=np.int64), rex_bucket_keys()


def rex_bucket_keys():
    buf = (ctypes.c_uint64 * REX_MAX_BUCKETS)()
    nb = _check(lib().rex_bucket_keys(buf), "rex_bucket_keys")
    return np.array(buf[:nb], dtype=np.uint64)


def rex_gather(src, perm, dst=None):
    """dst[r, j] = src[r, perm[j]]; src [..., n_src] float64 CUDA (leading dims are rows), perm int32 CUDA [n_dst]."""
    torch = _torch()
    n_src, n_dst = src.shape[-1], perm.numel()
    nrows = src.numel() // n_src if n_src else 0
    if dst is None:
        dst = torch.empty(src.shape[:-1] + (n_dst,), dtype=torch.float64, device=src.device)
    _check(lib().rex_gather(_dev(src, torch.float64, "src"), n_src, _dev(dst, torch.float64, "dst"), n_dst, nrows,
                            _dev(perm, torch.int32, "perm")), "rex_gather")
    return dst


def rex_scatter(src, perm, dst):
    """dst[r, perm[j]] = src[r, j]."""
    torch = _torch()
    n_src, n_dst = src.shape[-1], dst.shape[-1]
    nrows = src.numel() // n_src if n_src else 0
    _check(lib().rex_scatter(_dev(src, torch.float64, "src"), n_src, _dev(dst, torch.float64, "dst"), n_dst, nrows,
                             _dev(perm, torch.int32, "perm")), "rex_scatter")
    return dst


def trex_reweight(subproc_id, momenta_soa, theta_old, theta_new, w_in, w_out=None, me2_old=None, me2_new=None,
                  want_me2=True):
    """momenta_soa [npar,4,n], w_in [n]: float64 CUDA tensors. Returns (w_out, me2_old, me2_new) CUDA tensors."""
    torch = _torch()
    n = w_in.numel()
    npar = trex_npar(subproc_id)
    if npar > 0 and tuple(momenta_soa.shape) != (npar, 4, n):
        raise TrexError("momenta_soa must have shape (%d, 4, %d), got %s" % (npar, n, tuple(momenta_soa.shape)))
    if w_out is None:
        w_out = torch.empty_like(w_in)
    if want_me2 and me2_old is None:
        me2_old = torch.empty_like(w_in)
    if want_me2 and me2_new is None:
        me2_new = torch.empty_like(w_in)
    _shapes("trex_reweight", n, rows=(("w_out", w_out), ("me2_old", me2_old), ("me2_new", me2_new)))
    to, pto = _theta(theta_old)
    tn, ptn = _theta(theta_new)
    f64 = torch.float64
    _check(lib().trex_reweight(subproc_id, _dev(momenta_soa, f64, "momenta_soa") if n else None, n, pto, ptn,
                               _dev(w_in, f64, "w_in") if n else None, _dev(w_out, f64, "w_out") if n else None,
                               _dev(me2_old, f64, "me2_old"), _dev(me2_new, f64, "me2_new")), "trex_reweight")
    return w_out, me2_old, me2_new


def trex_run(pdg_keys, momenta_soa, theta_old, theta_new, w_in, w_out=None, me2_old=None, me2_new=None, want_me2=True):
    """Whole path on device tensors in input order. Returns (w_out, me2_old, me2_new, nbuckets)."""
    torch = _torch()
    n = w_in.numel()
    npar = momenta_soa.shape[0]
    if w_out is None:
        w_out = torch.empty_like(w_in)
    if want_me2 and me2_old is None:
        me2_old = torch.empty_like(w_in)
    if want_me2 and me2_new is None:
        me2_new = torch.empty_like(w_in)
    _shapes("trex_run", n, momenta_soa, pdg_keys, rows=(("w_out", w_out), ("me2_old", me2_old), ("me2_new", me2_new)))
    to, pto = _theta(theta_old)
    tn, ptn = _theta(theta_new)
    f64 = torch.float64
    nb = _check(lib().trex_run(_dev(pdg_keys, torch.int64, "pdg_keys"), _dev(momenta_soa, f64, "momenta_soa"), n, npar,
                               pto, ptn, _dev(w_in, f64, "w_in"), _dev(w_out, f64, "w_out"),
                               _dev(me2_old, f64, "me2_old"), _dev(me2_new, f64, "me2_new")), "trex_run")
    return w_out, me2_old, me2_new, nb


def trex_run_alphas(pdg_keys, momenta_soa, theta_old, theta_new, alpha_s, w_in, w_out=None, me2_old=None, me2_new=None, want_me2=True):
    """trex_run with a per-event strong coupling: alpha_s (CUDA tensor [n]) replaces theta[0] of both parameter points for
    that event. Returns (w_out, me2_old, me2_new, nbuckets)."""
    torch = _torch()
    n = w_in.numel()
    npar = momenta_soa.shape[0]
    if w_out is None:
        w_out = torch.empty_like(w_in)
    if want_me2 and me2_old is None:
        me2_old = torch.empty_like(w_in)
    if want_me2 and me2_new is None:
        me2_new = torch.empty_like(w_in)
    _shapes("trex_run_alphas", n, momenta_soa, pdg_keys,
            rows=(("alpha_s", alpha_s), ("w_out", w_out), ("me2_old", me2_old), ("me2_new", me2_new)))
    to, pto = _theta(theta_old)
    tn, ptn = _theta(theta_new)
    f64 = torch.float64
    nb = _check(lib().trex_run_alphas(_dev(pdg_keys, torch.int64, "pdg_keys"), _dev(momenta_soa, f64, "momenta_soa"), n, npar,
                                      pto, ptn, _dev(alpha_s, f64, "alpha_s"), _dev(w_in, f64, "w_in"), _dev(w_out, f64, "w_out"),
                                      _dev(me2_old, f64, "me2_old"), _dev(me2_new, f64, "me2_new")), "trex_run_alphas")
    return w_out, me2_old, me2_new, nb


def rex_keys(pdg_soa, n_in, want_legmap=True):
    """Flavour keys (int64 view of the uint64 keys) and leg maps (int8 [npar, n]) of events given by PDG codes
    (int32 CUDA tensor [npar, n], first n_in legs incoming, any order inside each side)."""
    torch = _torch()
    npar, n = int(pdg_soa.shape[0]), int(pdg_soa.shape[1])
    keys = torch.empty(n, dtype=torch.int64, device=pdg_soa.device)
    legmap = torch.empty((npar, n), dtype=torch.int8, device=pdg_soa.device) if want_legmap else None
    _check(lib().rex_keys(_dev(pdg_soa, torch.int32, "pdg_soa"), npar, int(n_in), n, _dev(keys, torch.int64, "keys"),
                          _dev(legmap, torch.int8, "legmap")), "rex_keys")
    return keys, legmap


def rex_keys_filtered(pdg_soa, status_soa, status_filter=(-1, 1)):
    """Flavour keys under a comparator with a status filter: pdg_soa int32 [nlegs, n], status_soa int8 [nlegs, n] CUDA
    tensors; returns the keys (int64 view of the uint64 keys) [n]."""
    torch = _torch()
    nlegs, n = int(pdg_soa.shape[0]), int(pdg_soa.shape[1])
    if tuple(status_soa.shape) != (nlegs, n):
        raise TrexError("rex_keys_filtered: status_soa must have shape (%d, %d)" % (nlegs, n))
    f = np.ascontiguousarray(list(status_filter), dtype=np.int32)
    keys = torch.empty(n, dtype=torch.int64, device=pdg_soa.device)
    _check(lib().rex_keys_filtered(_dev(pdg_soa, torch.int32, "pdg_soa"), _dev(status_soa, torch.int8, "status_soa"), nlegs, n,
                                   f.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), len(f), _dev(keys, torch.int64, "keys")), "rex_keys_filtered")
    return keys


def trex_run_pdg(pdg_soa, momenta_soa, n_in, theta_old, theta_new, w_in, w_out=None, me2_old=None, me2_new=None, want_me2=True):
    """trex_run for events given by PDG codes in arbitrary parton order. Returns (w_out, me2_old, me2_new, nbuckets)."""
    torch = _torch()
    n = w_in.numel()
    npar = momenta_soa.shape[0]
    if w_out is None:
        w_out = torch.empty_like(w_in)
    if want_me2 and me2_old is None:
        me2_old = torch.empty_like(w_in)
    if want_me2 and me2_new is None:
        me2_new = torch.empty_like(w_in)
    _shapes("trex_run_pdg", n, momenta_soa, rows=(("w_out", w_out), ("me2_old", me2_old), ("me2_new", me2_new)))
    if tuple(pdg_soa.shape) != (npar, n):
        raise TrexError("trex_run_pdg: pdg_soa must have shape (%d, %d), got %s" % (npar, n, tuple(pdg_soa.shape)))
    to, pto = _theta(theta_old)
    tn, ptn = _theta(theta_new)
    f64 = torch.float64
    nb = _check(lib().trex_run_pdg(_dev(pdg_soa, torch.int32, "pdg_soa"), _dev(momenta_soa, f64, "momenta_soa"), n, npar, int(n_in),
                                   pto, ptn, _dev(w_in, f64, "w_in"), _dev(w_out, f64, "w_out"),
                                   _dev(me2_old, f64, "me2_old"), _dev(me2_new, f64, "me2_new")), "trex_run_pdg")
    return w_out, me2_old, me2_new, nb


def trex_run_multi(pdg_keys, momenta_soa, theta_old, thetas_new, w_in, w_out=None, me2_old=None, me2_new=None, want_me2=True):
    """Many parameter points on one categorisation: thetas_new [K][TREX_NTHETA]. Returns (w_out [K, n], me2_old [n],
    me2_new [K, n], nbuckets); row k is what trex_run gives for (theta_old, thetas_new[k])."""
    torch = _torch()
    n = w_in.numel()
    npar = momenta_soa.shape[0]
    tn = np.ascontiguousarray(np.asarray(thetas_new, dtype=np.float64).reshape(-1, TREX_NTHETA))
    K = tn.shape[0]
    if w_out is None:
        w_out = torch.empty((K, n), dtype=torch.float64, device=w_in.device)
    if want_me2 and me2_old is None:
        me2_old = torch.empty_like(w_in)
    if want_me2 and me2_new is None:
        me2_new = torch.empty((K, n), dtype=torch.float64, device=w_in.device)
    _shapes("trex_run_multi", n, momenta_soa, pdg_keys, rows=(("me2_old", me2_old),), mats=(("w_out", w_out), ("me2_new", me2_new)), K=K)
    to, pto = _theta(theta_old)
    f64 = torch.float64
    nb = _check(lib().trex_run_multi(_dev(pdg_keys, torch.int64, "pdg_keys"), _dev(momenta_soa, f64, "momenta_soa"), n, npar,
                                     pto, tn.ctypes.data_as(_dp), K, _dev(w_in, f64, "w_in"), _dev(w_out, f64, "w_out"),
                                     _dev(me2_old, f64, "me2_old"), _dev(me2_new, f64, "me2_new")), "trex_run_multi")
    return w_out, me2_old, me2_new, nb


def _host(t, dtype, what):
    """Host pointer of a contiguous CPU torch tensor or numpy array (None -> NULL)."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        if t.dtype != dtype or not t.flags.c_contiguous:
            raise TrexError("%s must be a C-contiguous numpy array of dtype %s" % (what, dtype))
        return ctypes.c_void_p(t.ctypes.data)
    import torch
    want = {np.float64: torch.float64, np.int64: torch.int64, np.uint64: torch.int64}[dtype]
    if t.is_cuda or not t.is_contiguous() or t.dtype != want:
        raise TrexError("%s must be a contiguous host tensor of dtype %s" % (what, want))
    return ctypes.c_void_p(t.data_ptr())


def trex_run_host(pdg_keys, momenta_soa, theta_old, theta_new, w_in, w_out, me2_old=None, me2_new=None):
    """Whole path with HOST buffers (numpy arrays or pinned CPU torch tensors); synchronous. Returns nbuckets."""
    _torch()
    n = int(np.prod(w_in.shape))
    npar = momenta_soa.shape[0]
    _shapes("trex_run_host", n, momenta_soa, pdg_keys, rows=(("w_out", w_out), ("me2_old", me2_old), ("me2_new", me2_new)))
    to, pto = _theta(theta_old)
    tn, ptn = _theta(theta_new)
    f64 = np.float64
    kdt = np.uint64 if isinstance(pdg_keys, np.ndarray) and pdg_keys.dtype == np.uint64 else np.int64
    return _check(lib().trex_run_host(_host(pdg_keys, kdt, "pdg_keys"), _host(momenta_soa, f64, "momenta_soa"), n, npar,
                                      pto, ptn, _host(w_in, f64, "w_in"), _host(w_out, f64, "w_out"),
                                      _host(me2_old, f64, "me2_old"), _host(me2_new, f64, "me2_new")), "trex_run_host")


def trex_xsec_moments(w_in, w_out):
    """(N, sum w', sum w'/w, M2) of one shard of events; device tensors in, numpy [4] out."""
    torch = _torch()
    n = int(w_out.numel())
    mom = np.zeros(4)
    _check(lib().trex_xsec_moments(_dev(w_in, torch.float64, "w_in"), _dev(w_out, torch.float64, "w_out"), n,
                                   mom.ctypes.data_as(ctypes.c_void_p)), "trex_xsec_moments")
    return mom


TREX_XSEC_NOALLOC_MAX_EVENTS = 16777216


def trex_xsec_moments_noalloc(w_in, w_out, moments_out):
    """trex_xsec_moments without any allocation inside the library: moments_out is a CUDA float64 tensor [4] of the
    caller, filled asynchronously on the library stream (N, sum w', sum w'/w, M2). At most
    TREX_XSEC_NOALLOC_MAX_EVENTS events per call."""
    torch = _torch()
    n = int(w_out.numel())
    if int(w_in.numel()) != n or moments_out is None or int(moments_out.numel()) != 4:
        raise TrexError("trex_xsec_moments_noalloc: w_in and w_out must have the same length and moments_out 4 entries")
    _check(lib().trex_xsec_moments_noalloc(_dev(w_in, torch.float64, "w_in"), _dev(w_out, torch.float64, "w_out"), n,
                                           _dev(moments_out, torch.float64, "moments_out")), "trex_xsec_moments_noalloc")
    return moments_out


def trex_xsec_finish(moments, C, sigma, dsigma):
    """Combine shard moments ([4] or [nparts, 4]) -> (sigma', Delta sigma', fallback_used). Host only: no GPU needed."""
    m = np.ascontiguousarray(np.asarray(moments, dtype=np.float64).reshape(-1, 4))
    out = np.zeros(3)
    _check(lib().trex_xsec_finish(m.ctypes.data_as(ctypes.c_void_p), int(m.shape[0]), float(C), float(sigma), float(dsigma),
                                  out.ctypes.data_as(ctypes.c_void_p)), "trex_xsec_finish")
    return float(out[0]), float(out[1]), bool(out[2])


def trex_probe_fma(fp32=False, blocks=148 * 8, iters=4096):
    """Enqueue one FMA-chain probe launch on the library stream; returns the flop count it executes."""
    _torch()
    flops = lib().trex_probe_fma(int(fp32), int(blocks), int(iters))
    if flops < 0:
        raise TrexError("trex_probe_fma failed: %s" % trex_last_error())
    return flops


def trex_debug_flow_amps(subproc_id, momenta_one, theta):
    """Colour-flow amplitudes of one event: complex array [nhel, ncolor, 2 (orders in kappa)]."""
    _torch()
    npar, nc, nh = trex_npar(subproc_id), trex_ncolor(subproc_id), trex_nhel(subproc_id)
    m = np.ascontiguousarray(momenta_one, dtype=np.float64).reshape(npar, 4)
    th, pth = _theta(theta)
    out = np.empty((nh, nc, 2, 2))
    _check(lib().trex_debug_flow_amps(subproc_id, m.ctypes.data_as(_dp), pth, out.ctypes.data_as(_dp)), "trex_debug_flow_amps")
    return out[..., 0] + 1j * out[..., 1]


def trex_debug_helicity_me2(subproc_id, momenta_one, theta_old, theta_new):
    """Per-helicity |M_h|^2 of one event from the PRODUCTION quark-channel kernels: array [nhel, 2 (theta_old, theta_new)],
    bit `leg` of h = helicity of that leg, couplings and average included."""
    _torch()
    npar, nh = trex_npar(subproc_id), trex_nhel(subproc_id)
    m = np.ascontiguousarray(momenta_one, dtype=np.float64).reshape(npar, 4)
    to, pto = _theta(theta_old)
    tn, ptn = _theta(theta_new)
    out = np.empty((nh, 2))
    _check(lib().trex_debug_helicity_me2(subproc_id, m.ctypes.data_as(_dp), pto, ptn, out.ctypes.data_as(_dp)), "trex_debug_helicity_me2")
    return out


def trex_debug_xtile(subproc_id, momenta_one, theta_old, theta_new):
    """Colour-flow amplitudes of one event from the PRODUCTION kernel: complex array [nhel, ncolor, 2 (theta_old, theta_new)]."""
    _torch()
    npar, nc, nh = trex_npar(subproc_id), trex_ncolor(subproc_id), trex_nhel(subproc_id)
    m = np.ascontiguousarray(momenta_one, dtype=np.float64).reshape(npar, 4)
    to, pto = _theta(theta_old)
    tn, ptn = _theta(theta_new)
    out = np.empty((nh, nc, 2, 2))
    _check(lib().trex_debug_xtile(subproc_id, m.ctypes.data_as(_dp), pto, ptn, out.ctypes.data_as(_dp)), "trex_debug_xtile")
    return out[..., 0] + 1j * out[..., 1]
