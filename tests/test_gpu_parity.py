"""Parity of the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs (-m gpu).

Tolerances (BASELINE.json north_star): bucketing / permutations bit-exact; per-event |M|^2 and weight ratios within a
relative 1e-11 in fp64; fp32 / mixed modes median 5e-5, maximum 1e-3."""
import numpy as np
import pytest

from oracle import oracle as O
from trex_inputs import make_config, default_theta, SUBPROCESSES, REX_NPOS, TH_CTG, TH_GAMMAT, TH_ALPHA_S, shuffled_legs

pytestmark = pytest.mark.gpu

RTOL64 = 1e-11


@pytest.fixture(scope="module")
def T():
    import torch
    assert torch.cuda.is_available()
    import paper_2510_05100_b200 as T
    T.lib()                                   # raises if the CUDA library is not built: no fallback
    T.trex_set_stream(None)
    T.trex_set_precision(0)
    return T


def dev(a):
    import torch
    a = np.ascontiguousarray(a)
    if a.dtype == np.uint64:
        a = a.view(np.int64)
    return torch.from_numpy(a).cuda()


def rel(a, b):
    return np.abs(a - b) / np.abs(b)


def gpu_reweight(T, sid, mom, tho, thn, w):
    wo, mo, mn = T.trex_reweight(sid, dev(mom), tho, thn, dev(w))
    import torch
    torch.cuda.synchronize()
    return wo.cpu().numpy(), mo.cpu().numpy(), mn.cpu().numpy()


# ---------------------------------------------------------------- bucketing (bit-exact)
def _check_bucket(T, keys):
    perm, offsets, bkeys = T.rex_bucket(dev(keys))
    rperm, roff, rkeys = O.bucket(keys)
    assert np.array_equal(offsets, roff)
    assert np.array_equal(bkeys, rkeys)
    assert np.array_equal(perm.cpu().numpy(), rperm)


@pytest.mark.parametrize("n", [1, 2, 31, 32, 33, 1000, 1024, 1025, 40000, 300001])
def test_bucket_random_keys_bit_exact(T, n):
    rng = np.random.default_rng(n)
    pool = np.array([int(sp.key) for sp in SUBPROCESSES] + [int(REX_NPOS), 12345, 2**63 + 17], dtype=np.uint64)
    p = rng.random(len(pool)) ** 3
    keys = pool[rng.choice(len(pool), size=n, p=p / p.sum())]
    _check_bucket(T, keys)


def test_bucket_edge_cases(T):
    _check_bucket(T, np.full(5000, REX_NPOS, dtype=np.uint64))                 # only the "no class" bucket
    _check_bucket(T, np.full(70000, 7, dtype=np.uint64))                       # one class
    rng = np.random.default_rng(3)
    keys = rng.integers(1, 2**62, size=256, dtype=np.uint64)                   # REX_MAX_BUCKETS distinct keys
    _check_bucket(T, keys[rng.integers(0, 256, size=100000)])
    keys65 = rng.integers(1, 2**62, size=65, dtype=np.uint64)                  # the paper's QCD sample: 65 classes,
    p = 1.0 / np.arange(1, 66) ** 2                                            # very uneven
    _check_bucket(T, keys65[rng.choice(65, size=200000, p=p / p.sum())])
    perm, offsets, bkeys = T.rex_bucket(dev(np.zeros(0, dtype=np.uint64)))     # empty input
    assert perm.numel() == 0 and list(offsets) == [0] and len(bkeys) == 0
    with pytest.raises(T.TrexError):                                           # 257 distinct keys
        T.rex_bucket(dev(np.arange(1, 258, dtype=np.uint64)))


def test_bucket_cfg3_full_size_and_transposition(T):
    import torch
    w = make_config(3)
    perm, offsets, bkeys = T.rex_bucket(dev(w.keys))
    rperm, roff, rkeys = O.bucket(w.keys)
    assert np.array_equal(offsets, roff) and np.array_equal(bkeys, rkeys)
    assert np.array_equal(perm.cpu().numpy(), rperm)
    mom = dev(w.momenta)
    g = T.rex_gather(mom, perm)
    assert np.array_equal(g.cpu().numpy(), O.gather(w.momenta, rperm))
    back = torch.zeros_like(mom)
    T.rex_scatter(g, perm, back)
    assert torch.equal(back, mom)
    # a bucket-local gather (perm + offsets[b]) gives that bucket's SoA block
    b = 2
    sub = perm[int(offsets[b]):int(offsets[b + 1])].contiguous()
    blk = T.rex_gather(mom, sub)
    assert np.array_equal(blk.cpu().numpy(), w.momenta[:, :, rperm[roff[b]:roff[b + 1]]])


# ---------------------------------------------------------------- |M|^2 and weights, element by element
# (sid, config, events): several 32-event tiles and a ragged tail, sized so the oracle finishes in seconds
CASES = [(0, 1, 4096), (1, 2, 4133), (2, 3, 677), (3, 4, 101), (4, 5, 37)]


@pytest.mark.parametrize("sid,cfg,nev", CASES)
def test_reweight_matches_oracle(T, sid, cfg, nev):
    w = make_config(cfg, n=max(nev, 64))
    mom = np.ascontiguousarray(w.momenta[:, :, :nev])
    win = w.w_in[:nev]
    wo, mo, mn = gpu_reweight(T, sid, mom, w.theta_old, w.theta_new, win)
    rw, ro, rn = O.reweight(sid, mom, w.theta_old, w.theta_new, win)
    assert rel(mo, ro).max() < RTOL64 and rel(mn, rn).max() < RTOL64, (rel(mo, ro).max(), rel(mn, rn).max())
    assert rel(wo, rw).max() < RTOL64
    assert np.all(wo != win)                       # the reweighting really changed something


@pytest.mark.parametrize("sid,cfg,nev,algo", [(2, 3, 333, 3), (2, 3, 333, 0), (2, 3, 333, 4), (3, 4, 67, 0), (4, 5, 9, 0), (3, 4, 67, 4), (1, 2, 555, 0)])
def test_both_evaluation_strategies_match_oracle(T, sid, cfg, nev, algo):
    """trex_set_algorithm: the fused current-table kernel and the one-thread-per-helicity-unit walk are both oracle-exact."""
    w = make_config(cfg, n=max(nev, 64))
    mom = np.ascontiguousarray(w.momenta[:, :, :nev])
    win = w.w_in[:nev]
    T.trex_set_algorithm(algo)
    try:
        wo, mo, mn = gpu_reweight(T, sid, mom, w.theta_old, w.theta_new, win)
    finally:
        T.trex_set_algorithm(3)
    rw, ro, rn = O.reweight(sid, mom, w.theta_old, w.theta_new, win)
    assert rel(mo, ro).max() < RTOL64 and rel(mn, rn).max() < RTOL64 and rel(wo, rw).max() < RTOL64


@pytest.mark.parametrize("sid,cfg,nev", [(1, 2, 300), (2, 3, 70), (4, 5, 5), (5, 3, 20)])
def test_top_width_and_mass_change_two_pass_kernels(T, sid, cfg, nev):
    """theta_new with another top width / mass: the top line is carried once per parameter point (NPASS = 2 kernels)."""
    w = make_config(cfg, n=4096)
    sel = np.where(w.keys == SUBPROCESSES[sid].key)[0][:nev]
    mom = np.ascontiguousarray(w.momenta[:, :, sel])
    tho, thn = w.theta_old.copy(), w.theta_new.copy()
    tho[6], thn[6] = 1.5, 1.2                      # Gamma_t
    if sid == 1:
        thn[5] = 171.5                             # m_t enters the propagators only through theta: externals keep their momenta
    wo, mo, mn = gpu_reweight(T, sid, mom, tho, thn, w.w_in[sel])
    rw, ro, rn = O.reweight(sid, mom, tho, thn, w.w_in[sel])
    assert rel(mo, ro).max() < RTOL64 and rel(mn, rn).max() < RTOL64 and rel(wo, rw).max() < RTOL64


@pytest.mark.parametrize("sid", [5, 6, 7, 8])
def test_quark_channels_match_explicit_colour_oracle(T, sid):
    w = make_config(3, n=2048)
    sel = np.where(w.keys == SUBPROCESSES[sid].key)[0][:37]
    mom = np.ascontiguousarray(w.momenta[:, :, sel])
    wo, mo, mn = gpu_reweight(T, sid, mom, w.theta_old, w.theta_new, w.w_in[sel])
    rw, ro, rn = O.reweight(sid, mom, w.theta_old, w.theta_new, w.w_in[sel])
    assert rel(mo, ro).max() < RTOL64 and rel(mn, rn).max() < RTOL64 and rel(wo, rw).max() < RTOL64


@pytest.mark.parametrize("sid,cfg", [(1, 2), (2, 3), (3, 4)])
def test_colour_flow_amplitudes_match_oracle(T, sid, cfg):
    """every J_c of every helicity, both orders in kappa (finer than |M|^2)."""
    w = make_config(cfg, n=64)
    th = w.theta_old
    for e in (0, 5):
        mom1 = np.ascontiguousarray(w.momenta[:, :, e:e + 1])
        got = T.trex_debug_flow_amps(sid, mom1[:, :, 0], th)
        scale = np.abs(got).max(axis=(0, 1))
        for h in range(T.trex_nhel(sid)):
            ref = O.ttng_amps(sid, mom1, th, h)
            assert np.all(np.abs(got[h] - ref) <= 1e-12 * scale), h


def test_debug_flow_amps_five_gluons_one_helicity(T):
    w = make_config(5, n=64)
    mom1 = np.ascontiguousarray(w.momenta[:, :, 3:4])
    got = T.trex_debug_flow_amps(4, mom1[:, :, 0], w.theta_old)
    scale = np.abs(got).max(axis=(0, 1))
    for h in (0, 77, 127):
        ref = O.ttng_amps(4, mom1, w.theta_old, h)
        assert np.all(np.abs(got[h] - ref) <= 1e-12 * scale)


@pytest.mark.parametrize("sid,cfg,hels", [(1, 2, None), (2, 3, None), (3, 4, None), (4, 5, (0, 37, 77, 90, 127))])
def test_production_kernels_colour_flow_amplitudes_match_oracle(T, sid, cfg, hels):
    """SURVEY.md I-4 on the kernels trex_reweight launches and bench.py times (k_gg_tt, k_table<3>, k_table4w,
    k_table<5>): the operand of their colour sum, every flow J_c at theta_old and theta_new, against the oracle's
    colour-ordered amplitudes J0 + kappa J1 -- finer than the helicity- and colour-summed |M|^2."""
    w = make_config(cfg, n=64)
    tho, thn = w.theta_old, w.theta_new
    for e in (0, 9):
        mom1 = np.ascontiguousarray(w.momenta[:, :, e:e + 1])
        got = T.trex_debug_xtile(sid, mom1[:, :, 0], tho, thn)
        assert np.all(np.isfinite(got)) and np.abs(got).max() > 0
        scale = np.abs(got).max(axis=(0, 1))
        for h in (range(T.trex_nhel(sid)) if hels is None else hels):
            for k, th in enumerate((tho, thn)):
                ref = O.ttng_amps(sid, mom1, th, h)
                want = ref[:, 0] + O.kappa(th) * ref[:, 1]
                assert np.all(np.abs(got[h, :, k] - want) <= 1e-12 * scale[k]), (e, h, k)


# ---------------------------------------------------------------- properties that hold at any size / edge cases
def test_unit_ratio_zero_guard_and_empty(T):
    import torch
    w = make_config(2, n=1000)
    wo, mo, mn = gpu_reweight(T, 1, w.momenta, w.theta_old, w.theta_old, w.w_in)
    assert np.array_equal(mo, mn) and np.allclose(wo, w.w_in, rtol=4e-16, atol=0)
    th0 = w.theta_old.copy()
    th0[TH_ALPHA_S] = 0.0                                  # me2_old == 0 exactly -> weight 0
    wo, mo, mn = gpu_reweight(T, 1, w.momenta, th0, w.theta_new, w.w_in)
    assert np.all(mo == 0) and np.all(wo == 0) and np.all(mn > 0)
    e = torch.empty(0, dtype=torch.float64, device="cuda")
    out = T.trex_reweight(1, torch.empty((4, 4, 0), dtype=torch.float64, device="cuda"), w.theta_old, w.theta_new, e)
    assert out[0].numel() == 0
    with pytest.raises(T.TrexError):
        T.trex_reweight(42, dev(w.momenta), w.theta_old, w.theta_new, dev(w.w_in))
    bad = w.theta_old.copy()
    bad[TH_ALPHA_S] = -1.0
    with pytest.raises(T.TrexError):
        T.trex_reweight(1, dev(w.momenta), bad, w.theta_new, dev(w.w_in))


def test_me2_exactly_quadratic_in_ctg_on_gpu(T):
    w = make_config(4, n=96)
    cs = np.array([0.0, 0.7, 1.9, -2.6, 4.0])
    vals = []
    for c in cs:
        th = default_theta()
        th[TH_CTG] = c
        vals.append(gpu_reweight(T, 3, w.momenta, default_theta(), th, w.w_in)[2])
    vals = np.array(vals)
    for e in range(vals.shape[1]):
        coef = np.polyfit(cs, vals[:, e], 4)
        assert abs(coef[0]) < 1e-10 * abs(vals[0, e]) and abs(coef[1]) < 1e-10 * abs(vals[0, e])


FULL = [(1, 0, 64), (2, 1, 64), (4, 3, 24), (5, 4, 6)]


@pytest.mark.parametrize("cfg,sid,nsample", FULL)
def test_full_size_configs_sampled_against_oracle(T, cfg, sid, nsample):
    """BASELINE.json's full sizes in the launch configuration bench.py times (trex_run on the whole sample)."""
    import torch
    w = make_config(cfg)
    wo, mo, mn, nb = T.trex_run(dev(w.keys), dev(w.momenta), w.theta_old, w.theta_new, dev(w.w_in))
    torch.cuda.synchronize()
    wo, mo, mn = wo.cpu().numpy(), mo.cpu().numpy(), mn.cpu().numpy()
    assert nb == 1 and np.all(np.isfinite(wo)) and np.all(mo > 0) and np.all(mn > 0)
    rng = np.random.default_rng(100 + cfg)
    idx = np.sort(rng.choice(w.n, size=nsample, replace=False))
    idx[-1] = w.n - 1                                                        # the ragged end of the last tile
    mom = np.ascontiguousarray(w.momenta[:, :, idx])
    rw, ro, rn = O.reweight(sid, mom, w.theta_old, w.theta_new, w.w_in[idx])
    assert rel(mo[idx], ro).max() < RTOL64 and rel(mn[idx], rn).max() < RTOL64 and rel(wo[idx], rw).max() < RTOL64


def test_cfg3_full_path_bucket_gather_reweight_scatter(T):
    import torch
    w = make_config(3)
    wo, mo, mn, nb = T.trex_run(dev(w.keys), dev(w.momenta), w.theta_old, w.theta_new, dev(w.w_in))
    torch.cuda.synchronize()
    wo, mo, mn = wo.cpu().numpy(), mo.cpu().numpy(), mn.cpu().numpy()
    assert nb == 5 and np.all(np.isfinite(wo)) and np.all(mo > 0)
    rng = np.random.default_rng(33)
    for sp in w.classes:
        cand = np.where(w.keys == sp.key)[0]
        idx = np.sort(rng.choice(cand, size=24 if sp.sid == 2 else 6, replace=False))
        mom = np.ascontiguousarray(w.momenta[:, :, idx])
        rw, ro, rn = O.reweight(sp.sid, mom, w.theta_old, w.theta_new, w.w_in[idx])
        assert rel(mo[idx], ro).max() < RTOL64 and rel(mn[idx], rn).max() < RTOL64 and rel(wo[idx], rw).max() < RTOL64, sp.name


def test_unknown_classes_get_zero_weights(T):
    """events no procReweightor claims are given zero weights."""
    import torch
    w = make_config(3, n=5000)
    keys = w.keys.copy()
    keys[::7] = np.uint64(REX_NPOS)
    keys[3::11] = np.uint64(424242)
    wo, mo, mn, nb = T.trex_run(dev(keys), dev(w.momenta), w.theta_old, w.theta_new, dev(w.w_in))
    torch.cuda.synchronize()
    wo = wo.cpu().numpy()
    unknown = (keys == np.uint64(REX_NPOS)) | (keys == np.uint64(424242))
    assert nb == 7 and np.all(wo[unknown] == 0) and np.all(mo.cpu().numpy()[unknown] == 0) and np.all(wo[~unknown] > 0)
    ref, _, _, _ = T.trex_run(dev(w.keys), dev(w.momenta), w.theta_old, w.theta_new, dev(w.w_in))
    assert np.array_equal(ref.cpu().numpy()[~unknown], wo[~unknown])


def test_host_buffer_entry_point_matches_device_path(T):
    import torch
    w = make_config(3, n=20000)
    ref, _, _, _ = T.trex_run(dev(w.keys), dev(w.momenta), w.theta_old, w.theta_new, dev(w.w_in))
    out = np.empty(w.n)
    mo = np.empty(w.n)
    nb = T.trex_run_host(w.keys, w.momenta, w.theta_old, w.theta_new, w.w_in, out, mo, None)
    assert nb == 5 and np.array_equal(out, ref.cpu().numpy()) and np.all(mo > 0)


# ---------------------------------------------------------------- reduced-precision modes (PAPER.md:1209 fptype m / f)
@pytest.mark.parametrize("mode", [1, 2])
def test_reduced_precision_modes_cfg4(T, mode):
    w = make_config(4, n=4096)
    ref_w, ref_o, ref_n = gpu_reweight(T, 3, w.momenta, w.theta_old, w.theta_new, w.w_in)
    T.trex_set_precision(mode)
    try:
        assert T.trex_get_precision() == mode
        wo, mo, mn = gpu_reweight(T, 3, w.momenta, w.theta_old, w.theta_new, w.w_in)
    finally:
        T.trex_set_precision(0)
    for got, ref in ((wo, ref_w), (mo, ref_o), (mn, ref_n)):
        r = rel(got, ref)
        assert np.median(r) < 5e-5 and r.max() < 1e-3, (mode, np.median(r), r.max())
    # and the fp64 reference itself is oracle-checked on a sample
    idx = np.arange(0, 4096, 512)
    rw, ro, rn = O.reweight(3, np.ascontiguousarray(w.momenta[:, :, idx]), w.theta_old, w.theta_new, w.w_in[idx])
    assert rel(ref_o[idx], ro).max() < RTOL64 and rel(ref_w[idx], rw).max() < RTOL64


# ---------------------------------------------------------------- reweighted cross section
@pytest.mark.parametrize("n", [1, 255, 100017])
def test_xsec_moments_match_oracle(T, n):
    import torch
    rng = np.random.default_rng(n)
    w = rng.lognormal(0, 0.5, n)
    w[5::17] = 0.0
    wo = w * rng.uniform(0.5, 2.0, n)
    dw, dwo = dev(w), dev(wo)
    m1 = T.trex_xsec_moments(dw, dwo)
    m2 = T.trex_xsec_moments(dw, dwo)
    assert np.array_equal(m1, m2)                               # fixed summation order
    got = T.trex_xsec_finish(m1, 0.01, 3.0, 0.25)
    ref = O.xsec(w, wo, 0.01, 3.0, 0.25)
    assert abs(got[0] / ref[0] - 1) < 1e-12 and abs(got[1] / ref[1] - 1) < 1e-11 and got[2] == ref[2]
    # three shards reduced separately and combined
    cut = [0, n // 3, n // 3, n]
    parts = [T.trex_xsec_moments(dev(w[a:b]), dev(wo[a:b])) if b > a else np.zeros(4) for a, b in zip(cut[:-1], cut[1:])]
    got3 = T.trex_xsec_finish(parts, 0.01, 3.0, 0.25)
    assert abs(got3[0] / ref[0] - 1) < 1e-12 and abs(got3[1] / ref[1] - 1) < 1e-11


def test_xsec_of_a_reweighted_full_sample(T):
    """cfg3 at full size: weights straight from trex_run (zero weights for unknown classes included)."""
    import torch
    w = make_config(3)
    keys = w.keys.copy()
    keys[::1001] = np.uint64(424242)
    win = dev(w.w_in)
    wo, _, _, nb = T.trex_run(dev(keys), dev(w.momenta), w.theta_old, w.theta_new, win)
    got = T.trex_xsec_finish(T.trex_xsec_moments(win, wo), 1e-3, 40.0, 0.4)
    ref = O.xsec(w.w_in, wo.cpu().numpy(), 1e-3, 40.0, 0.4)
    assert nb == 6 and abs(got[0] / ref[0] - 1) < 1e-12 and abs(got[1] / ref[1] - 1) < 1e-11 and not got[2]


# ---------------------------------------------------------------- many parameter points on one categorisation (NEXT-1)
@pytest.mark.parametrize("cfg,n", [(3, 30011), (2, 5000)])
def test_run_multi_equals_one_run_per_parameter_point(T, cfg, n):
    """PAPER.md:1306-1310 "sort once": K parameter points after ONE rex_bucket + transposition; every row must equal
    the single-point path bit for bit, and the oracle on a sample."""
    import torch
    w = make_config(cfg, n=n)
    keys = w.keys.copy()
    if cfg == 3:
        keys[::97] = np.uint64(REX_NPOS)
    thetas = []
    for ctg, gt in ((0.25, 0.0), (1.0, 0.0), (-0.7, 1.4)):
        th = w.theta_new.copy(); th[TH_CTG] = ctg; th[TH_GAMMAT] = gt
        thetas.append(th)
    dk, dm, dw = dev(keys), dev(w.momenta), dev(w.w_in)
    wo, mo, mn, nb = T.trex_run_multi(dk, dm, w.theta_old, thetas, dw)
    torch.cuda.synchronize()
    for k, th in enumerate(thetas):
        w1, mo1, mn1, nb1 = T.trex_run(dk, dm, w.theta_old, th, dw)
        assert nb1 == nb and torch.equal(w1, wo[k]) and torch.equal(mn1, mn[k])
        # |M(theta_old)|^2 is written once (k = 0); another k may run a different kernel variant (two top-line passes)
        a1, a0 = mo1.cpu().numpy(), mo.cpu().numpy()
        nz = a0 != 0
        assert np.array_equal(a1 == 0, a0 == 0) and rel(a1[nz], a0[nz]).max() < 1e-13
    # oracle on a few events of the largest class
    sp = w.classes[0]
    idx = np.where(keys == sp.key)[0][:12]
    mom = np.ascontiguousarray(w.momenta[:, :, idx])
    for k, th in enumerate(thetas):
        rw, ro, rn = O.reweight(sp.sid, mom, w.theta_old, th, w.w_in[idx])
        assert rel(wo[k].cpu().numpy()[idx], rw).max() < RTOL64 and rel(mn[k].cpu().numpy()[idx], rn).max() < RTOL64


@pytest.mark.parametrize("cfg,n", [(3, 20011), (2, 9001), (4, 300)])
def test_run_multi_polynomial_path(T, cfg, n):
    """Parameter points that differ in kappa only: three evaluations + the exact quadratic (R-4) against the
    direct path and the oracle."""
    import torch
    w = make_config(cfg, n=n)
    keys = w.keys.copy()
    if cfg == 3:
        keys[::97] = np.uint64(REX_NPOS)
    tho = w.theta_old.copy()
    if cfg == 4:
        tho[TH_GAMMAT] = 1.5
    tho[TH_CTG] = 0.2
    thetas = []
    for ctg in (-1.0, -0.3, 0.0, 0.2, 0.45, 2.0):
        th = tho.copy(); th[TH_CTG] = ctg
        thetas.append(th)
    thetas[1][8] = 1200.0                                    # another Lambda: still only kappa moves
    dk, dm, dw = dev(keys), dev(w.momenta), dev(w.w_in)
    wp, mop, mnp, nb = T.trex_run_multi(dk, dm, tho, thetas, dw)
    T.trex_set_poly_multi(False)
    try:
        wd, mod, mnd, nbd = T.trex_run_multi(dk, dm, tho, thetas, dw)
    finally:
        T.trex_set_poly_multi(True)
    torch.cuda.synchronize()
    assert nb == nbd
    a, b = wp.cpu().numpy(), wd.cpu().numpy()
    nz = b != 0
    assert np.array_equal(a == 0, b == 0) and rel(a[nz], b[nz]).max() < 1e-12
    a, b = mnp.cpu().numpy(), mnd.cpu().numpy()
    assert rel(a[nz], b[nz]).max() < 1e-12 and torch.equal(mop, mod)
    assert not np.allclose(wp[0].cpu().numpy()[nz[0]], wp[5].cpu().numpy()[nz[0]])     # the rows really differ
    sp = w.classes[0]
    idx = np.where(keys == sp.key)[0][:6]
    mom = np.ascontiguousarray(w.momenta[:, :, idx])
    for k in (0, 1, 5):
        rw, ro, rn = O.reweight(sp.sid, mom, tho, thetas[k], w.w_in[idx])
        assert rel(wp[k].cpu().numpy()[idx], rw).max() < RTOL64 and rel(mnp[k].cpu().numpy()[idx], rn).max() < RTOL64


# ---------------------------------------------------------------- PDG codes in arbitrary parton order (NEXT-3)
def test_rex_keys_and_legmap_bit_exact(T):
    import torch
    w = make_config(3, n=30017)
    pdg, mom, n_in = shuffled_legs(w, 9, unknown_every=41)
    pdg[2, 5] = 1000022                                                  # a code the key cannot hold -> REX_NPOS
    keys, lm = T.rex_keys(torch.from_numpy(pdg).cuda(), n_in)
    rk, rl = O.keys_and_legmap(pdg, n_in, [sp.pdg for sp in SUBPROCESSES])
    assert np.array_equal(keys.cpu().numpy().view(np.uint64), rk) and np.array_equal(lm.cpu().numpy(), rl)
    assert rk[5] == np.uint64(REX_NPOS)


@pytest.mark.parametrize("cfg,n", [(3, 20011), (4, 700), (2, 3000)])
def test_run_pdg_reindexes_partons(T, cfg, n):
    """events whose partons come in another order than the process string are re-indexed inside the
    transposition; weights equal the oracle's on the re-indexed momenta, unknown classes get zero."""
    import torch
    w = make_config(cfg, n=n)
    pdg, mom, n_in = shuffled_legs(w, 100 + cfg, unknown_every=53)
    wo, mo, mn, nb = T.trex_run_pdg(torch.from_numpy(pdg).cuda(), dev(mom), n_in, w.theta_old, w.theta_new, dev(w.w_in))
    torch.cuda.synchronize()
    wo, mo, mn = wo.cpu().numpy(), mo.cpu().numpy(), mn.cpu().numpy()
    rk, rl = O.keys_and_legmap(pdg, n_in, [sp.pdg for sp in SUBPROCESSES])
    unknown = np.ones(w.n, dtype=bool)
    for sp in w.classes:
        sel = np.where(rk == sp.key)[0]
        unknown[sel] = False
        idx = sel[:: max(1, len(sel) // 8)][:8]
        canon = np.ascontiguousarray(mom[rl[:, idx], :, idx].transpose(0, 2, 1))
        rw, ro, rn = O.reweight(sp.sid, canon, w.theta_old, w.theta_new, w.w_in[idx])
        assert rel(wo[idx], rw).max() < RTOL64 and rel(mo[idx], ro).max() < RTOL64 and rel(mn[idx], rn).max() < RTOL64, sp.name
    assert unknown.sum() > 0 and np.all(wo[unknown] == 0) and np.all(mo[unknown] == 0) and np.all(wo[~unknown] > 0)
    assert nb == len(np.unique(rk))
    # against the canonical sample through trex_run: the same physics, identical up to the order of identical gluons
    w0, _, _, _ = T.trex_run(dev(w.keys), dev(w.momenta), w.theta_old, w.theta_new, dev(w.w_in))
    w0 = w0.cpu().numpy()
    assert rel(wo[~unknown], w0[~unknown]).max() < 1e-12


@pytest.mark.parametrize("n", [1, 2, 31, 33, 100, 8191, 8192, 8193, 70001])
def test_run_sizes_around_every_threshold(T, n):
    """trex_run against one trex_reweight per class on the gathered block: sizes around the warp, the single-block
    bucketing (8192) and the graph-replay thresholds; the second identical call replays the captured graph."""
    import torch
    w = make_config(3, n=max(n, 64))
    keys, mom, win = w.keys[:n].copy(), np.ascontiguousarray(w.momenta[:, :, :n]), w.w_in[:n]
    if n > 40:
        keys[7::29] = np.uint64(REX_NPOS)
    dk, dm, dw = dev(keys), dev(mom), dev(win)
    outs = [T.trex_run(dk, dm, w.theta_old, w.theta_new, dw) for _ in range(3)]
    torch.cuda.synchronize()
    wo, mo, mn, nb = outs[0]
    for o in outs[1:]:
        assert torch.equal(o[0], wo) and torch.equal(o[2], mn) and o[3] == nb
    wo = wo.cpu().numpy()
    ref = np.zeros(n)
    for sp in w.classes:
        sel = np.where(keys == sp.key)[0]
        if len(sel):
            r, _, _ = gpu_reweight(T, sp.sid, np.ascontiguousarray(mom[:, :, sel]), w.theta_old, w.theta_new, win[sel])
            ref[sel] = r
    assert np.array_equal(wo, ref)


@pytest.mark.parametrize("n", [3000, 40000])
def test_run_with_too_many_classes_fails_loudly(T, n):
    """More than REX_MAX_BUCKETS distinct flavour keys: rex_bucket and trex_run report the error (both bucketing paths:
    one block for small samples, six launches otherwise); the library stays usable afterwards."""
    import torch
    w = make_config(2, n=n)
    keys = w.keys.copy()
    keys[: T.REX_MAX_BUCKETS + 5] = np.arange(1, T.REX_MAX_BUCKETS + 6, dtype=np.uint64) * np.uint64(1000003)
    with pytest.raises(T.TrexError):
        T.rex_bucket(dev(keys))
    with pytest.raises(T.TrexError):
        T.trex_run(dev(keys), dev(w.momenta), w.theta_old, w.theta_new, dev(w.w_in))
    wo, mo, mn, nb = T.trex_run(dev(w.keys), dev(w.momenta), w.theta_old, w.theta_new, dev(w.w_in))
    assert nb == 1 and bool((wo > 0).all())


@pytest.mark.parametrize("cfg,n", [(1, 4096), (2, 20000), (3, 20000), (5, 512)])
@pytest.mark.parametrize("mode", [1, 2])
def test_reduced_precision_modes_every_config(T, cfg, n, mode):
    """fptype m / f through the whole path on every configuration: median 5e-5 / maximum 1e-3 against
    the fp64 path (north star); kinematic invariants stay in fp64 in every mode (R-12)."""
    import torch
    w = make_config(cfg, n=n)
    k, m, wi = dev(w.keys), dev(w.momenta), dev(w.w_in)
    ref = [x.cpu().numpy() for x in T.trex_run(k, m, w.theta_old, w.theta_new, wi)[:3]]
    T.trex_set_precision(mode)
    try:
        got = [x.cpu().numpy() for x in T.trex_run(k, m, w.theta_old, w.theta_new, wi)[:3]]
    finally:
        T.trex_set_precision(0)
    for g, r0 in zip(got, ref):
        r = rel(g, r0)
        assert np.median(r) < 5e-5 and r.max() < 1e-3, (cfg, mode, np.median(r), r.max())


# ---------------------------------------------------------------- adversarial kinematics, long double oracle as adjudicator
def _event(sqrt_s, finals, th_star, phi_star, mt=173.0):
    """2 -> t t~ + massless partons with the partons' momenta GIVEN (list of (E, theta, phi)): the t t~ pair recoils
    against them and decays with angles (th_star, phi_star) in its rest frame. Test-side construction only."""
    ps = []
    for E, th, ph in finals:
        ps.append(np.array([E, E * np.sin(th) * np.cos(ph), E * np.sin(th) * np.sin(ph), E * np.cos(th)]))
    tot = np.array([sqrt_s, 0.0, 0.0, 0.0]) - sum(ps, np.zeros(4))
    M = np.sqrt(tot[0] ** 2 - tot[1:] @ tot[1:])
    assert M > 2 * mt
    pstar = np.sqrt(M * M / 4 - mt * mt)
    d = np.array([np.sin(th_star) * np.cos(phi_star), np.sin(th_star) * np.sin(phi_star), np.cos(th_star)])
    out = []
    beta = tot[1:] / tot[0]
    g = tot[0] / M
    for sgn in (1.0, -1.0):
        k = sgn * pstar * d
        e = M / 2
        bk = beta @ k
        b2 = beta @ beta
        kk = k + ((g - 1.0) * bk / b2 + g * e) * beta if b2 > 0 else k
        out.append(np.concatenate([[g * (e + bk)], kk]))
    mom = [np.array([sqrt_s / 2, 0, 0, sqrt_s / 2]), np.array([sqrt_s / 2, 0, 0, -sqrt_s / 2])] + out + ps
    return np.ascontiguousarray(np.array(mom)[:, :, None])


ADVERSARIAL = [
    # (sid, label, sqrt_s, partons (E, theta, phi), th*, phi*)
    (1, "tops along the beam", 500.0, [], 0.0, 0.0),
    (1, "tops nearly along the beam", 500.0, [], 1e-9, 0.3),
    (1, "tops at threshold", 2 * 173.0 * (1 + 1e-9), [], 0.7, 1.1),
    # (a massless final-state parton EXACTLY on the beam axis sits on the collinear pole 1 / (2 k_in . k_out) = 1 / 0 of
    # the amplitude itself: there is no finite value to compare; the cases below approach it)
    (2, "gluon 1e-3 from +z", 900.0, [(120.0, 1e-3, 0.0)], 0.8, 0.4),
    (2, "gluon 1e-3 from -z", 900.0, [(120.0, np.pi - 1e-3, 2.0)], 0.8, 0.4),
    (2, "gluon 1e-5 from +z", 900.0, [(120.0, 1e-5, 2.0)], 0.8, 0.4),
    (2, "soft gluon", 900.0, [(0.09, 1.1, 0.2)], 1.3, 2.4),
    (2, "gluon collinear to the beam", 900.0, [(200.0, 1e-4, 1.0)], 1.3, 2.4),
    (2, "t t~ pair at threshold", 900.0, [((900.0 ** 2 - (2 * 173.0 * (1 + 1e-8)) ** 2) / (2 * 900.0), 0.9, 0.1)], 0.5, 0.6),
    (3, "one gluon 1e-3 from -z, one soft", 1500.0, [(300.0, np.pi - 1e-3, 0.0), (0.15, 0.7, 1.9)], 1.0, 0.2),
    (3, "collinear gluon pair", 1500.0, [(250.0, 1.0, 0.5), (180.0, 1.0 + 1e-4, 0.5)], 1.0, 0.2),
    (4, "one gluon 1e-3 from +z, collinear pair", 2000.0, [(200.0, 1e-3, 0.0), (250.0, 2.0, 0.5), (100.0, 2.0 + 1e-4, 0.5)], 1.0, 0.2),
    (5, "q q~: gluon 1e-3 from +z", 900.0, [(120.0, 1e-3, 0.0)], 0.8, 0.4),
    (7, "q g: final quark 1e-3 from -z", 900.0, [(120.0, np.pi - 1e-3, 0.0)], 0.8, 0.4),
    (8, "g q~: soft final antiquark", 900.0, [(0.09, 1.1, 0.2)], 0.8, 0.4),
]


@pytest.mark.parametrize("sid,label,sqrt_s,partons,ths,phs", ADVERSARIAL, ids=[a[1] for a in ADVERSARIAL])
def test_adversarial_kinematics_against_long_double_oracle(T, sid, label, sqrt_s, partons, ths, phs):
    """Degenerate phase-space corners (SURVEY P-13): tops on the beam axis (the pT -> 0 branch of the two-spinors),
    final-state partons close to it, soft and collinear emissions, tops at threshold. The adjudicator is the
    oracle in long double; the bar is 1e-11 where the double-precision oracle itself reaches it, else ten times the
    oracle's own double-precision deviation (both sides then lose the same digits to the physical cancellation)."""
    mom = _event(sqrt_s, partons, ths, phs)
    tho, thn = default_theta(), default_theta()
    thn[TH_CTG] = 0.8
    if sid in (3, 4):
        tho[TH_GAMMAT], thn[TH_GAMMAT] = 1.5, 1.35
    w = np.array([1.7])
    got = gpu_reweight(T, sid, mom, tho, thn, w)
    ld = O.reweight(sid, mom, tho, thn, w, long_double=True)
    db = O.reweight(sid, mom, tho, thn, w)
    K = mom[:, :, 0].copy()
    K[2:] *= -1.0                                            # all-incoming convention
    light = [i for i in range(K.shape[0]) if i not in (2, 3)]
    cond = 1.0
    for i in light:
        for j in light:
            if i < j:
                P = K[i] + K[j]
                cond = max(cond, (abs(K[i, 0]) + abs(K[j, 0])) ** 2 / abs(P[0] ** 2 - P[1:] @ P[1:]))
    for k, (g, a, b) in enumerate(zip(got, ld, db)):
        assert np.all(np.isfinite(g)) and np.all(a > 0)
        bar = max(RTOL64, 10.0 * float(rel(b, a).max()), 4 * 2.2e-16 * cond)
        assert rel(g, a).max() < bar, (label, rel(g, a).max(), rel(b, a).max(), cond)
    # the weight ratio is well conditioned wherever |M|^2 itself is finite
    assert rel(got[0], ld[0]).max() < max(RTOL64, 10.0 * float(rel(db[0], ld[0]).max())), label


@pytest.mark.parametrize("cfg,n", [(1, 2048), (2, 4096), (3, 1536), (4, 96), (5, 12)])
@pytest.mark.parametrize("mode", [1, 2])
def test_reduced_precision_modes_against_the_oracle(T, cfg, n, mode):
    """fptype m / f on every configuration against the ORACLE (not against the library's own fp64 result): median 5e-5,
    maximum 1e-3 (north star)."""
    w = make_config(cfg, n=n)
    k, m, wi = dev(w.keys), dev(w.momenta), dev(w.w_in)
    T.trex_set_precision(mode)
    try:
        got = [x.cpu().numpy() for x in T.trex_run(k, m, w.theta_old, w.theta_new, wi)[:3]]
    finally:
        T.trex_set_precision(0)
    ref = [np.zeros(n), np.zeros(n), np.zeros(n)]
    for sp in w.classes:
        sel = np.where(w.keys == sp.key)[0]
        if sp.sid >= 5:
            sel = sel[:24]                                   # explicit-colour engine: a sample of the quark channels
        r = O.reweight(sp.sid, np.ascontiguousarray(w.momenta[:, :, sel]), w.theta_old, w.theta_new, w.w_in[sel])
        for a, b in zip(ref, r):
            a[sel] = b
    ok = ref[1] != 0
    for g, r0 in zip(got, ref):
        r = rel(g[ok], r0[ok])
        assert np.median(r) < 5e-5 and r.max() < 1e-3, (cfg, mode, np.median(r), r.max())


def test_status_filter_comparators_on_the_device(T):
    """NEXT-3 (Alg.1 :419-444): keys under comparators with a status filter, bit-exact against the
    oracle; under the final-state-only comparator g g > t t~ g and q q~ > t t~ g fall into one class, and rex_bucket
    orders the classes by first appearance as ever."""
    import torch
    w = make_config(3, n=20011)
    pdg, mom, n_in = shuffled_legs(w, 17, unknown_every=0)
    rng = np.random.default_rng(8)
    nl = w.npar + 1                                          # one intermediate parton (status 2) per event record
    pdg2 = np.vstack([pdg, rng.choice([23, 25, 6], size=(1, w.n)).astype(np.int32)])
    st = np.vstack([np.full((2, w.n), -1), np.ones((w.npar - 2, w.n)), np.full((1, w.n), 2)]).astype(np.int8)
    col = rng.permuted(np.tile(np.arange(nl)[:, None], (1, w.n)), axis=0)         # records in arbitrary parton order
    pdg2, st = np.take_along_axis(pdg2, col, 0), np.take_along_axis(st, col, 0)
    dp, ds = torch.from_numpy(np.ascontiguousarray(pdg2)).cuda(), torch.from_numpy(np.ascontiguousarray(st)).cuda()
    for filt in ((-1, 1), (1,), (), (1, 2)):
        keys = T.rex_keys_filtered(dp, ds, filt).cpu().numpy().view(np.uint64)
        ref = np.array([O.flavour_key_filtered(pdg2[:, i], st[:, i], status_filter=filt) for i in range(w.n)], dtype=np.uint64)
        assert np.array_equal(keys, ref), filt
        perm, offsets, bkeys = T.rex_bucket(dev(keys))
        rperm, roff, rkeys = O.bucket(ref)
        assert np.array_equal(perm.cpu().numpy(), rperm) and np.array_equal(offsets, roff) and np.array_equal(bkeys, rkeys)
    ext = T.rex_keys_filtered(dp, ds, (-1, 1)).cpu().numpy().view(np.uint64)
    fin = T.rex_keys_filtered(dp, ds, (1,)).cpu().numpy().view(np.uint64)
    assert np.array_equal(ext, w.keys)                       # the external-leg comparator is the default key
    assert len(np.unique(ext)) == 5 and len(np.unique(fin)) == 3          # t t~ g | t t~ u | t t~ u~
