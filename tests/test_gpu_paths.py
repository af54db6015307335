"""Host-visible behaviour of the CUDA path beyond plain parity (-m gpu): CUDA-graph replay, user streams, failure paths
that must not touch memory, and all-event cross-checks between the kernel families at bench-like sizes."""
import numpy as np
import pytest

from oracle import oracle as O
from trex_inputs import make_config, REX_NPOS

pytestmark = pytest.mark.gpu

RTOL64 = 1e-11


@pytest.fixture(scope="module")
def T():
    import torch
    assert torch.cuda.is_available()
    import paper_2510_05100_b200 as T
    T.lib()
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


@pytest.mark.parametrize("cfg,n", [(3, 30011), (2, 65536), (3, 5000)])
def test_graph_replay_is_taken_and_bit_equal(T, cfg, n):
    """trex_run with the SAME buffers, sizes and parameter points replays the captured CUDA graph (the configuration
    bench.py times): the replay must really be taken and give the bits of the plain launches."""
    import torch
    w = make_config(cfg, n=n)
    keys = w.keys.copy()
    if cfg == 3:
        keys[5::131] = np.uint64(REX_NPOS)
    dk, dm, dw = dev(keys), dev(w.momenta), dev(w.w_in)
    first = T.trex_run(dk, dm, w.theta_old, w.theta_new, dw)                    # fresh outputs: plain launches
    torch.cuda.synchronize()
    ref = [x.clone() for x in first[:3]]
    wo, mo, mn = (torch.full_like(dw, -1.0) for _ in range(3))
    r0 = T.trex_graph_replays()
    for it in range(4):
        wo.fill_(-1.0); mo.fill_(-1.0); mn.fill_(-1.0)
        _, _, _, nb = T.trex_run(dk, dm, w.theta_old, w.theta_new, dw, w_out=wo, me2_old=mo, me2_new=mn)
        torch.cuda.synchronize()
        assert nb == first[3]
        assert torch.equal(wo, ref[0]) and torch.equal(mo, ref[1]) and torch.equal(mn, ref[2]), it
    assert T.trex_graph_replays() - r0 >= 2                                      # call 2 captures + replays, 3 and 4 replay
    # a changed size or parameter point must not replay the stale graph
    r1 = T.trex_graph_replays()
    m = n - 17
    dk2, dm2, dw2 = dev(keys[:m]), dev(np.ascontiguousarray(w.momenta[:, :, :m])), dev(w.w_in[:m])
    out2 = T.trex_run(dk2, dm2, w.theta_old, w.theta_new, dw2)
    torch.cuda.synchronize()
    assert T.trex_graph_replays() == r1
    # (bucket order may differ for the prefix; compare per event)
    assert torch.equal(out2[0], ref[0][:m])
    th2 = w.theta_new.copy(); th2[7] = 0.77
    out3 = T.trex_run(dk, dm, w.theta_old, th2, dw, w_out=wo, me2_old=mo, me2_new=mn)
    torch.cuda.synchronize()
    assert T.trex_graph_replays() == r1 and not torch.equal(wo, ref[0])
    sp = w.classes[0]
    idx = np.where(keys == sp.key)[0][:5]
    rw, _, _ = O.reweight(sp.sid, np.ascontiguousarray(w.momenta[:, :, idx]), w.theta_old, th2, w.w_in[idx])
    assert rel(wo.cpu().numpy()[idx], rw).max() < RTOL64


def test_user_stream_including_graph_replay(T):
    """The library enqueues on the stream given to trex_set_stream; the graph is captured on a private stream and
    replayed on the user's."""
    import torch
    w = make_config(3, n=20000)
    dk, dm, dw = dev(w.keys), dev(w.momenta), dev(w.w_in)
    ref = T.trex_run(dk, dm, w.theta_old, w.theta_new, dw)
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    wo, mo, mn = (torch.empty_like(dw) for _ in range(3))
    T.trex_set_stream(s)
    try:
        r0 = T.trex_graph_replays()
        with torch.cuda.stream(s):
            for it in range(4):
                wo.fill_(-1.0)
                T.trex_run(dk, dm, w.theta_old, w.theta_new, dw, w_out=wo, me2_old=mo, me2_new=mn)
                s.synchronize()
                assert torch.equal(wo, ref[0]) and torch.equal(mn, ref[2]), it
            assert T.trex_graph_replays() - r0 >= 2
            # per-class call and the bucketing alone on the same stream
            sel = np.where(w.keys == w.classes[0].key)[0]
            o = T.trex_reweight(w.classes[0].sid, dev(np.ascontiguousarray(w.momenta[:, :, sel])), w.theta_old, w.theta_new,
                                dev(w.w_in[sel]))
            s.synchronize()
            assert np.array_equal(o[0].cpu().numpy(), ref[0].cpu().numpy()[sel])
            perm, offsets, _ = T.rex_bucket(dk)
            rperm, roff, _ = O.bucket(w.keys)
            assert np.array_equal(perm.cpu().numpy(), rperm) and np.array_equal(offsets, roff)
    finally:
        T.trex_set_stream(None)
    again = T.trex_run(dk, dm, w.theta_old, w.theta_new, dw)
    torch.cuda.synchronize()
    assert torch.equal(again[0], ref[0])


@pytest.mark.parametrize("n", [3000, 9000, 40000])
def test_too_many_classes_after_a_larger_run_touches_no_memory(T, n):
    """More than REX_MAX_BUCKETS keys: the categorisation fails on the device, so no permutation exists. The rest of the
    already enqueued chain (transposition, |M|^2 kernels, transposition back) must then do nothing -- in particular not
    gather / scatter through the stale permutation a larger earlier run left in the scratch buffer."""
    import torch
    big = make_config(3, n=120000)
    T.trex_run(dev(big.keys), dev(big.momenta), big.theta_old, big.theta_new, dev(big.w_in))    # leaves indices up to 119999
    torch.cuda.synchronize()
    w = make_config(3, n=n)
    keys = w.keys.copy()
    keys[: T.REX_MAX_BUCKETS + 5] = np.arange(1, T.REX_MAX_BUCKETS + 6, dtype=np.uint64) * np.uint64(1000003)
    pad = 4096
    buf = torch.full((3 * n + 4 * pad,), -7.0, dtype=torch.float64, device="cuda")      # canaries around and between
    wo = buf[pad:pad + n]
    mo = buf[2 * pad + n:2 * pad + 2 * n]
    mn = buf[3 * pad + 2 * n:3 * pad + 3 * n]
    dm, dw = dev(w.momenta), dev(w.w_in)
    with pytest.raises(T.TrexError):
        T.trex_run(dev(keys), dm, w.theta_old, w.theta_new, dw, w_out=wo, me2_old=mo, me2_new=mn)
    torch.cuda.synchronize()
    assert bool((buf == -7.0).all())
    th = np.tile(w.theta_new, (5, 1)); th[:, 7] = np.linspace(-1, 1, 5)
    buf2 = torch.full((5 * n + 2 * pad,), -7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(T.TrexError):
        T.trex_run_multi(dev(keys), dm, w.theta_old, th, dw, w_out=buf2[pad:pad + 5 * n].view(5, n), want_me2=False)
    torch.cuda.synchronize()
    assert bool((buf2[:pad] == -7.0).all()) and bool((buf2[pad + 5 * n:] == -7.0).all())
    # the library stays usable and correct
    out = T.trex_run(dev(w.keys), dm, w.theta_old, w.theta_new, dw)
    torch.cuda.synchronize()
    assert out[3] == 5 and bool((out[0] > 0).all())


def test_binding_rejects_mismatched_shapes(T):
    import torch
    w = make_config(2, n=500)
    dk, dm, dw = dev(w.keys), dev(w.momenta), dev(w.w_in)
    with pytest.raises(T.TrexError):
        T.trex_run(dk, dm[:, :, :400].contiguous(), w.theta_old, w.theta_new, dw)
    with pytest.raises(T.TrexError):
        T.trex_run(dk[:300].contiguous(), dm, w.theta_old, w.theta_new, dw)
    with pytest.raises(T.TrexError):
        T.trex_run(dk, dm, w.theta_old, w.theta_new, dw, w_out=torch.empty(499, dtype=torch.float64, device="cuda"))
    with pytest.raises(T.TrexError):
        T.trex_run_host(w.keys, w.momenta.astype(np.float32), w.theta_old, w.theta_new, w.w_in, np.empty(w.n))
    with pytest.raises(T.TrexError):
        T.trex_run_host(w.keys, torch.from_numpy(w.momenta).float(), w.theta_old, w.theta_new, w.w_in, np.empty(w.n))


def test_multi_polynomial_path_with_zero_vev_reference(T):
    """theta_old with vev = 0 (kappa_old = 0 whatever c_tG is): the polynomial path carries kappa itself, no division by vev."""
    import torch
    w = make_config(2, n=3000)
    tho = w.theta_old.copy(); tho[9] = 0.0; tho[7] = 0.4
    thetas = []
    for ctg in (-1.0, -0.3, 0.2, 0.45, 2.0):
        th = w.theta_old.copy(); th[7] = ctg
        thetas.append(th)
    dk, dm, dw = dev(w.keys), dev(w.momenta), dev(w.w_in)
    wp = T.trex_run_multi(dk, dm, tho, thetas, dw)[0]
    T.trex_set_poly_multi(False)
    try:
        wd = T.trex_run_multi(dk, dm, tho, thetas, dw)[0]
    finally:
        T.trex_set_poly_multi(True)
    torch.cuda.synchronize()
    a, b = wp.cpu().numpy(), wd.cpu().numpy()
    assert np.all(np.isfinite(a)) and rel(a, b).max() < 1e-12


# ---------------------------------------------------------------- all-event cross-checks at bench-like sizes
@pytest.mark.parametrize("sid,cfg,n", [(3, 4, 65536), (4, 5, 4096), (2, 3, 200000)])
def test_table_kernel_equals_first_path_on_every_event(T, sid, cfg, n):
    """k_table (the kernel bench.py times) against the independent one-thread-per-helicity walk k_ttng on EVERY event of
    a multi-wave launch (persistent blocks, strided events, ragged tail): catches stride / tail / reuse bugs that a
    handful of oracle-sampled events cannot. A sample of the same launch is oracle-checked."""
    import torch
    w = make_config(cfg, n=n + 13)
    if cfg == 3:
        sel = np.where(w.keys == w.classes[0].key)[0]
        mom, win = np.ascontiguousarray(w.momenta[:, :, sel]), w.w_in[sel]
    else:
        mom, win = w.momenta, w.w_in
    dm, dw = dev(mom), dev(win)
    a = T.trex_reweight(sid, dm, w.theta_old, w.theta_new, dw)
    T.trex_set_algorithm(0)
    try:
        b = T.trex_reweight(sid, dm, w.theta_old, w.theta_new, dw)
    finally:
        T.trex_set_algorithm(3)
    torch.cuda.synchronize()
    for x, y in zip(a, b):
        x, y = x.cpu().numpy(), y.cpu().numpy()
        assert np.all(np.isfinite(x)) and rel(x, y).max() < 1e-12
    idx = np.linspace(0, len(win) - 1, 7).astype(int)
    rw, ro, rn = O.reweight(sid, np.ascontiguousarray(mom[:, :, idx]), w.theta_old, w.theta_new, win[idx])
    assert rel(a[0].cpu().numpy()[idx], rw).max() < RTOL64 and rel(a[1].cpu().numpy()[idx], ro).max() < RTOL64


def test_full_cfg3_run_equals_per_class_calls_on_every_event(T):
    """trex_run on the full 1,048,576-event mixed sample against one trex_reweight per class on the class's events."""
    import torch
    w = make_config(3)
    out = T.trex_run(dev(w.keys), dev(w.momenta), w.theta_old, w.theta_new, dev(w.w_in))
    torch.cuda.synchronize()
    got = [x.cpu().numpy() for x in out[:3]]
    for sp in w.classes:
        sel = np.where(w.keys == sp.key)[0]
        ref = T.trex_reweight(sp.sid, dev(np.ascontiguousarray(w.momenta[:, :, sel])), w.theta_old, w.theta_new, dev(w.w_in[sel]))
        torch.cuda.synchronize()
        for g, r in zip(got, ref):
            assert np.array_equal(g[sel], r.cpu().numpy()), sp.name


@pytest.mark.parametrize("sid,cfg,n", [(3, 4, 40000), (4, 5, 3000), (2, 3, 150000), (1, 2, 65536)])
def test_repeated_launches_are_bit_identical(T, sid, cfg, n):
    """The barrier-heavy kernels (k_table4w: event pipeline with double-buffered tables and a named barrier; k_table:
    phases separated by block / warp barriers, shared-memory regions reused across iterations) must give the same bits
    on every launch: a shared-memory race shows up as run-to-run differences long before it shows up as a wrong digit.
    (compute-sanitizer is closed on this GPU pool, so racecheck cannot be run; this and the all-event cross-checks above
    stand in for it.)"""
    import torch
    w = make_config(cfg, n=n)
    if cfg == 3:
        sel = np.where(w.keys == w.classes[0].key)[0]
        mom, win = np.ascontiguousarray(w.momenta[:, :, sel]), w.w_in[sel]
    else:
        mom, win = w.momenta, w.w_in
    dm, dw = dev(mom), dev(win)
    ref = None
    for rep in range(6):
        if rep == 3:                                         # other work in between: different SM residency / timing
            big = make_config(2, n=200000)
            T.trex_reweight(1, dev(big.momenta), big.theta_old, big.theta_new, dev(big.w_in))
        out = T.trex_reweight(sid, dm, w.theta_old, w.theta_new, dw)
        torch.cuda.synchronize()
        if ref is None:
            ref = [x.clone() for x in out]
        else:
            for x, y in zip(out, ref):
                assert torch.equal(x, y), rep


def test_multi_channel_sample_one_quark_family_launch(T):
    """cfg6 (NEXT-4): a p p -> t t~ + parton sample with all 16 one-light-line classes (5 massless flavours). The whole path
    takes ONE launch for the gluonic channel and ONE for every quark-channel class together (the kernel finds its class in
    the device plan): weights against the oracle per class, launch count independent of the number of classes, and
    every event equal to a per-class trex_reweight call."""
    import torch
    w = make_config(6, n=60000)
    assert len(w.classes) == 16
    dk, dm, dw = dev(w.keys), dev(w.momenta), dev(w.w_in)
    l0 = T.trex_launch_count()
    wo, mo, mn, nb = T.trex_run(dk, dm, w.theta_old, w.theta_new, dw)
    torch.cuda.synchronize()
    launches = T.trex_launch_count() - l0
    assert nb == 16 and launches <= 10, launches          # 6 bucketing + gather + k_table<3> + k_qq + scatter
    got = [x.cpu().numpy() for x in (wo, mo, mn)]
    assert np.all(got[0] > 0) and np.all(np.isfinite(got[0]))
    for sp in w.classes:
        sel = np.where(w.keys == sp.key)[0]
        ref = T.trex_reweight(sp.sid, dev(np.ascontiguousarray(w.momenta[:, :, sel])), w.theta_old, w.theta_new, dev(w.w_in[sel]))
        torch.cuda.synchronize()
        for g, r in zip(got, ref):
            assert np.array_equal(g[sel], r.cpu().numpy()), sp.name
        idx = sel[:3]
        rw, ro, rn = O.reweight(sp.sid, np.ascontiguousarray(w.momenta[:, :, idx]), w.theta_old, w.theta_new, w.w_in[idx])
        assert rel(got[0][idx], rw).max() < RTOL64 and rel(got[1][idx], ro).max() < RTOL64 and rel(got[2][idx], rn).max() < RTOL64, sp.name
    # a sample that holds quark channels only, and one with a single quark class (reweighted in place, no transposition)
    for keep in ([sp.key for sp in w.classes if sp.sid != 2], [w.classes[5].key]):
        sel = np.where(np.isin(w.keys, np.array(keep, dtype=np.uint64)))[0]
        out = T.trex_run(dev(w.keys[sel]), dev(np.ascontiguousarray(w.momenta[:, :, sel])), w.theta_old, w.theta_new, dev(w.w_in[sel]))
        torch.cuda.synchronize()
        assert out[3] == len(keep) and np.array_equal(out[0].cpu().numpy(), got[0][sel])


def test_both_beam_orders_reach_the_same_class_through_the_parton_reindexing(T):
    """q g and g q (q q~ and q~ q, ...) share one flavour key -- legs are compared unordered -- and
    trex_run_pdg brings either order to the process string: cfg6 with shuffled legs gives the canonical weights."""
    import torch
    from trex_inputs import shuffled_legs
    w = make_config(6, n=30000)
    pdg, mom, n_in = shuffled_legs(w, 23)
    assert (pdg[0] != np.array([w.classes[0].pdg[0]] * w.n)).any()
    wo, _, _, nb = T.trex_run_pdg(torch.from_numpy(pdg).cuda(), dev(mom), n_in, w.theta_old, w.theta_new, dev(w.w_in))
    w0, _, _, nb0 = T.trex_run(dev(w.keys), dev(w.momenta), w.theta_old, w.theta_new, dev(w.w_in))
    torch.cuda.synchronize()
    assert nb == nb0 == 16 and rel(wo.cpu().numpy(), w0.cpu().numpy()).max() < 1e-12


def test_host_entry_point_pipelines_chunks_without_changing_a_bit(T):
    """trex_run_host cuts large samples into column ranges whose transfers overlap the kernels: per-event results and the
    number of buckets must be those of one trex_run over the whole sample (unknown classes and REX_NPOS included)."""
    import torch
    w = make_config(3, n=300001)
    keys = w.keys.copy()
    keys[3::1001] = np.uint64(REX_NPOS)
    keys[250000:] = np.where(keys[250000:] == w.classes[1].key, np.uint64(424242), keys[250000:])   # a class that first appears late
    ref = T.trex_run(dev(keys), dev(w.momenta), w.theta_old, w.theta_new, dev(w.w_in))
    torch.cuda.synchronize()
    out, mo, mn = np.full(w.n, -1.0), np.full(w.n, -1.0), np.full(w.n, -1.0)
    nb = T.trex_run_host(keys, w.momenta, w.theta_old, w.theta_new, w.w_in, out, mo, mn)
    assert nb == ref[3] == 7
    assert np.array_equal(out, ref[0].cpu().numpy()) and np.array_equal(mo, ref[1].cpu().numpy()) and np.array_equal(mn, ref[2].cpu().numpy())
    # pinned torch tensors, single-class sample (reweighted in place on the staged block: row stride != chunk length)
    w4 = make_config(4, n=140000)
    r4 = T.trex_run(dev(w4.keys), dev(w4.momenta), w4.theta_old, w4.theta_new, dev(w4.w_in))
    hk = torch.from_numpy(w4.keys.view(np.int64)).pin_memory()
    hm, hw = torch.from_numpy(w4.momenta).pin_memory(), torch.from_numpy(w4.w_in).pin_memory()
    ho = torch.empty(w4.n, dtype=torch.float64).pin_memory()
    assert T.trex_run_host(hk, hm, w4.theta_old, w4.theta_new, hw, ho) == 1
    assert np.array_equal(ho.numpy(), r4[0].cpu().numpy())


def test_four_leg_sample_with_both_classes(T):
    """A four-leg sample has two candidate classes (e- e+ > mu- mu+ and g g > t t~). A sample that really holds both (and a
    sample of each alone) must give what per-class trex_reweight calls give, and those agree with the oracle."""
    import torch
    a, b = make_config(1, n=3000), make_config(2, n=5000)
    rng = np.random.default_rng(8)
    th_old, th_new = b.theta_old.copy(), b.theta_new.copy()
    th_new[2] = a.theta_new[2]                                   # sin^2 theta_W moves as in cfg 1, c_tG as in cfg 2
    keys = np.concatenate([a.keys, b.keys])
    mom = np.concatenate([a.momenta, b.momenta], axis=2)
    w_in = np.concatenate([a.w_in, b.w_in])
    order = rng.permutation(len(keys))
    keys, mom, w_in = keys[order], np.ascontiguousarray(mom[:, :, order]), w_in[order]
    for sel_name, sel in (("both", np.arange(len(keys))), ("ee", np.where(keys == a.keys[0])[0]), ("gg", np.where(keys == b.keys[0])[0])):
        k, m, w = keys[sel], np.ascontiguousarray(mom[:, :, sel]), w_in[sel]
        l0 = T.trex_launch_count()
        out = T.trex_run(dev(k), dev(m), th_old, th_new, dev(w))
        torch.cuda.synchronize()
        nl = T.trex_launch_count() - l0
        got = [x.cpu().numpy() for x in out[:3]]
        assert out[3] == (2 if sel_name == "both" else 1), sel_name
        for sid, key in ((0, a.keys[0]), (1, b.keys[0])):
            idx = np.where(k == key)[0]
            if len(idx) == 0:
                continue
            r = T.trex_reweight(sid, dev(np.ascontiguousarray(m[:, :, idx])), th_old, th_new, dev(w[idx]))
            for g, x in zip(got, r):
                assert np.array_equal(g[idx], x.cpu().numpy()), (sel_name, sid)
            j = idx[:5]
            want = O.reweight(sid, np.ascontiguousarray(m[:, :, j]), th_old, th_new, w[j])
            for g, x in zip(got, want):
                assert rel(g[j], x).max() < RTOL64, (sel_name, sid)
        assert nl <= 6, nl                                        # small sample: bucketing, gather, two candidate launches, scatter
    # different top widths at the two points: the two-pass g g kernel runs
    th2 = th_new.copy(); th2[6] = 1.4
    out = T.trex_run(dev(keys), dev(mom), th_old, th2, dev(w_in))
    idx = np.where(keys == a.keys[0])[0][:4]
    want = O.reweight(0, np.ascontiguousarray(mom[:, :, idx]), th_old, th2, w_in[idx])
    assert rel(out[0].cpu().numpy()[idx], want[0]).max() < RTOL64
    idx = np.where(keys == b.keys[0])[0][:4]
    want = O.reweight(1, np.ascontiguousarray(mom[:, :, idx]), th_old, th2, w_in[idx])
    assert rel(out[0].cpu().numpy()[idx], want[0]).max() < RTOL64
