#!/usr/bin/env python
"""bench.py -- reweighted events/s of the whole hot path on B200 (contract: see DESIGN.md section 7).

One "step" = one pass of the whole path (rex_bucket -> transposition -> |M|^2(old,new) launches -> transposition back;
`trex_run`) over one batch of seeded synthetic events. Headline workload: cfg4 of BASELINE.json (g g -> t t~ g g,
1,048,576 events, c_tG 0 -> 0.3 and Gamma_t 1.50 -> 1.35), the largest configuration whose step is dominated by one
kernel family and the one the paper's cost statement is about ("completely dominated by scattering amplitude
evaluations"; GPU plateau at >= 1e5 events). The other configs are reported under "configs".

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--configs all|headline]

--gpus N > 1 without a torchrun environment starts N ranks itself (paper_2510_05100_b200.shard.launch_ranks).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from trex_inputs import make_config  # noqa: E402

METRIC = "reweighted events/s (old+new |M|^2)"
UNIT = "events/s"
HEADLINE_CFG = 4
HEADLINE_EVENTS = 1048576
L2_NOTE = "256 MiB buffer written between timed iterations (L2 flush)"
SID_OF_CFG = {1: 0, 2: 1, 4: 3, 5: 4}
KERNEL_OF_CFG = {1: "k_eemumu<double>", 2: "k_gg_tt<double,double>", 3: "k_table<double,double,3,1> + k_qq<double,double>",
                 4: "k_table4w<double,double,2>", 5: "k_table<double,double,5,1>", 6: "k_table<double,double,3,1> + k_qq<double,double>",
                 7: "k_table4w<double,double,1> + k_qq2<double,double>"}
# nominal FP64 vector peak of B200: 148 SMs x 64 DFMA/clk x 2 flop x 1.965 GHz
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12


def headline_config():
    """`config` of the JSON line: identical for both arms (ours / reference)."""
    return {"workload": "cfg4 gg->tt~gg (c_tG 0->0.3, Gamma_t 1.50->1.35), %d seeded massive-RAMBO events per GPU at sqrt(s)=1500 GeV "
                        "(BASELINE.json configs[3]: the largest single-kernel-family configuration)" % HEADLINE_EVENTS,
            "events_per_gpu": HEADLINE_EVENTS, "l2": L2_NOTE}


def load_flops():
    """Algorithmic FP64 work per reweighted event of the |M|^2 kernels: thread-level DFMA/DMUL/DADD counted by ncu
    (DFMA = 2 flop) on the committed kernels / events of the launch (profiles/flops_per_event.json)."""
    out = {"flops": {}, "tensor": {}, "traffic": {}, "oracle": {}, "flops_hsym": {}, "tensor_hsym": {}}
    path = os.path.join(ROOT, "profiles", "flops_per_event.json")
    if os.path.exists(path):
        with open(path) as fh:
            d = json.load(fh)
        for k, v in d.items():
            if k.isdigit():
                out["flops"][int(k)] = v
        out["tensor"] = {int(k): v for k, v in d.get("tensor_flop_per_event", {}).items()}
        out["traffic"] = {int(k): v for k, v in d.get("traffic_bytes", {}).items()}
        hs = d.get("helicity_symmetry", {})
        out["flops_hsym"] = {int(k): v for k, v in hs.items() if k.isdigit()}
        out["tensor_hsym"] = {int(k): v for k, v in hs.get("tensor_flop_per_event", {}).items()}
    opath = os.path.join(ROOT, "profiles", "oracle_flops_per_event.json")
    if os.path.exists(opath):
        with open(opath) as fh:
            out["oracle"] = json.load(fh)
    return out


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.25)
            self.proc.terminate()
            self.t.join(timeout=2)

    def summary(self):
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        pw = [float(r[2]) for r in self.rows if len(r) > 2 and r[2].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 7 for i in range(4) if r[3 + i].lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "reasons": reasons, "samples": len(sm)}


# seeded sample of each workload the oracle is timed on (about 10-30 s of host work; the rate is per event, so the
# sample size only sets the resolution)
ORACLE_SAMPLE = {1: 4096, 2: 65536, 3: 2048, 4: 4096, 5: 384, 6: 4096}


def cpu_oracle_rate(cfg, budget_s=20.0, n_sample=None):
    """The oracle as it stands (oracle/build.py: -O3 -march=native, OpenMP over events), timed on the host cores on a
    bounded seeded sample of workload `cfg`."""
    from oracle import oracle as O
    n_sample = n_sample or ORACLE_SAMPLE[cfg]
    w = make_config(cfg, n=n_sample)
    O.reweight(SID_OF_CFG.get(cfg, 2), np.ascontiguousarray(w.momenta[:, :, :8]), w.theta_old, w.theta_new, w.w_in[:8])  # load + colour tables
    cores = os.cpu_count()
    if cfg in (3, 6):
        t_class = {}
        for sp in w.classes:
            sel = np.where(w.keys == sp.key)[0]
            if sp.sid != 2:
                sel = sel[:max(1, len(sel) // 64)]      # the explicit-colour engine is ~250x slower: subsample, then rescale
            t1 = time.perf_counter()
            O.reweight(sp.sid, np.ascontiguousarray(w.momenta[:, :, sel]), w.theta_old, w.theta_new, w.w_in[sel])
            t_class[sp.sid] = (time.perf_counter() - t1) / len(sel)
        # time per event of the mixed sample = sum_class fraction * time per event of that class
        frac = {sp.sid: float(np.mean(w.keys == sp.key)) for sp in w.classes}
        per_event = sum(frac[s] * t_class[s] for s in frac)
        return {"value": 1.0 / per_event, "unit": UNIT, "cores": cores, "kind": "oracle",
                "sample": "cfg%d seeded sample of %d events; per-class time per event weighted by class fraction "
                          "(quark channels on 1/64 of their events)" % (cfg, n_sample)}
    done, t0 = 0, time.perf_counter()
    while True:
        O.reweight(SID_OF_CFG[cfg], w.momenta, w.theta_old, w.theta_new, w.w_in)
        done += w.n
        dt = time.perf_counter() - t0
        if dt > budget_s or done >= 4 * w.n:
            break
    return {"value": done / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "cfg%d seeded sample of %d events x %d pass(es), %.1f s" % (cfg, w.n, done // w.n, dt)}


def run_reference(args):
    """--impl reference: for this tier the reference arm is the CPU oracle (there is no reference code to install).
    Each step = the oracle on a bounded seeded sample of the headline workload; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    steps, n_step = max(1, args.steps), 1024
    for _ in range(min(args.warmup, 1)):
        cpu_oracle_rate(HEADLINE_CFG, budget_s=0.0, n_sample=256)
    vals, t0 = [], time.perf_counter()
    for _ in range(steps):
        vals.append(cpu_oracle_rate(HEADLINE_CFG, budget_s=0.0, n_sample=n_step))
        if time.perf_counter() - t0 > 150:
            break
    v = float(np.mean([x["value"] for x in vals]))
    cb = {"value": v, "unit": UNIT, "cores": vals[-1]["cores"], "kind": "oracle",
          "sample": "each of the %d steps = the oracle on a seeded %d-event sample of the workload, one pass" % (len(vals), n_step)}
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": len(vals),
                      "warmup": args.warmup, "ms_per_step": 1e3 * n_step / v, "higher_is_better": True, "scaling": "weak",
                      "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": headline_config(),
                      "cpu_baseline": cb,
                      "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def stats(ms):
    ms = np.asarray(ms, dtype=np.float64)
    return {"ms_per_step": float(ms.mean()), "ms_median": float(np.median(ms)), "ms_min": float(ms.min()), "ms_max": float(ms.max())}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--configs", default="all", choices=["all", "headline"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--profile", default="", help="comma-separated configs: run each (after one warm-up call) on --events "
                    "events through trex_run and exit; the command ncu / compute-sanitizer wrap for profiles/")
    ap.add_argument("--events", type=int, default=0)
    ap.add_argument("--precision", type=int, default=0)
    ap.add_argument("--extra-paths", action="store_true", help="with --profile: also one trex_run_pdg and one trex_run_multi call")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # not under torchrun: start the ranks ourselves (one process per GPU, NCCL rendezvous on 127.0.0.1)
        from paper_2510_05100_b200.shard import launch_ranks
        sys.exit(launch_ranks(os.path.abspath(__file__), args.gpus, sys.argv[1:]))

    import torch
    import torch.distributed as dist
    import paper_2510_05100_b200 as T
    from paper_2510_05100_b200.shard import shard_arrays, xsec_all_ranks

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the reweighting path has no CPU fallback")
    T.lib()
    F = load_flops()
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    stream = torch.cuda.current_stream()
    T.trex_set_stream(stream)
    T.trex_set_precision(0)
    W = max(3, args.warmup)
    K = max(1, args.steps)
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def dev(a):
        a = np.ascontiguousarray(a)
        return torch.from_numpy(a.view(np.int64) if a.dtype == np.uint64 else a).cuda()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def max_over_ranks(ms):
        if world == 1:
            return ms
        t = torch.tensor(ms, dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return t.cpu().tolist()

    def time_steps(fn, warm, steps):
        """Device time [ms] of each of `steps` calls of fn, L2 flushed (untimed) before each; max over ranks per step."""
        for _ in range(warm):
            fn()
        barrier()
        evs = []
        for _ in range(steps):
            flush_buf.zero_()
            s, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            s.record(stream)
            fn()
            e.record(stream)
            evs.append((s, e))
        barrier()
        return max_over_ranks([s.elapsed_time(e) for s, e in evs])

    def roofline_of(cfg, n, kernel_ms, fp64_peak, dmma_peak, hsym=True):
        """Executed FP64 flop of the |M|^2 kernel(s) of one step / their live CUDA-event duration, against the FP64 vector
        pipe peak measured in this run; tensor-pipe (DMMA) work is reported against its own peak, never summed in."""
        # with the helicity symmetry in use (library default; cfg 2, 3, 5, 6, 7 have Gamma_t = 0) the kernels execute fewer operations
        fpe = (F["flops_hsym"].get(cfg) if hsym else None) or F["flops"].get(cfg)
        if not fpe or not kernel_ms:
            return None
        ach = fpe * n / (kernel_ms * 1e-3) / 1e12
        r = {"bound": "alu", "achieved": ach, "peak": fp64_peak, "unit": "TFLOP/s", "frac": ach / fp64_peak,
             "traffic": F["traffic"].get(cfg), "kernel": KERNEL_OF_CFG[cfg], "kernel_ms": kernel_ms, "flop_per_event": fpe,
             "frac_of_nominal": ach / FP64_NOMINAL_TFLOPS}
        tfe = (F["tensor_hsym"].get(cfg) if hsym else None) or F["tensor"].get(cfg)
        if tfe:
            tach = tfe * n / (kernel_ms * 1e-3) / 1e12
            r["tensor_pipe"] = {"achieved": tach, "peak": dmma_peak, "frac": tach / dmma_peak if dmma_peak else None,
                                "flop_per_event": tfe, "note": "mma.sync.m8n8k4.f64 colour sum, separate pipe: not part of `achieved`"}
        return r

    def measure(cfg, warm, steps, precision=0, with_e2e=False, kernel_in_region=False, hsym=True):
        """One config: whole-path step time (trex_run), the |M|^2 kernels' own time (CUDA events recorded by the library
        around every |M|^2 launch on its stream) and optionally the end-to-end number with host buffers."""
        w = make_config(cfg)
        keys, mom, win = dev(w.keys), dev(w.momenta), dev(w.w_in)
        wout = torch.empty_like(win)
        T.trex_set_precision(precision)
        T.trex_set_helicity_symmetry(hsym)
        res = {"workload": w.name, "events": w.n, "steps": steps, "warmup": warm,
               "helicity_symmetry": bool(hsym and w.theta_old[6] == 0.0 and w.theta_new[6] == 0.0 and cfg in (2, 3, 5, 6, 7))}
        run = lambda: T.trex_run(keys, mom, w.theta_old, w.theta_new, win, w_out=wout, want_me2=False)  # noqa: E731
        if kernel_in_region:
            # the kernel is timed inside the timed region itself (the chain is launched directly, not as a graph replay:
            # at a step of >= 100 ms the launch overhead is invisible)
            T.trex_kernel_timing(True)
            for _ in range(warm):
                run()
            T.trex_kernel_time()
            l0 = T.trex_launch_count()
            ms = time_steps(run, 0, steps)
            nl = T.trex_launch_count() - l0
            kms, kcnt = T.trex_kernel_time()
            T.trex_kernel_timing(False)
            res["kernel_ms"] = kms / steps
            res["kernel_timing"] = "CUDA events around the |M|^2 launches inside the timed steps (%d launches)" % kcnt
        else:
            l0 = T.trex_launch_count()
            ms = time_steps(run, warm, steps)
            nl = (T.trex_launch_count() - l0) * steps // (warm + steps)
            T.trex_kernel_timing(True)
            run(); T.trex_kernel_time()
            ksteps = max(3, steps // 2)
            for _ in range(ksteps):
                flush_buf.zero_()
                run()
            kms, kcnt = T.trex_kernel_time()
            T.trex_kernel_timing(False)
            res["kernel_ms"] = kms / ksteps
            res["kernel_timing"] = "CUDA events around the |M|^2 launches, %d further steps without graph replay" % ksteps
        res.update(stats(ms))
        res["gpu_launches"] = int(nl)
        res["value"] = world * w.n * steps / (sum(ms) * 1e-3)
        assert bool(torch.isfinite(wout).all())
        if with_e2e:
            hk = torch.from_numpy(w.keys.view(np.int64)).pin_memory()
            hm = torch.from_numpy(w.momenta).pin_memory()
            hw = torch.from_numpy(w.w_in).pin_memory()
            ho = torch.empty(w.n, dtype=torch.float64).pin_memory()
            ems = time_steps(lambda: T.trex_run_host(hk, hm, w.theta_old, w.theta_new, hw, ho), 3, steps)
            res["e2e"] = {"value": world * w.n * steps / (sum(ems) * 1e-3), "unit": UNIT,
                          "h2d_bytes_per_step": int(hk.numel() * 8 + hm.numel() * 8 + hw.numel() * 8),
                          "d2h_bytes_per_step": int(ho.numel() * 8), "ms_median": float(np.median(ems)), "ms_min": float(min(ems))}
            assert bool(torch.isfinite(ho).all())
        T.trex_set_precision(0)
        T.trex_set_helicity_symmetry(True)
        del keys, mom, win, wout
        return res

    def measure_multi(cfg, npts, poly, warm, steps):
        """NEXT-1: npts parameter points (c_tG scan) on one categorisation; value = events x parameter points per second."""
        w = make_config(cfg)
        keys, mom, win = dev(w.keys), dev(w.momenta), dev(w.w_in)
        thetas = np.tile(w.theta_new, (npts, 1))
        thetas[:, 7] = np.linspace(-1.0, 1.0, npts)
        wout = torch.empty((npts, w.n), dtype=torch.float64, device="cuda")
        T.trex_set_poly_multi(poly)
        ms = time_steps(lambda: T.trex_run_multi(keys, mom, w.theta_old, thetas, win, w_out=wout, want_me2=False), warm, steps)
        T.trex_set_poly_multi(True)
        assert bool(torch.isfinite(wout).all())
        r = {"workload": w.name + ", %d parameter points (c_tG scan), %s" % (npts, "polynomial path" if poly else "one pass per point"),
             "events": w.n, "parameter_points": npts, "steps": steps, "warmup": warm,
             "value": world * w.n * npts * steps / (sum(ms) * 1e-3), "unit": "event-parameter-points/s"}
        r.update(stats(ms))
        return r

    def measure_strong(cfg, warm, steps):
        """Strong scaling: ONE sample split into contiguous event ranges, one per rank; no data-path
        collective; the eq.(6)-(7) moments of the shards are all-gathered (32 B per rank) and combined on every rank."""
        w = make_config(cfg)
        k, m, wi = shard_arrays(w.n, rank, world, w.keys, w.momenta, w.w_in)
        keys, mom, win = dev(k), dev(m), dev(wi)
        wout = torch.empty_like(win)
        ms = time_steps(lambda: T.trex_run(keys, mom, w.theta_old, w.theta_new, win, w_out=wout, want_me2=False), warm, steps)
        xs = xsec_all_ranks(T.trex_xsec_moments(win, wout), 1.0, 1.0, 0.01)
        r = {"workload": w.name + " split over %d rank(s)" % world, "events_total": w.n, "events_this_rank": int(win.numel()),
             "steps": steps, "warmup": warm, "value": w.n * steps / (sum(ms) * 1e-3), "unit": UNIT, "scaling": "strong",
             "xsec_ratio_sigma_new_over_old": xs[0] / float(w.w_in.sum()), "xsec_fallback": xs[2]}
        r.update(stats(ms))
        return r

    if args.profile:
        T.trex_set_precision(args.precision)
        for cfg in [int(c) for c in args.profile.split(",")]:
            w = make_config(cfg, n=args.events or None)
            keys, mom, win = dev(w.keys), dev(w.momenta), dev(w.w_in)
            for _ in range(2):
                T.trex_run(keys, mom, w.theta_old, w.theta_new, win)
            if args.extra_paths:
                from trex_inputs import shuffled_legs
                pdg, pmom, n_in = shuffled_legs(w, seed=5, unknown_every=7)
                T.trex_run_pdg(dev(pdg), dev(pmom), n_in, w.theta_old, w.theta_new, win)
                thetas = np.tile(w.theta_new, (6, 1)); thetas[:, 7] = np.linspace(-1, 1, 6)
                T.trex_run_multi(keys, mom, w.theta_old, thetas, win)
                T.trex_set_poly_multi(False)
                T.trex_run_multi(keys, mom, w.theta_old, thetas[:2], win)
                T.trex_set_poly_multi(True)
            torch.cuda.synchronize()
        print("profile run ok")
        return

    # ---- FP64 pipe peak, measured in this run
    def probe(mode):
        """mode 0 / 1: FP64 / FP32 FMA chains with constant-bank operands (pipe peak); 2 / 3: three register operands;
        4: FP64 tensor cores (DMMA)."""
        holder = {}

        def once():
            holder["flops"] = T.trex_probe_fma(mode, blocks=148 * 16, iters=2048)
        ms = time_steps(once, 2, 5)
        return holder["flops"] / (min(ms) * 1e-3) / 1e12

    with ClockSampler(local) as clk:
        head = measure(HEADLINE_CFG, W, K, with_e2e=True, kernel_in_region=True)
        fp64_peak = probe(0)
    clocks = clk.summary()
    fp32_peak, fp64_peak_3reg, dmma_peak = probe(1), probe(2), probe(4)

    configs = {}
    if args.configs == "all":
        for cfg, warm, steps in ((1, 3, 20), (2, 3, 20), (3, 3, 10), (5, 3, 10), (6, 3, 10), (7, 3, 10)):
            configs["cfg%d" % cfg] = measure(cfg, warm, steps, with_e2e=(cfg != 1))
        # the same samples with every helicity configuration evaluated (trex_set_helicity_symmetry(0)): the round-1 arithmetic
        for cfg, warm, steps in ((2, 3, 20), (3, 3, 10), (5, 3, 10), (7, 3, 10)):
            configs["cfg%d_all_helicities" % cfg] = measure(cfg, warm, steps, hsym=False)
        configs["cfg4_mixed"] = measure(4, 3, 10, precision=1)
        configs["cfg4_fp32"] = measure(4, 3, 10, precision=2)
        configs["cfg3_multi8_direct"] = measure_multi(3, 8, False, 2, 5)
        configs["cfg3_multi8_poly"] = measure_multi(3, 8, True, 2, 5)
        configs["cfg3_multi64_poly"] = measure_multi(3, 64, True, 2, 5)
        for name, r in configs.items():
            if name[3:].isdigit():
                r["roofline"] = roofline_of(int(name[3:]), r["events"], r.get("kernel_ms"), fp64_peak, dmma_peak)
            elif name.endswith("_all_helicities"):
                r["roofline"] = roofline_of(int(name[3]), r["events"], r.get("kernel_ms"), fp64_peak, dmma_peak, hsym=False)
    strong = measure_strong(HEADLINE_CFG, W, max(3, K // 2)) if world > 1 else None

    cpu = None
    if rank == 0 and not args.no_cpu_baseline:
        cpu = cpu_oracle_rate(HEADLINE_CFG)
        if args.configs == "all" and world == 1:
            for cfg in (1, 2, 3, 5, 6):
                configs["cfg%d" % cfg]["cpu_baseline"] = cpu_oracle_rate(cfg, budget_s=8.0)
            # cfg7: the oracle's explicit-colour engine needs about a minute per event and core for the two-gluon quark
            # channels (tests/test_oracle_two_gluon_channels.py): no bounded sample of it fits this run
            configs["cfg7"]["cpu_baseline"] = None

    if rank == 0:
        roof = roofline_of(HEADLINE_CFG, head["events"], head["kernel_ms"], fp64_peak, dmma_peak) or {
            "bound": "alu", "achieved": None, "peak": fp64_peak, "unit": "TFLOP/s", "frac": None, "traffic": None}
        roof.update({
            "peak_source": "FP64 FMA register-chain probe (trex_probe_fma, two constant-bank operands) timed in this run; "
                           "nominal %.1f TFLOP/s = 148 SM x 64 DFMA/clk x 2 x 1.965 GHz" % FP64_NOMINAL_TFLOPS,
            "kernel_share_of_step": head["kernel_ms"] / head["ms_per_step"],
            "fp32_peak_measured": fp32_peak, "fp64_tensor_peak_measured": dmma_peak,
            # the same probe with three REGISTER operands per FMA (what amplitude code issues): secondary roof, DESIGN.md 6
            "peak_three_register_operands": fp64_peak_3reg,
            "oracle_flop_per_event": F["oracle"].get("cfg4 g g > t t~ g g", {}).get("flop")})
        line = {"metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": head["ms_per_step"], "ms_median": head["ms_median"], "ms_min": head["ms_min"],
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic", "config": headline_config(),
                "clocks": clocks, "e2e": head["e2e"], "gpu_launches": head["gpu_launches"],
                "gpu_launches_per_step": head["gpu_launches"] / K,
                "roofline": roof, "cpu_baseline": cpu, "configs": configs}
        if strong:
            line["strong_scaling"] = strong
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
