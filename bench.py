#!/usr/bin/env python
"""bench.py -- reweighted events/s of the whole hot path on B200 (contract: see DESIGN.md section 7).

One "step" = one pass of the whole path (rex_bucket -> transposition -> one |M|^2(old,new) launch per subprocess ->
transposition back; `trex_run`) over one batch of seeded synthetic events. Headline workload: BASELINE.json configs[1]
(gg -> tt~ + chromomagnetic operator, 65,536 events); the other four configs are reported under "configs".

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--configs all|headline]
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
HEADLINE_CFG = 2
HEADLINE_WORKLOAD = ("cfg2 gg->tt~ (+c_tG 0->0.5), 65536 seeded massive-RAMBO events per GPU "
                     "(BASELINE.json configs[1]); inputs resident in HBM")

# Algorithmic FP64 work per reweighted event of the dominant kernel of each config: thread-level DFMA/DMUL/DADD counted
# by ncu (smsp__sass_thread_inst_executed_op_d{fma,mul,add}_pred_on.sum; DFMA = 2 flop) on the committed kernels,
# divided by the events of that launch (profiles/flops_per_event.json, profiles/r01c_kernels.md). None = not yet counted.
FLOP_PER_EVENT = {1: None, 2: None, 3: None, 4: None, 5: None}
SID_OF_CFG = {1: 0, 2: 1, 4: 3, 5: 4}
# nominal FP64 vector peak of B200: 148 SMs x 64 DFMA/clk x 2 flop x 1.965 GHz
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12


ORACLE_FLOPS = {}


def load_flops():
    opath = os.path.join(ROOT, "profiles", "oracle_flops_per_event.json")
    if os.path.exists(opath):
        with open(opath) as fh:
            ORACLE_FLOPS.update(json.load(fh))
    path = os.path.join(ROOT, "profiles", "flops_per_event.json")
    if os.path.exists(path):
        with open(path) as fh:
            for k, v in json.load(fh).items():
                if k.isdigit():
                    FLOP_PER_EVENT[int(k)] = v


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
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 7 for i in range(4) if r[3 + i].lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def cpu_oracle_rate(cfg, budget_s=12.0):
    """The oracle as it stands, timed on the host cores on a bounded seeded sample of workload `cfg`."""
    from oracle import oracle as O
    n_sample = {1: 4096, 2: 65536, 3: 2048, 4: 768, 5: 48}[cfg]
    w = make_config(cfg, n=n_sample)
    O.reweight(SID_OF_CFG.get(cfg, 2), np.ascontiguousarray(w.momenta[:, :, :8]), w.theta_old, w.theta_new, w.w_in[:8])  # load + colour tables
    done, t0 = 0, time.perf_counter()
    while True:
        if cfg == 3:
            for sp in w.classes:
                sel = np.where(w.keys == sp.key)[0]
                if sp.sid != 2:
                    sel = sel[:max(1, len(sel) // 64)]      # the explicit-colour engine is ~250x slower: subsample, then rescale
                t1 = time.perf_counter()
                O.reweight(sp.sid, np.ascontiguousarray(w.momenta[:, :, sel]), w.theta_old, w.theta_new, w.w_in[sel])
                w.__dict__.setdefault("_t", {})[sp.sid] = (time.perf_counter() - t1) / len(sel)
            # time per event of the mixed sample = sum_class fraction * time per event of that class
            frac = {sp.sid: float(np.mean(w.keys == sp.key)) for sp in w.classes}
            per_event = sum(frac[s] * w._t[s] for s in frac)
            return {"value": 1.0 / per_event, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
                    "sample": "cfg3 seeded prefix of %d events; per-class time per event weighted by class fraction "
                              "(quark channels on 1/64 of their events)" % n_sample}
        O.reweight(SID_OF_CFG[cfg], w.momenta, w.theta_old, w.theta_new, w.w_in)
        done += w.n
        dt = time.perf_counter() - t0
        if dt > budget_s or done >= 4 * w.n:
            break
    return {"value": done / dt, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
            "sample": "cfg%d seeded sample of %d events x %d pass(es), %.1f s" % (cfg, w.n, done // w.n, dt)}


def run_reference(args):
    """--impl reference: for this tier the reference arm is the CPU oracle (there is no reference code to install)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    steps = max(1, args.steps)
    for _ in range(min(args.warmup, 1)):
        cpu_oracle_rate(HEADLINE_CFG, budget_s=0.5)
    vals, t0 = [], time.perf_counter()
    for _ in range(steps):
        vals.append(cpu_oracle_rate(HEADLINE_CFG, budget_s=60.0 / steps))
        if time.perf_counter() - t0 > 150:
            break
    v = float(np.mean([x["value"] for x in vals]))
    cb = dict(vals[-1]); cb["value"] = v
    n = 65536
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": len(vals),
                      "warmup": args.warmup, "ms_per_step": 1e3 * n / v, "higher_is_better": True, "scaling": "weak",
                      "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": HEADLINE_WORKLOAD, "events_per_gpu": n,
                                 "sample": "each step = the oracle on the whole 65536-event sample for a bounded time"},
                      "cpu_baseline": cb,
                      "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--configs", default="all", choices=["all", "headline"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--profile", default="", help="comma-separated configs: run each once (after one warm-up) on --events "
                    "events through trex_run and exit; the command ncu wraps for profiles/")
    ap.add_argument("--events", type=int, default=0)
    ap.add_argument("--precision", type=int, default=0)
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    import paper_2510_05100_b200 as T

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the reweighting path has no CPU fallback")
    T.lib()
    load_flops()
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl")
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

    def max_over_ranks(x):
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def time_steps(fn, warm, steps):
        """Device time of `steps` calls of fn, L2 flushed (untimed) before each; returns seconds (max over ranks)."""
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
        return max_over_ranks(sum(s.elapsed_time(e) for s, e in evs) * 1e-3)

    def measure(cfg, warm, steps, precision=0, with_e2e=False):
        w = make_config(cfg)
        keys, mom, win = dev(w.keys), dev(w.momenta), dev(w.w_in)
        wout = torch.empty_like(win)
        T.trex_set_precision(precision)
        res = {"workload": w.name, "events": w.n}
        l0 = T.trex_launch_count()
        sec = time_steps(lambda: T.trex_run(keys, mom, w.theta_old, w.theta_new, win, w_out=wout, want_me2=False), warm, steps)
        res["gpu_launches"] = (T.trex_launch_count() - l0) * steps // (warm + steps)
        res["ms_per_step"] = 1e3 * sec / steps
        res["value"] = world * w.n * steps / sec
        assert bool(torch.isfinite(wout).all())
        if precision == 0 and FLOP_PER_EVENT.get(cfg):
            # FP64 work of the |M|^2 kernels over the WHOLE step time (bucketing, transposition, launch gaps included)
            res["step_tflops"] = FLOP_PER_EVENT[cfg] * w.n * steps / sec / 1e12
        # the dominant kernel alone (single-class configs: the one |M|^2 launch of the step)
        if cfg in SID_OF_CFG:
            sid = SID_OF_CFG[cfg]
            ksec = time_steps(lambda: T.trex_reweight(sid, mom, w.theta_old, w.theta_new, win, w_out=wout, want_me2=False),
                              2, max(2, steps)) / max(2, steps)
            res["kernel_ms"] = 1e3 * ksec
            fpe = FLOP_PER_EVENT.get(cfg) if precision == 0 else None
            if fpe:
                res["kernel_tflops"] = fpe * w.n / ksec / 1e12
        if with_e2e:
            hk = torch.from_numpy(w.keys.view(np.int64)).pin_memory()
            hm = torch.from_numpy(w.momenta).pin_memory()
            hw = torch.from_numpy(w.w_in).pin_memory()
            ho = torch.empty(w.n, dtype=torch.float64).pin_memory()
            esec = time_steps(lambda: T.trex_run_host(hk, hm, w.theta_old, w.theta_new, hw, ho), 3, steps)
            res["e2e"] = {"value": world * w.n * steps / esec, "unit": UNIT,
                          "h2d_bytes_per_step": int(hk.numel() * 8 + hm.numel() * 8 + hw.numel() * 8),
                          "d2h_bytes_per_step": int(ho.numel() * 8)}
        T.trex_set_precision(0)
        del keys, mom, win, wout
        return res

    def measure_multi(cfg, K, poly, warm, steps):
        """NEXT-1: K parameter points (c_tG scan) on one categorisation; value = events x parameter points per second."""
        w = make_config(cfg)
        keys, mom, win = dev(w.keys), dev(w.momenta), dev(w.w_in)
        thetas = np.tile(w.theta_new, (K, 1))
        thetas[:, 7] = np.linspace(-1.0, 1.0, K)
        wout = torch.empty((K, w.n), dtype=torch.float64, device="cuda")
        T.trex_set_poly_multi(poly)
        sec = time_steps(lambda: T.trex_run_multi(keys, mom, w.theta_old, thetas, win, w_out=wout, want_me2=False), warm, steps)
        T.trex_set_poly_multi(True)
        assert bool(torch.isfinite(wout).all())
        return {"workload": w.name + ", %d parameter points (c_tG scan), %s" % (K, "polynomial path" if poly else "one pass per point"),
                "events": w.n, "parameter_points": K, "ms_per_step": 1e3 * sec / steps,
                "value": world * w.n * K * steps / sec, "unit": "event-parameter-points/s"}

    if args.profile:
        T.trex_set_precision(args.precision)
        for cfg in [int(c) for c in args.profile.split(",")]:
            w = make_config(cfg, n=args.events or None)
            keys, mom, win = dev(w.keys), dev(w.momenta), dev(w.w_in)
            for _ in range(2):
                T.trex_run(keys, mom, w.theta_old, w.theta_new, win)
            torch.cuda.synchronize()
        return

    # ---- FP64 pipe peak, measured in this run
    def probe(mode):
        """mode 0 / 1: FP64 / FP32 FMA chains with constant-bank operands (pipe peak); 2 / 3: three register operands."""
        holder = {}

        def once():
            holder["flops"] = T.trex_probe_fma(mode, blocks=148 * 16, iters=2048)
        sec = time_steps(once, 2, 5) / 5
        return holder["flops"] / sec / 1e12

    with ClockSampler(local) as clk:
        head = measure(HEADLINE_CFG, W, K, with_e2e=True)
        fp64_peak = probe(0)
    clocks = clk.summary()
    fp32_peak = probe(1)
    fp64_peak_3reg = probe(2)

    configs = {}
    if args.configs == "all":
        for cfg, warm, steps in ((1, 3, 10), (3, 1, 3), (4, 1, 2), (5, 1, 1)):
            configs["cfg%d" % cfg] = measure(cfg, warm, steps)
        configs["cfg4_mixed"] = measure(4, 1, 2, precision=1)
        configs["cfg4_fp32"] = measure(4, 1, 2, precision=2)
        configs["cfg3_multi8_direct"] = measure_multi(3, 8, False, 1, 2)
        configs["cfg3_multi8_poly"] = measure_multi(3, 8, True, 1, 2)
        configs["cfg3_multi64_poly"] = measure_multi(3, 64, True, 1, 2)
        for name, r in configs.items():
            if "kernel_tflops" in r:
                r["roofline_frac_fp64_measured"] = r["kernel_tflops"] / fp64_peak

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_oracle_rate(HEADLINE_CFG)
        if args.configs == "all":
            for cfg in (1, 3, 4, 5):
                configs["cfg%d" % cfg]["cpu_baseline"] = cpu_oracle_rate(cfg, budget_s=6.0)

    if rank == 0:
        ach = head.get("kernel_tflops")
        roof = {"bound": "alu", "achieved": ach, "peak": fp64_peak, "unit": "TFLOP/s",
                "frac": (ach / fp64_peak) if ach else None, "traffic": None,
                "kernel": "k_gg_tt<double,double>", "kernel_ms": head.get("kernel_ms"),
                "peak_source": "FP64 FMA register-chain probe (trex_probe_fma) timed in this run; nominal %.1f TFLOP/s" % FP64_NOMINAL_TFLOPS,
                "fp32_peak_measured": fp32_peak, "flop_per_event": FLOP_PER_EVENT.get(HEADLINE_CFG),
                # the same probe with three REGISTER operands per FMA (what amplitude code issues): the register file
                # feeds the FP64 pipe at this rate at most
                "peak_three_register_operands": fp64_peak_3reg,
                # what the oracle's plain algorithm spends on the same event (oracle/count_flops.py: counting scalar type)
                "oracle_flop_per_event": ORACLE_FLOPS.get("cfg%d g g > t t~" % HEADLINE_CFG, {}).get("flop"),
                "frac_of_three_register_peak": (ach / fp64_peak_3reg) if ach else None}
        tpath = os.path.join(ROOT, "profiles", "flops_per_event.json")
        if os.path.exists(tpath):
            with open(tpath) as fh:
                roof["traffic"] = json.load(fh).get("traffic_bytes_cfg2")
        line = {"metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": head["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": HEADLINE_WORKLOAD,
                           "l2": "256 MiB buffer written between timed iterations (L2 flush)",
                           "events_per_gpu": head["events"]},
                "clocks": clocks, "e2e": head["e2e"], "gpu_launches": head["gpu_launches"],
                "roofline": roof, "cpu_baseline": cpu, "configs": configs}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
