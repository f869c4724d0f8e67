#!/usr/bin/env python
"""bench.py — throughput of the fts-b200 hot path on B200, one JSON line.

A "step" is one pass of the whole hot path over one batch of synthetic fields: for the default workload
(BASELINE.json config 5: fluctuating AB diblock melt, complex Langevin, 256^3, Ns = 100, fp64) that is one
fts_cl_step = Boltzmann factors + 2 x 100 RQM4 contour steps (q and q+) + Q + Simpson densities + the
Euler-Maruyama update with Philox noise.  metric = grid-pt·contour-steps/s = M * 2*Ns * steps / time.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg5|cfg5s|cfg4|cfg3|cfg2|cfg1] [--precision f64|f32]
  python bench.py --impl reference ...      times the CPU oracle (the only other place oracle/ may be executed)
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1204_5434_b200 import inputs  # noqa: E402

METRIC, UNIT = "grid-pt·contour-steps/s", "grid-pt·contour-steps/s"
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12      # 148 SMs x 64 DFMA/clk x 2 flop x 1965 MHz (max clock) = 37.2
FP32_NOMINAL_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12     # 74.5


def make_workload(name):
    """(Config, kind) for a BASELINE.json configuration; kind in {'cl', 'scft', 'propagate'}."""
    if name == "cfg5":
        return inputs.config5(256), "cl"
    if name == "cfg5s":
        return inputs.config5(128), "cl"
    if name == "cfg4":
        return inputs.config4(), "cl"
    if name == "cfg3":
        return inputs.config3(), "scft"
    if name == "cfg2":
        return inputs.config2(), "scft"
    if name == "cfg1":
        return inputs.config1(), "propagate"
    raise SystemExit(f"unknown workload {name}")


def rqm4_steps_per_step(cfg, kind):
    """RQM4 steps of the METHOD per bench step (q and q+ counted separately, also when the real-field path marches them packed)."""
    nprop = 2 if cfg.model == "diblock" else 1
    solves = 2 if kind == "scft" else 1          # seidel = 1: two propagator solves per SCFT iteration
    return nprop * cfg.Ns * solves


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            self.proc.terminate()
            self.thread.join(timeout=2)

    def summary(self):
        ok = [r for r in self.rows if len(r) == 6 and r[0].isdigit()]
        if not ok:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[2 + i].lower().startswith("active") for r in ok)]
        return {"sm_mhz": float(np.median([int(r[0]) for r in ok])), "sm_max_mhz": float(ok[0][1]), "reasons": reasons, "samples": len(ok)}


_ORACLE_RATE = {}          # measured RQM4 grid-pt·steps/s of the oracle per workload, to size later samples


def oracle_sample(cfg, budget_s):
    """The oracle as it stands on one host core, on a bounded sample of the workload's contour march.

    Preferred sample: the first n contour steps of every propagator (Boltzmann factors + n RQM4 steps each, Eq. 12);
    when even n = 1 would exceed the budget, single RQM4 steps of one propagator.  Returns (units/s, seconds, text)."""
    from oracle import binding as ob
    M = int(np.prod(cfg.grid))
    nprop = 2 if cfg.model == "diblock" else 1
    rate = _ORACLE_RATE.get(cfg.name, 2.5e6)                                # first guess: the oracle's measured ~2.5e6 grid-pt·steps/s per core
    n = int(budget_s * rate / (M * nprop))
    if n >= 1:
        n = min(n, cfg.Ns)
        o = ob.Oracle(cfg.grid, cfg.cell, cfg.Ns, cfg.model, fA=cfg.fA, chiN=cfg.chiN, B=cfg.B, Cc=cfg.C)
        o.set_fields(cfg.f0, cfg.f1)
        t0 = time.perf_counter()
        o.propagate(n)
        dt = time.perf_counter() - t0
        units, what = M * nprop * n, f"first {n} of {cfg.Ns} contour steps of {'q and q+' if nprop == 2 else 'q'} ({nprop * n} RQM4 steps + Boltzmann factors)"
    else:
        w = cfg.f0 if cfg.model != "diblock" else cfg.f0 - cfg.f1
        q = np.ones(cfg.grid, np.complex128)
        n = max(1, int(budget_s * rate / M))
        t0 = time.perf_counter()
        for _ in range(n):
            q = ob.rqm4_step(cfg.grid, cfg.cell, 1.0 / cfg.Ns, w, q)
        dt = time.perf_counter() - t0
        units, what = M * n, f"{n} RQM4 step(s) of q in the species-A field (one Eq. 12 step each, tables rebuilt per call)"
    _ORACLE_RATE[cfg.name] = units / dt
    return units / dt, dt, what + ", cost linear in steps"


def config_dict(cfg, kind, prec, world, extra=None):
    """The same keys in both arms (the driver compares them)."""
    d = {"workload": cfg.name, "grid": list(cfg.grid), "Ns": cfg.Ns, "kind": kind, "precision": prec,
         "rqm4_steps_per_step": rqm4_steps_per_step(cfg, kind), "l2": "flushed between timed steps (256 MiB write)",
         "parallelism": f"replicas x{world}" if world > 1 else "1 GPU"}
    d.update(extra or {})
    return d


def run_options(args, kind):
    opts = dict((kv.split("=")[0], int(kv.split("=")[1])) for kv in args.opt)
    if kind == "scft" and "real_fields" not in opts:
        opts["real_fields"] = 1                     # SCFT fields are real: q and q+ share one packed march (N1)
    return opts


def run_extras(args, kind):
    """config keys that name HOW the workload is run; identical in both arms (the oracle ignores them: it always keeps every slice)."""
    return {"options": run_options(args, kind), "ops_every": args.ops_every, "slice_store": args.store}


def oracle_host_aggregate(workload, budget_s, n_steps_hint):
    """BASELINE.md plan (ii): P independent oracle processes concurrently on the host's cores (no threading inside the oracle);
    P = the box's core count, capped by memory and at 32.  Returns (aggregate units/s, P, cpu_count, text)."""
    import psutil
    cfg, _ = make_workload(workload)
    M = int(np.prod(cfg.grid))
    per_proc = 16.0 * M * (14 + 2 * (n_steps_hint + 1))          # bytes: tables, fields, Boltzmann factors, temporaries, the slices of the sample
    ncpu = os.cpu_count() or 1
    P = max(1, min(ncpu, 32, int(0.5 * psutil.virtual_memory().available / per_proc)))
    procs = [subprocess.Popen([sys.executable, os.path.abspath(__file__), "--oracle-worker", "--workload", workload, "--budget", str(budget_s)],
                              stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True) for _ in range(P)]
    t0 = time.perf_counter()
    outs = [p.communicate()[0] for p in procs]
    wall = time.perf_counter() - t0
    units = 0.0
    for o in outs:
        try:
            units += json.loads(o.strip().splitlines()[-1])["units"]
        except Exception:
            pass
    return units / wall, P, ncpu, f"{P} concurrent oracle processes (host has {ncpu} cores), each the one-core sample; wall {wall:.1f} s incl. process start-up"


def run_oracle_worker(args):
    cfg, _ = make_workload(args.workload)
    v, dt, what = oracle_sample(cfg, args.budget)
    print(json.dumps({"units": v * dt, "seconds": dt}))


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the same workload/metric; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cfg, kind = make_workload(args.workload)
    budget = min(20.0, 150.0 / (args.steps + args.warmup))
    for _ in range(args.warmup):
        oracle_sample(cfg, budget)
    units_s, secs, what = [], 0.0, ""
    for _ in range(args.steps):
        v, dt, what = oracle_sample(cfg, budget)
        units_s.append(v)
        secs += dt
    value = float(np.mean(units_s))
    full_units = int(np.prod(cfg.grid)) * rqm4_steps_per_step(cfg, kind)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * full_units / value, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": config_dict(cfg, kind, args.precision, max(1, args.gpus), run_extras(args, kind)),
        "note": "ms_per_step is the full step extrapolated from the bounded sample (the oracle's cost is linear in contour steps)",
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": f"per step: {what}"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


TRAFFIC_SOURCES = ("fts_march2.cuh", "fts_pencil.h")      # the files that define the kernel profiles/traffic.json was captured from


def march_source_sha():
    """sha256 over the march kernel's source files (there is no .git on the GPU box, so the stamp is a content hash)."""
    import hashlib
    h = hashlib.sha256()
    for f in TRAFFIC_SOURCES:
        h.update(open(os.path.join(ROOT, "paper_1204_5434_b200", "csrc", f), "rb").read())
    return h.hexdigest()[:16]


def executed_rqm4_per_propagate(cfg, opts):
    """RQM4 steps one fts_propagate EXECUTES: q and q+ share one packed march under real_fields (the roofline
    counts executed work; the headline metric keeps counting the method's two propagators)."""
    nprop = 2 if cfg.model == "diblock" else 1
    return (1 if opts.get("real_fields") else nprop) * cfg.Ns


def fma_peak_tflops(B, prec, dev):
    """Vector-FMA peak of this GPU in `prec`, register-resident chains timed with CUDA events; best of 3."""
    import torch
    scratch = torch.empty(148 * 8 * 256, dtype=torch.float64, device=dev)
    B.fma_peak_launch(prec, 512, scratch)
    best = 0.0
    for _ in range(3):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        nf = B.fma_peak_launch(prec, 8192, scratch)
        b.record()
        torch.cuda.synchronize()
        best = max(best, 2.0 * nf / (a.elapsed_time(b) * 1e-3) / 1e12)
    return best


def roofline_core(M, E, rq_exec, ms_march, peak_tflops, hbm_gbs):
    """F_alg = 30 M log2 M flop and B_alg = 3 E M bytes per executed RQM4 step of one propagator."""
    f_alg, b_alg = 30.0 * M * math.log2(M), 3.0 * E * M
    t_fp, t_hbm = f_alg / (peak_tflops * 1e12), b_alg / (hbm_gbs * 1e9)
    t_step = ms_march * 1e-3 / rq_exec
    if t_fp >= t_hbm:
        core = {"bound": "alu", "achieved": f_alg / t_step / 1e12, "peak": peak_tflops, "unit": "TFLOP/s", "frac": t_fp / t_step}
    else:
        core = {"bound": "hbm", "achieved": b_alg / t_step / 1e9, "peak": hbm_gbs, "unit": "GB/s", "frac": t_hbm / t_step}
    return core, f_alg, b_alg, t_hbm / t_step


def also_measure(B, workload, prec, store, steps, warmup, dev, flush, peak_tflops, hbm_gbs, seed):
    """One more shape of the north_star target, measured in the same run with the same events: the whole step
    (value, ms_per_step) and fts_propagate alone (march_ms, roofline fraction)."""
    import torch
    cfg, kind = make_workload(workload)
    cdt = torch.complex128 if prec == "f64" else torch.complex64
    M, E = int(np.prod(cfg.grid)), (16 if prec == "f64" else 8)
    g = B.Fts(cfg.grid, cfg.cell, cfg.Ns, cfg.model, precision=prec, device=dev, fA=cfg.fA, chiN=cfg.chiN, B=cfg.B, Cc=cfg.C,
              store_both=1 if store == "full" else 0)
    g.set_fields(*[torch.from_numpy(np.ascontiguousarray(f)).to(cdt).to(dev) for f in (cfg.f0, cfg.f1) if f is not None])

    def timed(fn, n, first):
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
        for i in range(n):
            flush.zero_()
            ev[i][0].record()
            fn(first + i)
            ev[i][1].record()
        torch.cuda.synchronize()
        return sum(a.elapsed_time(b) for a, b in ev)

    for i in range(warmup):
        g.cl_step(cfg.dt, 0, seed, i)
    ms = timed(lambda i: g.cl_step(cfg.dt, 0, seed, i), steps, warmup)
    g.propagate()
    ms_march = timed(lambda i: g.propagate(), steps, 0) / steps
    rq = executed_rqm4_per_propagate(cfg, {})
    core, _, _, _ = roofline_core(M, E, rq, ms_march, peak_tflops, hbm_gbs)
    out = {"workload": cfg.name, "precision": prec, "slice_store": store, "value": M * rqm4_steps_per_step(cfg, kind) * steps / (ms * 1e-3), "unit": UNIT,
           "ms_per_step": ms / steps, "march_ms": ms_march, "workspace_GB": round(g.workspace.numel() / 1e9, 2), "roofline": core}
    g.close()
    del g
    torch.cuda.empty_cache()
    return out


def max_over_ranks(values, device, world):
    """Device times of one replica per rank -> the slowest rank's (the job is as slow as its slowest replica).
    Replicas share nothing on the data path, so this is the only collective of the bench."""
    if world <= 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.tolist()]


def replica_seed(rank):
    """Each replica is an independent CL run: its own Philox key."""
    return 1000 + rank


def run_gpu(args):
    import torch
    import torch.distributed as dist
    from paper_1204_5434_b200 import binding as B

    rank, world, local = (int(os.environ.get(k, d)) for k, d in (("RANK", "0"), ("WORLD_SIZE", "1"), ("LOCAL_RANK", "0")))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback for the product path")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    B.lib()
    cfg, kind = make_workload(args.workload)
    prec = args.precision
    cdt = torch.complex128 if prec == "f64" else torch.complex64
    M, nprop = int(np.prod(cfg.grid)), (2 if cfg.model == "diblock" else 1)
    E = 16 if prec == "f64" else 8
    opts = run_options(args, kind)
    g = B.Fts(cfg.grid, cfg.cell, cfg.Ns, cfg.model, precision=prec, device=dev, options=opts, fA=cfg.fA, chiN=cfg.chiN, B=cfg.B, Cc=cfg.C,
              store_both=1 if args.store == "full" else 0)
    host = [torch.from_numpy(np.ascontiguousarray(f)).to(cdt).pin_memory() for f in (cfg.f0, cfg.f1) if f is not None]
    devf = [h.to(dev) for h in host]
    back = [torch.empty_like(h).pin_memory() for h in host]
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)           # > 126 MB L2
    seed = replica_seed(rank)

    def step(i):
        if kind == "cl":
            g.cl_step(cfg.dt, 0, seed, i)
            if args.ops_every and i % args.ops_every == 0:      # operator sampling (config 4: <mu>, <Pi>): out of the step's own solve
                g.operators(want_pi=args.store == "full")
        elif kind == "scft":
            g.scft_step(cfg.dt_scft[0], cfg.dt_scft[1], 1)
        else:
            g.propagate()
            g.density_operators()

    def timed(fn, n, first):
        """n calls, each bracketed by its own CUDA events on the launch stream, L2 flushed in between; returns ms total."""
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
        for i in range(n):
            flush.zero_()
            ev[i][0].record()
            fn(first + i)
            ev[i][1].record()
        torch.cuda.synchronize()
        return sum(a.elapsed_time(b) for a, b in ev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    g.set_fields(*devf)
    for i in range(args.warmup):
        step(i)
    barrier()
    launches0 = B.launch_count()
    with ClockSampler(local) as clk:
        ms = timed(step, args.steps, args.warmup)
    launches = B.launch_count() - launches0
    barrier()

    def e2e_step(i):
        for d, h in zip(devf, host):
            d.copy_(h, non_blocking=True)
        g.set_fields(*devf)
        step(i)
        if kind == "propagate":
            outs = list(g.density_operators()[1:2])
        else:
            outs = [t for t in g.get_fields() if t is not None]
        for o, b in zip(outs, back):
            b.copy_(o, non_blocking=True)

    e2e_step(0)
    barrier()
    ms_e2e = timed(e2e_step, args.steps, 1)
    barrier()

    # the march alone (fts_propagate: Boltzmann factors + the persistent march kernel + Q), for the roofline of march_kernel
    g.set_fields(*devf)
    g.propagate()
    barrier()
    l0 = B.launch_count()
    ms_march = timed(lambda i: g.propagate(), args.steps, 0) / args.steps
    march_launches = (B.launch_count() - l0) // args.steps

    # vector-FMA peak of this GPU, measured with the same events
    best = fma_peak_tflops(B, prec, dev)

    ms, ms_e2e, ms_march = max_over_ranks([ms, ms_e2e, ms_march], dev, world)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    units = M * rqm4_steps_per_step(cfg, kind)                # per step per GPU
    value = world * units * args.steps / (ms * 1e-3)
    pk, pk_kind = peaks()
    rq = executed_rqm4_per_propagate(cfg, opts)                # RQM4 steps one fts_propagate executes (packed march: Ns, not 2 Ns)
    roof, f_alg, b_alg, hbm_frac = roofline_core(M, E, rq, ms_march, best, pk["hbm_gbs"])
    t_step = ms_march * 1e-3 / rq
    if roof["bound"] == "alu":
        roof["peak_kind"] = f"vector {prec} FMA chains measured in this run (nominal {FP64_NOMINAL_TFLOPS if prec == 'f64' else FP32_NOMINAL_TFLOPS:.1f})"
    else:
        roof["peak_kind"] = pk_kind
    if opts.get("real_fields"):
        roof["counts"] = ("executed work: q and q+ march packed as ONE complex propagator (real_fields), Ns RQM4 steps per solve; the headline metric counts "
                          "the method's 2 Ns, so value / (M * achieved-rate) differs by that factor 2")
        roof["frac_if_method_steps_counted"] = 2.0 * roof["frac"]
    pass_launches = max(1, march_launches - 3)                 # fts_propagate = boltzmann + march launch(es) + 2 reduction kernels; cubic grids: ONE persistent march launch
    traffic, traffic_src, traffic_stale = None, None, None
    tp = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tp):
        tj = json.load(open(tp))
        traffic = tj.get(f"{args.workload}_{prec}_{args.store}", tj.get(f"{args.workload}_{prec}") if args.store == "full" else None)
        traffic_src = {k: tj.get(k) for k in ("_note", "_commit", "_sm_mhz", "_source_sha")}
        traffic_stale = tj.get("_source_sha") != march_source_sha()      # the kernel's source changed since the ncu capture
    roof.update({"traffic": traffic, "traffic_source": traffic_src, "traffic_stale": traffic_stale, "kernel": "march2_kernel (128^3, 256^3) / march_kernel (persistent: all T/Y1/Z/Y2 items of one propagator solve" + (")" if args.store == "full" else ", densities accumulated in the T items)"), "launches_per_march": pass_launches,
                 "avg_launch_us": ms_march * 1e3 / pass_launches, "alg_flops_per_launch": f_alg * rq / pass_launches,
                 "alg_bytes_per_launch": b_alg * rq / pass_launches, "march_ms": ms_march, "march_launches_all_kernels": march_launches,
                 "hbm_view": {"achieved_GBs_algorithmic": b_alg / t_step / 1e9, "peak_GBs": pk["hbm_gbs"], "peak_kind": pk_kind,
                              "frac_of_floor": hbm_frac}})
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": prec, "data": "synthetic",
           "config": config_dict(cfg, kind, prec, world, run_extras(args, kind)), "workspace_GB": round(g.workspace.numel() / 1e9, 2),
           "iterations_per_s": {"value": world * args.steps / (ms * 1e-3), "iteration": {"cl": "fts_cl_step (1 propagator solve)", "scft": "fts_scft_step, seidel=1 (2 propagator solves)",
                                                                                      "propagate": "fts_propagate + fts_density_operators"}[kind]},
           "clocks": clk.summary(),
           "e2e": {"value": world * units * args.steps / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": sum(h.numel() * h.element_size() for h in host),
                   "d2h_bytes_per_step": sum(b.numel() * b.element_size() for b in back[:1 if kind == 'propagate' else None])},
           "gpu_launches": launches, "roofline": roof}
    if world == 1 and args.workload == "cfg5" and prec == "f64" and not args.opt and not args.no_also:
        # the other shapes north_star names (128^3, fp32) and the library-default store, same run, same events
        g.close()
        del g, devf
        torch.cuda.empty_cache()
        best32 = fma_peak_tflops(B, "f32", dev)
        also = {}
        for wl, pr, st in (("cfg5", "f64", "mitm" if args.store == "full" else "full"), ("cfg5s", "f64", args.store), ("cfg5s", "f32", args.store), ("cfg5", "f32", args.store)):
            try:
                also[f"{wl}_{pr}_{st}"] = also_measure(B, wl, pr, st, args.steps, 3, dev, flush, best if pr == "f64" else best32, pk["hbm_gbs"], seed)
                if os.path.exists(tp):                           # ncu DRAM bytes of that variant's march launch (same stamp as roofline.traffic)
                    also[f"{wl}_{pr}_{st}"]["roofline"]["traffic"] = tj.get(f"{wl}_{pr}_{st}", tj.get(f"{wl}_{pr}") if st == "full" else None)
            except Exception as e:                               # context: never lose the bench line over it
                also[f"{wl}_{pr}_{st}"] = {"unavailable": repr(e)}
        out["also"] = also
    if world == 1 and not args.no_cpu_baseline:
        v, dt, what = oracle_sample(cfg, 20.0)
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": what, "seconds": dt}
        try:
            n_hint = max(1, int(20.0 * v / (M * nprop)))
            va, P, ncpu, text = oracle_host_aggregate(args.workload, 20.0, n_hint)
            out["cpu_baseline"]["whole_host"] = {"value": va, "unit": UNIT, "cores": P, "host_cores": ncpu, "sample": text}
        except Exception as e:                                   # the aggregate is context; never lose the bench line over it
            out["cpu_baseline"]["whole_host"] = {"unavailable": repr(e)}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="cfg5")
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-also", action="store_true", help="default workload only: skip the extra shapes (128^3, fp32, the other slice store) of the `also` block")
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=VALUE", help="fts_set_option (tuning experiments), e.g. --opt march=2")
    ap.add_argument("--store", default="full", choices=["full", "mitm"],
                    help="slice store: full = every slice kept, densities by one streaming pass (fastest on a 180 GB part, the default here); "
                         "mitm = the library's default meet-in-the-middle store, densities accumulated inside the march (half the memory)")
    ap.add_argument("--ops-every", type=int, default=0, help="CL workloads: call fts_operators (H, mu, Pi) every K steps inside the timed region (0 = never)")
    ap.add_argument("--oracle-worker", action="store_true", help=argparse.SUPPRESS)
    ap.add_argument("--budget", type=float, default=20.0, help=argparse.SUPPRESS)
    args = ap.parse_args()
    if args.oracle_worker:
        run_oracle_worker(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
