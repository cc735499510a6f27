#!/usr/bin/env python
"""bench.py -- FP64 Poisson + wall-normal Helmholtz grid points/s on B200, fraction of the HBM roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2] [--impl ours|reference]

One "step" = one pass of the whole hot path over one batch of synthetic input: one pressure
Poisson solve (steps a1..a5) plus the wall-normal Helmholtz solve of every velocity component
(step a6) on the workload's grid.  Fields stay resident in HBM and are solved in place, step
after step (the solution of one step is the right-hand side of the next; the kernels' cost does
not depend on the values).  Every field is larger than the 126 MB L2, so no L2 flush is needed
between iterations.

Prints ONE JSON line.  The default (c2) line also carries, measured
OUTSIDE the c2 timed region and each with its own clock sample, the sub-records "poisson" (the
Poisson solve alone), "c3" (2048x1024x512, 20 solves with one plan) and "c4" (1024^3, 3 components,
100 solves), so that the driver's run holds every roofline target of BASELINE.json.

With N > 1 (torchrun, one rank per GPU):
  --scaling weak (default for c1, c2)   every rank solves its own independent problem of the
        workload's size (replicas; no data-path collective); value = sum over ranks / slowest rank.
  --scaling strong (default for c3, c4) ONE problem of the workload's size over all ranks: the
        Poisson solve by z-slabs with the paper's parallel tridiagonal solver around ONE NCCL
        all-gather of 2 nx ny boundary values per rank, the Helmholtz solves by
        y-slabs without any collective (sharded.py); value = the problem's points / slowest rank.

--impl reference times the CPU oracle (as it stands, never tuned) on the host cores on a bounded
sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "FP64 Poisson+Helmholtz grid points/s on 1 B200; % of HBM roofline"
UNIT = "grid points/s"
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled DURING the timed region."""

    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.lines = []
        self.proc = None
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.FIELDS}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            parts = [x.strip() for x in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
                pw.append(float(parts[2]))
            except ValueError:
                continue
            for nm, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample_shape(w, budget_pts):
    """Largest power-of-two sub-grid of the workload (same recipe) with at most budget_pts points."""
    nx, ny, nz = w.nx, w.ny, w.nz
    while nx * ny * nz > budget_pts:
        if nz >= nx and nz >= ny and nz > 16:
            nz //= 2
        elif nx >= ny and nx > 16:
            nx //= 2
        elif ny > 16:
            ny //= 2
        else:
            break
    return nx, ny, nz


def run_oracle_step(w_s, zc, zf, f, rs):
    import oracle

    t0 = time.perf_counter()
    if w_s.poisson:
        oracle.poisson_solve(w_s.lx, w_s.ly, zc, zf, f, 1)
    for r in rs:
        oracle.helmholtz_z_solve(zc, zf, w_s.a, r)
    return time.perf_counter() - t0


def cpu_baseline(w, target_seconds=15.0):
    """The oracle as it stands, timed on the host cores on a bounded sample of the workload."""
    import oracle
    from paper_2502_06296_b200 import workloads as wl

    cores = oracle.num_threads()
    fields = (1 if w.poisson else 0) + w.n_helmholtz
    # calibrate on a small sub-grid, then pick the sample size for ~target_seconds
    cal = wl.scaled(w, *oracle_sample_shape(w, 2 ** 21))
    zc, zf = wl.grid(cal)
    f = wl.poisson_rhs(cal) if cal.poisson else None
    rs = [wl.helmholtz_rhs(cal, c) for c in range(cal.n_helmholtz)]
    t_cal = run_oracle_step(cal, zc, zf, f, rs)
    rate = fields * cal.n / t_cal
    budget = min(w.n, max(cal.n, int(rate * target_seconds / fields)))
    smp = wl.scaled(w, *oracle_sample_shape(w, budget))
    zc, zf = wl.grid(smp)
    f = wl.poisson_rhs(smp) if smp.poisson else None
    rs = [wl.helmholtz_rhs(smp, c) for c in range(smp.n_helmholtz)]
    t = run_oracle_step(smp, zc, zf, f, rs)
    return {"value": fields * smp.n / t, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"1 step (1 Poisson + {w.n_helmholtz} Helmholtz solves, radix-2 FFT oracle variant) of the "
                      f"{w.name} recipe on a {smp.nx}x{smp.ny}x{smp.nz} sub-grid, {t:.2f} s",
            "seconds": t}


def bench_reference(args, w):
    """--impl reference: the oracle on the host cores, K steps, each a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    from paper_2502_06296_b200 import workloads as wl

    fields = (1 if w.poisson else 0) + w.n_helmholtz
    steps, warm = max(args.steps, 1), max(args.warmup, 0)
    # size each step for about 60 s total
    cal = wl.scaled(w, *oracle_sample_shape(w, 2 ** 21))
    zc, zf = wl.grid(cal)
    f = wl.poisson_rhs(cal) if cal.poisson else None
    rs = [wl.helmholtz_rhs(cal, c) for c in range(cal.n_helmholtz)]
    t_cal = run_oracle_step(cal, zc, zf, f, rs)
    rate = fields * cal.n / t_cal
    per_step = 60.0 / (steps + warm)
    smp = wl.scaled(w, *oracle_sample_shape(w, min(w.n, max(2 ** 18, int(rate * per_step / fields)))))
    zc, zf = wl.grid(smp)
    f = wl.poisson_rhs(smp) if smp.poisson else None
    rs = [wl.helmholtz_rhs(smp, c) for c in range(smp.n_helmholtz)]
    for _ in range(warm):
        run_oracle_step(smp, zc, zf, f, rs)
    t = sum(run_oracle_step(smp, zc, zf, f, rs) for _ in range(steps))
    value = fields * smp.n * steps / t
    sample = (f"each step = 1 Poisson + {w.n_helmholtz} Helmholtz solves of the {w.name} recipe on a "
              f"{smp.nx}x{smp.ny}x{smp.nz} sub-grid")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": warm, "ms_per_step": 1e3 * t / steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "grid": [w.nx, w.ny, w.nz], "sample_grid": [smp.nx, smp.ny, smp.nz]},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def traffic_of(workload, kernel):
    """dram bytes per launch of one kernel class from the newest committed ncu --set full capture
    (profiles/*_traffic.csv; columns workload,kernel,dram_bytes_per_launch[,commit]) and its label."""
    import csv
    import glob

    try:
        tfiles = sorted(glob.glob(os.path.join(ROOT, "profiles", "*_traffic.csv")))
        if not tfiles:
            return None, None
        with open(tfiles[-1]) as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload and row["kernel"] == kernel:
                    src = "profiles/" + os.path.basename(tfiles[-1]) + "@" + (row.get("commit") or "unlabelled")
                    return float(row["dram_bytes_per_launch"]), src
    except Exception:
        pass
    return None, None


def event_times(torch, fn, n, between=None):
    """n calls of fn, each bracketed by its own CUDA event pair on the current stream -> list of ms."""
    evs = []
    for _ in range(n):
        if between is not None:
            between()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        fn()
        b.record()
        evs.append((a, b))
    torch.cuda.synchronize()
    return [a.elapsed_time(b) for a, b in evs]


def kernel_table(pz, plan, n_calls):
    out = {}
    for ci, nm in enumerate(pz.KERNEL_CLASSES):
        ms, cnt = pz.pz_profile_read(plan, ci)
        if cnt:
            out[nm] = {"ms_per_launch": round(ms / cnt, 5), "launches_per_solve": cnt / n_calls}
    return out


def sub_poisson(torch, pz, plan, p, w, peak, n=10):
    """The Poisson solve alone (c2 grid), outside the timed region: ms per solve and the fraction of
    the measured copy rate on the 48 B/pt (three sweeps) and the strict 16 B/pt models."""
    for _ in range(2):
        pz.poisson_solve(plan, p)
    pz.pz_profile_enable(plan, True)
    ms = event_times(torch, lambda: pz.poisson_solve(plan, p), n)
    pz.pz_profile_enable(plan, False)
    med = statistics.median(ms)
    return {"ms_per_solve": med, "ms_mean": sum(ms) / len(ms), "solves": n, "points_per_s": w.n / (med * 1e-3),
            "frac_48B": 48.0 * w.n / (med * 1e-3) / 1e9 / peak, "frac_16B": 16.0 * w.n / (med * 1e-3) / 1e9 / peak,
            "kernels": kernel_table(pz, plan, n)}


def sub_c3(torch, pz, wl, peak, local):
    """BASELINE config 3: 2048x1024x512 Poisson, 20 solves with one plan, each solve between its own
    event pair, the right-hand side restored from a pristine copy outside the events."""
    w = wl.CONFIGS["c3"]
    zc, zf = wl.grid(w)
    plan = pz.poisson_plan_create(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf)
    f = wl.device_remove_weighted_mean(wl.device_field(w, w.poisson_seed), zf)
    p = f.clone()
    for _ in range(3):
        pz.poisson_solve(plan, p)
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.2)
    pz.pz_profile_enable(plan, True)
    ms = event_times(torch, lambda: pz.poisson_solve(plan, p), w.repeats, between=lambda: p.copy_(f))
    pz.pz_profile_enable(plan, False)
    clocks = sampler.stop()
    med = statistics.median(ms)
    rec = {"workload": "c3", "grid": [w.nx, w.ny, w.nz], "solves": w.repeats, "ms_per_solve": med,
           "ms_mean": sum(ms) / len(ms), "ms_min": min(ms), "ms_max": max(ms), "points_per_s": w.n / (med * 1e-3),
           "frac_48B": 48.0 * w.n / (med * 1e-3) / 1e9 / peak, "frac_16B": 16.0 * w.n / (med * 1e-3) / 1e9 / peak,
           "kernels": kernel_table(pz, plan, w.repeats), "clocks": clocks,
           "timing": "one CUDA event pair per solve; rhs restored from a pristine copy between solves (outside the events)"}
    pz.poisson_plan_destroy(plan)
    del p, f
    torch.cuda.empty_cache()
    return rec


def sub_c4(torch, pz, wl, peak, local):
    """BASELINE config 4: 1024^3 wall-normal Helmholtz, 3 components, coefficients once, 100 solves."""
    w = wl.CONFIGS["c4"]
    zc, zf = wl.grid(w)
    plan = pz.poisson_plan_create(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf)
    us = [wl.device_field(w, s) for s in w.helmholtz_seeds]
    t0 = time.perf_counter()
    pz.helmholtz_z_setup(plan, w.a)
    setup_ms = 1e3 * (time.perf_counter() - t0)
    for _ in range(3):
        pz.helmholtz_z_solve_n(plan, us)
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.2)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(w.repeats):
        pz.helmholtz_z_solve_n(plan, us)
    b.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = a.elapsed_time(b) / w.repeats
    nb = 16.0 * w.n_helmholtz * w.n
    rec = {"workload": "c4", "grid": [w.nx, w.ny, w.nz], "components": w.n_helmholtz, "solves": w.repeats,
           "ms_per_solve_of_3_components": ms, "setup_ms_host": setup_ms,
           "points_per_s": w.n_helmholtz * w.n / (ms * 1e-3), "GBps_algorithmic": nb / (ms * 1e-3) / 1e9,
           "frac_16B": nb / (ms * 1e-3) / 1e9 / peak, "clocks": clocks}
    pz.poisson_plan_destroy(plan)
    del us
    torch.cuda.empty_cache()
    return rec


def sub_paper_shape(torch, pz, wl, peak, local):
    """The paper's per-GPU weak-scaling grid 3456 x 3072 x 30: mixed-radix transforms
    (3456 = 2^7 27, 3072 = 2^10 3).  Poisson, 10 solves with one plan."""
    w = wl.scaled(wl.CONFIGS["c3"], 3456, 3072, 30, name="paper_weak_3456x3072x30")
    zc, zf = wl.grid(w)
    plan = pz.poisson_plan_create(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf)
    p = wl.device_remove_weighted_mean(wl.device_field(w, w.poisson_seed), zf)
    for _ in range(3):
        pz.poisson_solve(plan, p)
    torch.cuda.synchronize()
    pz.pz_profile_enable(plan, True)
    ms = event_times(torch, lambda: pz.poisson_solve(plan, p), 10)
    pz.pz_profile_enable(plan, False)
    med = statistics.median(ms)
    rec = {"workload": w.name, "grid": [w.nx, w.ny, w.nz], "solves": 10, "ms_per_solve": med,
           "points_per_s": w.n / (med * 1e-3), "frac_48B": 48.0 * w.n / (med * 1e-3) / 1e9 / peak,
           "frac_80B_five_passes": 80.0 * w.n / (med * 1e-3) / 1e9 / peak, "kernels": kernel_table(pz, plan, 10),
           "note": "mixed-radix kernels (pz_fft_generic.cu), five HBM passes"}
    pz.poisson_plan_destroy(plan)
    del p
    torch.cuda.empty_cache()
    return rec


def bench_strong(args, w, torch, pz, ranks, wl, rank, world, local, dist):
    """ONE problem of the workload over all ranks: Poisson by z-slabs around one all-gather
    (sharded.SlabPoisson), Helmholtz by y-slabs without a collective (sharded.YSlabHelmholtz)."""
    from paper_2502_06296_b200 import sharded

    steps, warm = max(args.steps, 1), max(args.warmup, 3)
    zc, zf = wl.grid(w)
    fields = (1 if w.poisson else 0) + w.n_helmholtz
    jp = jh = p = None
    us = []
    if w.poisson:
        exchange = args.exchange
        try:
            jp = sharded.SlabPoisson(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf, rank, world, exchange=exchange,
                                     group=(dist.group.WORLD if (dist is not None and exchange == "p2p") else None))
            if exchange == "p2p" and dist is None:
                sharded.SlabPoisson.connect([jp])
        except Exception as exc:  # symmetric memory not available on this node: the collective always is
            if exchange != "p2p":
                raise
            sys.stderr.write(f"bench.py: p2p exchange unavailable ({exc}); falling back to all-gather\n")
            exchange = "allgather"
            jp = sharded.SlabPoisson(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf, rank, world)
        for kv in args.option:
            k, v = kv.split("=")
            pz.pz_set_option(jp.plan, k, int(v))
        ws = wl.scaled(w, w.nx, w.ny, jp.k1 - jp.k0)
        p = wl.device_field(ws, ranks.rank_seed(w.poisson_seed, rank))
        # compatibility of the GLOBAL right-hand side: remove its volume mean (one scalar all-reduce, set-up only)
        dzf = torch.as_tensor(zf[jp.k0 + 1:jp.k1 + 1] - zf[jp.k0:jp.k1], dtype=torch.float64, device=p.device)
        wsum = torch.dot(dzf, p.mean(dim=(1, 2))).reshape(1)
        if dist is not None:
            dist.all_reduce(wsum)
        p -= wsum / float(zf[-1] - zf[0])
    if w.n_helmholtz:
        jh = sharded.YSlabHelmholtz(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf, w.a, rank, world)
        wh = wl.scaled(w, w.nx, jh.j1 - jh.j0, w.nz)
        us = [wl.device_field(wh, ranks.rank_seed(s, rank)) for s in w.helmholtz_seeds]

    def step():
        if jp is not None:
            jp.solve(p, dist)
        if jh is not None:
            jh.solve(us)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(warm):
        step()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    for j in (jp, jh):
        if j is not None:
            pz.pz_profile_enable(j.plan, True)
    n0 = pz.pz_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(steps):
        step()
    ev1.record()
    barrier()
    ms_total = ev0.elapsed_time(ev1)
    launches = pz.pz_launch_count() - n0
    clocks = sampler.stop()
    kernel_ms = {}
    for j in (jp, jh):
        if j is None:
            continue
        pz.pz_profile_enable(j.plan, False)
        for ci, nm in enumerate(pz.KERNEL_CLASSES):
            ms, cnt = pz.pz_profile_read(j.plan, ci)
            if cnt:
                kernel_ms[nm] = {"ms_total": ms, "launches": cnt, "ms_per_launch": ms / cnt}
    t_max = ranks.max_over_ranks(ms_total, dist, "cuda")
    value = fields * w.n * steps / (t_max * 1e-3)

    e2e = None
    if not args.no_e2e:
        # this rank's slabs on pinned host buffers; upload, solve (with the all-gather), download, every step
        devs = ([p] if p is not None else []) + us
        hosts = [torch.empty(d.shape, dtype=torch.float64).pin_memory() for d in devs]
        for h, d in zip(hosts, devs):
            h.copy_(d)
        torch.cuda.synchronize()

        def e2e_step():
            for h, d in zip(hosts, devs):
                d.copy_(h, non_blocking=True)
            step()
            for h, d in zip(hosts, devs):
                h.copy_(d, non_blocking=True)

        e2e_step()
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.e2e_steps):
            e2e_step()
        e1.record()
        barrier()
        e_ms = ranks.max_over_ranks(e0.elapsed_time(e1), dist, "cuda")
        nbytes = sum(d.numel() for d in devs) * 8
        e2e = {"value": fields * w.n * args.e2e_steps / (e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": nbytes,
               "d2h_bytes_per_step": nbytes, "steps": args.e2e_steps, "ms_per_step": e_ms / args.e2e_steps,
               "api": "sharded.SlabPoisson.solve / YSlabHelmholtz.solve on this rank's slabs, pinned host buffers; "
                      "bytes are per rank"}
    if rank != 0:
        return 0
    peak, peak_src = measured_peak()
    dom = max(kernel_ms, key=lambda k: kernel_ms[k]["ms_total"])
    pts_p = (w.n // w.nz) * (jp.k1 - jp.k0) if jp is not None else 0
    pts_h = w.nx * (jh.j1 - jh.j0) * w.nz if jh is not None else 0
    per_launch_pts = {nm: (pts_h * w.n_helmholtz if nm == "helmholtz" else pts_p) * steps / v["launches"] for nm, v in kernel_ms.items()}
    achieved = 16.0 * per_launch_pts[dom] / (kernel_ms[dom]["ms_per_launch"] * 1e-3) / 1e9
    step_bytes = ((48.0 if w.poisson else 0.0) + 16.0 * w.n_helmholtz) * w.n
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warm,
        "ms_per_step": t_max / steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "grid": [w.nx, w.ny, w.nz], "fields_per_step": fields,
                   "step": f"{1 if w.poisson else 0} Poisson solve + {w.n_helmholtz} Helmholtz solves of ONE problem, in place",
                   "parallelism": (f"z-slabs x{world} (P-TDMA, exchange = {jp.exchange if jp else None}: {jp.bytes_exchanged_per_solve if jp else 0} B per rank and solve)"
                                   if w.poisson else "") + (f" y-slabs x{world} (no collective)" if w.n_helmholtz else ""),
                   "l2": "every rank's slab is larger than the 126 MB L2 up to 8 ranks at c3 / c4; no flush",
                   "options": args.option},
        "clocks": clocks, "gpu_launches": launches,
        "roofline": {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": None, "peak_source": peak_src,
                     "algorithmic_bytes_per_launch": 16.0 * per_launch_pts[dom],
                     "share_of_step": kernel_ms[dom]["ms_total"] / ms_total, "note": "rank 0's kernels on its slab"},
        "hbm_roofline_step": {"bytes_per_step": step_bytes, "frac": step_bytes * steps / (t_max * 1e-3) / 1e9 / (peak * world),
                              "model": "48 B/pt Poisson + 16 B/pt per Helmholtz field, against world x the measured copy rate"},
        "kernels": {nm: {"ms_per_launch": round(v["ms_per_launch"], 5), "launches_per_step": v["launches"] / steps}
                    for nm, v in kernel_ms.items()},
    }
    if e2e is not None:
        line["e2e"] = e2e
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c2",
                    help="c1, c2 (default), c3 or c4 of BASELINE.json; 'paper' = only the 3456x3072x30 sub-record (for profiling)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--option", action="append", default=[], help="key=value passed to pz_set_option")
    ap.add_argument("--scaling", default=None, choices=["weak", "strong"],
                    help="N > 1: weak = replicas (default c1, c2), strong = one problem by z-/y-slabs (default c3, c4)")
    ap.add_argument("--no-extras", action="store_true", help="skip the sub-records measured outside the timed region")
    ap.add_argument("--exchange", default="allgather", choices=["allgather", "p2p"],
                    help="--scaling strong: boundary exchange of the z-slab Poisson solve (NCCL all-gather, or stores of the "
                         "reduction kernel into peer memory)")
    args = ap.parse_args()

    from paper_2502_06296_b200 import workloads as wl

    if args.workload == "paper":   # the mixed-radix sub-record on its own: one JSON object, not the bench line
        import torch

        from paper_2502_06296_b200 import binding as pz

        pz.lib()
        print(json.dumps(sub_paper_shape(torch, pz, wl, measured_peak()[0], 0)))
        return
    w = wl.CONFIGS[args.workload]
    if args.impl == "reference":
        return bench_reference(args, w)

    import numpy as np
    import torch

    from paper_2502_06296_b200 import binding as pz
    from paper_2502_06296_b200 import ranks

    pz.lib()  # fail loudly if the CUDA extension is missing
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; there is no CPU fallback")

    rank, world, local = ranks.env_rank()
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod

        dist = dist_mod
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    steps, warm = max(args.steps, 1), max(args.warmup, 3)
    scaling = args.scaling or ("strong" if (world > 1 and args.workload in ("c3", "c4")) else "weak")
    if scaling == "strong":
        rc = bench_strong(args, w, torch, pz, ranks, wl, rank, world, local, dist)
        if dist is not None:
            dist.destroy_process_group()
        return rc

    # ---- synthetic inputs, resident in HBM (device-side seeded generators; rank-dependent seeds)
    zc, zf = wl.grid(w)
    plan = pz.poisson_plan_create(w.nx, w.ny, w.nz, w.lx, w.ly, zc, zf)
    for kv in args.option:
        k, v = kv.split("=")
        pz.pz_set_option(plan, k, int(v))
    fields = (1 if w.poisson else 0) + w.n_helmholtz
    p = None
    if w.poisson:
        p = wl.device_remove_weighted_mean(wl.device_field(w, ranks.rank_seed(w.poisson_seed, rank)), zf)
    us = [wl.device_field(w, ranks.rank_seed(s, rank)) for s in w.helmholtz_seeds]
    if w.n_helmholtz:
        pz.helmholtz_z_setup(plan, w.a)

    def step():
        if p is not None:
            pz.poisson_solve(plan, p)
        if us:
            pz.helmholtz_z_solve_n(plan, us)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(warm):
        step()
    barrier()

    # ---- timed region: exactly K steps, CUDA events on the launching stream, per-kernel events on
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    pz.pz_profile_enable(plan, True)
    n0 = pz.pz_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(steps):
        step()
    ev1.record()
    barrier()
    ms_total = ev0.elapsed_time(ev1)
    launches = pz.pz_launch_count() - n0
    pz.pz_profile_enable(plan, False)
    clocks = sampler.stop()
    kernel_ms = {}
    for ci, nm in enumerate(pz.KERNEL_CLASSES):
        ms, cnt = pz.pz_profile_read(plan, ci)
        if cnt:
            kernel_ms[nm] = {"ms_total": ms, "launches": cnt, "ms_per_launch": ms / cnt}

    t_max = ranks.max_over_ranks(ms_total, dist, "cuda")
    value = ranks.whole_job_rate(fields * w.n * steps, world, t_max)

    # ---- the Poisson solve alone, outside the timed region
    extras = not args.no_extras
    psub = sub_poisson(torch, pz, plan, p, w, measured_peak()[0]) if (extras and w.poisson) else None

    # ---- next-row capability, outside the timed region: the fully implicit Helmholtz solve of Eq. (8)
    h3 = None
    if extras and w.poisson and w.nz <= 1024:
        pz.helmholtz3d_setup(plan, w.a if w.a > 0 else 2.5e-5)
        for _ in range(2):
            pz.helmholtz3d_solve(plan, p)
        h0, h1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        h0.record()
        for _ in range(5):
            pz.helmholtz3d_solve(plan, p)
        h1.record()
        torch.cuda.synchronize()
        h3_ms = h0.elapsed_time(h1) / 5
        h3 = {"ms_per_solve": h3_ms, "points_per_s": w.n / (h3_ms * 1e-3),
              "hbm_frac_48B_per_point": 48.0 * w.n / (h3_ms * 1e-3) / 1e9 / measured_peak()[0]}

    # ---- next-row capability, outside the timed region: the pressure-correction step of Eqs. (4)-(6)
    pc = None
    if extras and w.poisson and len(us) >= 3:
        work = torch.empty_like(p)
        gdt = 1e-3
        for _ in range(2):
            pz.pz_pressure_correction(plan, us[0], us[1], us[2], p, work, gdt)
        pz.pz_profile_enable(plan, True)
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        c0.record()
        for _ in range(5):
            pz.pz_pressure_correction(plan, us[0], us[1], us[2], p, work, gdt)
        c1.record()
        torch.cuda.synchronize()
        pz.pz_profile_enable(plan, False)
        pc_ms = c0.elapsed_time(c1) / 5
        pc_kernels = {}
        for ci, nm in enumerate(pz.KERNEL_CLASSES):
            ms, cnt = pz.pz_profile_read(plan, ci)
            if cnt:
                pc_kernels[nm] = round(ms / cnt, 5)
        pc = {"ms_per_step": pc_ms, "points_per_s": w.n / (pc_ms * 1e-3), "kernel_ms": pc_kernels,
              "note": "fft_x_fwd forms the right-hand side of Eq. (4) from u, v, w on the fly (algorithmic "
                      "32 B/pt); project moves 72 B/pt",
              "project_GBps_algorithmic": (72.0 * w.n / (pc_kernels["project"] * 1e-3) / 1e9
                                           if "project" in pc_kernels else None)}
        del work

    # ---- next-row capability, outside the timed region: the whole of Eq. (11) for one component
    hs = None
    if extras and len(us) >= 2:
        for _ in range(2):
            pz.helmholtz_z_step(plan, us[0], us[1])
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        s0.record()
        for _ in range(5):
            pz.helmholtz_z_step(plan, us[0], us[1])
        s1.record()
        torch.cuda.synchronize()
        hs_ms = s0.elapsed_time(s1) / 5
        hs = {"ms_per_field": hs_ms, "points_per_s": w.n / (hs_ms * 1e-3),
              "GBps_algorithmic_24B_per_point": 24.0 * w.n / (hs_ms * 1e-3) / 1e9}

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        # one pinned host buffer per field of the step; pz_solve_host_batch pipelines upload,
        # solve and download of consecutive fields (full-duplex PCIe)
        src = (p if p is not None else us[0]).flatten()
        hosts = []
        for _ in range(fields):
            h = torch.empty(w.n, dtype=torch.float64).pin_memory()
            h.copy_(src)
            hosts.append(h)
        torch.cuda.synchronize()

        def e2e_step():
            pz.pz_solve_host_batch(plan, hosts[0] if w.poisson else None, hosts[1:] if w.poisson else hosts)

        e2e_step()
        barrier()
        t0 = time.perf_counter()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.e2e_steps):
            e2e_step()
        e1.record()
        barrier()
        e_ms = e0.elapsed_time(e1)
        e_ms = ranks.max_over_ranks(e_ms, dist, "cuda")
        e2e = {"value": fields * w.n * world * args.e2e_steps / (e_ms * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": fields * w.n * 8, "d2h_bytes_per_step": fields * w.n * 8,
               "steps": args.e2e_steps, "ms_per_step": e_ms / args.e2e_steps,
               "api": "pz_solve_host_batch (pinned host buffers, one per field; upload / solve / download pipelined)"}
        del hosts

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    # ---- the other roofline targets of BASELINE.json (c3, c4), outside the timed region, own clock samples
    c3rec = c4rec = wkrec = None
    if extras and world == 1 and args.workload == "c2":
        pz.poisson_plan_destroy(plan)
        p = None
        us.clear()
        torch.cuda.empty_cache()
        c3rec = sub_c3(torch, pz, wl, measured_peak()[0], local)
        c4rec = sub_c4(torch, pz, wl, measured_peak()[0], local)
        wkrec = sub_paper_shape(torch, pz, wl, measured_peak()[0], local)

    # ---- roofline of the dominant kernel (largest share of the step), live event timings
    peak, peak_src = measured_peak()
    dom = max(kernel_ms, key=lambda k: kernel_ms[k]["ms_total"])
    bytes_per_launch = {  # algorithmic: every kernel reads and writes each of its points once
        nm: 16.0 * w.n * (steps * (w.n_helmholtz if nm == "helmholtz" else 1)) / kernel_ms[nm]["launches"]
        for nm in kernel_ms if not nm.startswith("pair0")}
    achieved = bytes_per_launch[dom] / (kernel_ms[dom]["ms_per_launch"] * 1e-3) / 1e9
    traffic, traffic_src = traffic_of(args.workload, dom)
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": bytes_per_launch[dom],
                "share_of_step": kernel_ms[dom]["ms_total"] / ms_total}
    # whole-step figures: 48 B/pt structural minimum for Poisson (3 sweeps), 16 B/pt per Helmholtz field
    step_bytes = ((48.0 if w.poisson else 0.0) + 16.0 * w.n_helmholtz) * w.n
    step_frac = step_bytes * steps / (ms_total * 1e-3) / 1e9 / peak
    per_kernel = {nm: {"ms_per_launch": round(v["ms_per_launch"], 5), "launches_per_step": v["launches"] / steps,
                       "share": round(v["ms_total"] / ms_total, 4),
                       "GBps_algorithmic": (round(bytes_per_launch[nm] / (v["ms_per_launch"] * 1e-3) / 1e9, 1)
                                            if nm in bytes_per_launch else None)}
                  for nm, v in kernel_ms.items()}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warm,
        "ms_per_step": t_max / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "grid": [w.nx, w.ny, w.nz], "fields_per_step": fields,
                   "step": f"{1 if w.poisson else 0} Poisson solve + {w.n_helmholtz} Helmholtz solves, in place",
                   "l2": "every field (%.2f GB) is larger than the 126 MB L2; no flush" % (w.n * 8 / 1e9),
                   "parallelism": "replicas" if world > 1 else "single GPU",
                   "options": args.option},
        "clocks": clocks, "gpu_launches": launches,
        "roofline": roofline,
        "hbm_roofline_step": {"bytes_per_step": step_bytes, "frac": step_frac,
                              "model": "48 B/pt Poisson (3 read+write sweeps) + 16 B/pt per Helmholtz field",
                              "strict_16B_poisson_frac": ((16.0 * fields) * w.n * steps / (ms_total * 1e-3) / 1e9 / peak)},
        "kernels": per_kernel,
    }
    if psub is not None:
        line["poisson"] = psub
    if c3rec is not None:
        line["c3"] = c3rec
    if c4rec is not None:
        line["c4"] = c4rec
    if wkrec is not None:
        line["paper_weak_shape"] = wkrec
    if h3 is not None:
        line["helmholtz3d"] = h3
    if pc is not None:
        line["pressure_correction"] = pc
    if hs is not None:
        line["helmholtz_z_step"] = hs
    if e2e is not None:
        line["e2e"] = e2e
    if not args.no_cpu_baseline and world == 1:
        # free the device first: nothing depends on it, and the oracle only uses host memory
        line["cpu_baseline"] = cpu_baseline(w)
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
