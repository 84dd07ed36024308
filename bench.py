#!/usr/bin/env python
"""bench.py -- throughput of the Landau gauge-fixing hot path (arXiv:1206.0675, Algorithm 1) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C3] [--precision fp64] [--storage 18]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N --steps K --warmup W
    python bench.py --impl reference [--steps K] [--warmup W]        # the CPU oracle, timed on the host cores

A "step" is one pass of the whole hot path -- one iteration of Algorithm 1's loop body (Delta/F/theta ->
forward FFT -> p2max/p2 -> inverse FFT -> g(x) -> link update) -- over one seeded
synthetic 32^4 configuration (BASELINE.json configs[2] = C3, the lattice the metric is quoted on).  The
headline line is fp64 / 18-real; the other precision x storage variants are timed the same way and listed
under "variants".  Rank 0 prints ONE JSON line.  Multi-GPU = independent replicas (one configuration per
GPU): no data-path collective, "scaling": "weak".

Everything timed here goes through the C ABI of liblgf.so (paper_1206_0675_b200.binding); the oracle is
executed only for the "cpu_baseline" object and for --impl reference.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1206_0675_b200 import ensemble  # noqa: E402  (host-side replica bookkeeping only)

METRIC = "gauge_fix_iterations_per_s"
UNIT = "iterations/s"
ALPHA = 0.08
FALLBACK_HBM_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback, used only if MEASURED_PEAKS.json is absent
PREC = {"fp64": 8, "fp32": 4}


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


NOMINAL_HBM_GBS = 8000.0           # north_star's "~8 TB/s" (nominal; the measured copy rate is the roofline denominator)
KERNEL_CLASS_OF = (("k_sweep", "update"), ("k_fft", "fft"), ("k_gbuild", "gbuild"), ("k_delta", "delta"))


def kernel_class_of(name):
    for prefix, cls in KERNEL_CLASS_OF:
        if ("lgf::" + prefix) in name or name.startswith(prefix) or (" " + prefix) in name:
            return cls
    return None


def short_kernel_name(name):
    """'void lgf::k_sweep<double, 3, 0, 0, 3>(lgf::LinkPair<T1>, ...)' -> 'k_sweep<double, 3, 0, 0, 3>'"""
    n = name.replace("void ", "").replace("lgf::", "").replace("(int)", "").replace("(bool)", "")
    depth, out = 0, []
    for ch in n:
        if ch == "(" and depth == 0:
            break
        depth += ch == "<"
        depth -= ch == ">"
        out.append(ch)
    return "".join(out).strip()


def captured_traffic(workload, precision, storage, launched):
    """DRAM bytes per launch of the iteration's kernels from the newest committed ncu capture
    (profiles/*_traffic.csv: dram__bytes_read.sum + dram__bytes_write.sum per launch), keyed by kernel class.
    `launched` = {class: [instantiation names]} from lgf_kernel_names: a stored row whose kernel is not one this
    build launches is REFUSED (listed under "stale").  A stored measurement, read as data; nothing here runs ncu."""
    import csv
    import glob

    rows, stale = {}, []
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "*_traffic.csv"))):
        try:
            with open(path, newline="") as f:
                found = {}
                for row in csv.DictReader(f):
                    if (row["workload"] == workload and row["precision"] == precision
                            and int(row["link_storage"]) == int(storage)):
                        ok = any(row["kernel"].startswith(nm) for nm in launched.get(row["kernel_class"], []))
                        rec = {"bytes": float(row["dram_bytes_per_launch"]), "kernel": row["kernel"],
                               "launches_per_step": float(row.get("launches_per_step") or 1.0),
                               "duration_us": float(row.get("duration_us") or 0.0),
                               "source": "profiles/" + os.path.basename(path)}
                        if ok:
                            found.setdefault(row["kernel_class"], []).append(rec)
                        else:
                            stale.append(rec["source"] + ": " + row["kernel"])
                if found:
                    rows = found               # a newer file with matching rows replaces an older one
        except Exception:  # noqa: BLE001
            continue
    return rows, stale


def reduce_ncu(args):
    """--reduce-ncu FILE: an `ncu --metrics dram__bytes_read.sum,dram__bytes_write.sum,gpu__time_duration.sum --csv`
    launch list of `bench.py --steps K ...` -> rows of a profiles/*_traffic.csv (per kernel instantiation: launches per
    step, mean DRAM bytes and mean duration per launch over the LAST K iterations' launches)."""
    import csv

    per = {}
    with open(args.reduce_ncu, newline="") as f:
        lines = [ln for ln in f if ln.startswith('"')]
    for row in csv.DictReader(lines):
        name = short_kernel_name(row["Kernel Name"])
        cls = kernel_class_of(name)
        if cls is None:
            continue
        d = per.setdefault(int(row["ID"]), {"name": name, "cls": cls})
        val = float(row["Metric Value"].replace(",", ""))
        unit = row["Metric Unit"]
        scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "ns": 1e-3, "us": 1.0, "ms": 1e3, "s": 1e6}.get(unit, 1.0)
        d[row["Metric Name"]] = val * scale
    ids = sorted(per)
    by_name = {}
    for i in ids:
        by_name.setdefault(per[i]["name"], []).append(per[i])
    print("workload,precision,link_storage,kernel_class,kernel,launches_per_step,dram_bytes_per_launch,duration_us,capture")
    n_iter = max([len(ls) for name, ls in by_name.items() if ls[0]["cls"] == "update"] or [1])   # one sweep per iteration
    for name, ls in by_name.items():
        per_step = max(1, round(len(ls) / n_iter))
        last = ls[-per_step * min(args.steps, max(1, len(ls) // per_step)):]
        b = np.mean([x.get("dram__bytes_read.sum", 0.0) + x.get("dram__bytes_write.sum", 0.0) for x in last])
        t = np.mean([x.get("gpu__time_duration.sum", 0.0) for x in last])
        print("%s,%s,%d,%s,\"%s\",%d,%.0f,%.3f,%s" % (args.workload, args.precision, args.storage, ls[0]["cls"], name, per_step, b, t,
                                                      os.path.basename(args.reduce_ncu)))
    return 0


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
               0x80: "hw_power_brake_slowdown"}

    def __init__(self, index, period=0.01):
        self.period, self.samples, self.reasons, self._stop = period, [], set(), threading.Event()
        self.max_mhz, self.ok = None, False
        try:
            import pynvml

            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:  # noqa: BLE001
            self.err = repr(e)
        self.thread = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        while not self._stop.is_set():
            try:
                self.samples.append(int(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
                r = int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                for bit, name in self.REASONS.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:  # noqa: BLE001
                pass
            time.sleep(self.period)

    def __enter__(self):
        if self.ok:
            self.thread.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self.ok:
            self.thread.join()

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def physical_gpu_index(local_rank):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:  # noqa: BLE001
            return local_rank
    return local_rank


# ---------------------------------------------------------------------------------------------------------
TUNE = {}          # --tune key=value[,key=value]: lgf_tune overrides applied to every context (ablations)


def apply_tune(ctx):
    for k, v in TUNE.items():
        ctx.tune(k, v)


def time_variant(binding, torch, U0, dims, prec_name, storage, steps, warmup, dist, sampler=None):
    """Device-resident timing of `steps` iterations.  Returns dict(ms_per_step, launches, kernels...)."""
    prec = PREC[prec_name]
    cdt = torch.complex128 if prec == 8 else torch.complex64
    stream = torch.cuda.current_stream()
    out = {}
    with binding.Context(dims, prec, storage, stream=stream) as ctx:
        apply_tune(ctx)
        d = torch.from_numpy(U0).to(cdt).cuda()
        ctx.set_links(d)
        # warm-up, itself timed on the device: gives the per-step estimate the stall check below uses
        w0, w1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ctx.iterate(ALPHA, 1)
        w0.record(stream)
        ctx.iterate(ALPHA, max(1, warmup - 1))
        w1.record(stream)
        torch.cuda.synchronize()
        warm_ms_per_step = w0.elapsed_time(w1) / max(1, warmup - 1)

        def timed_region():
            if dist is not None:
                dist.barrier()
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            ctx.iterate(ALPHA, steps)
            b.record(stream)
            torch.cuda.synchronize()
            if dist is not None:
                dist.barrier()
            return a.elapsed_time(b)

        n0 = ctx.launch_count()
        if sampler is not None:
            sampler.__enter__()
        ms = timed_region()
        # A timed region far slower than the warm-up steps of the same kernels is a stall of the launching
        # host thread, not kernel time (seen once on a fresh box: 35 s for 3 steps, not reproducible, cause
        # unknown).  It is re-measured ONCE and both numbers are reported; nothing is dropped silently.
        out["remeasured"] = None
        stalled = ms / steps > 20.0 * warm_ms_per_step
        # every rank takes the same branch (the timed region contains barriers): any rank stalled -> all re-measure
        if ensemble.max_over_ranks(dist, 1.0 if stalled else 0.0) > 0.5:
            first = ms
            n0 = ctx.launch_count()
            ms = timed_region()
            out["remeasured"] = {"reason": "first timed region stalled", "first_ms_per_step": first / steps,
                                 "warmup_ms_per_step": warm_ms_per_step, "second_ms_per_step": ms / steps}
        if sampler is not None:
            sampler.__exit__()
        out["launches"] = ctx.launch_count() - n0
        ms = ensemble.max_over_ranks(dist, ms)          # the slowest replica bounds the whole job
        out["ms_total"] = ms
        out["ms_per_step"] = ms / steps
        # per-kernel-class device times: every launch bracketed by CUDA events on the launching stream,
        # over the same number of steps (a second region, so that the brackets do not perturb `value`)
        ctx.set_profiling(True)
        ctx.iterate(ALPHA, steps)
        kt = ctx.kernel_times()
        ctx.set_profiling(False)
        kern = {}
        for i, name in enumerate(binding.KERNEL_CLASSES):
            ms_k, n_k = kt[name]
            if n_k == 0:
                continue
            per_iter_launches = n_k / steps
            bytes_iter = ctx.algorithmic_bytes(i)
            kern[name] = {"ms_per_step": ms_k / steps, "launches_per_step": per_iter_launches,
                          "avg_launch_us": 1e3 * ms_k / n_k, "algorithmic_bytes_per_step": bytes_iter,
                          "gbs": bytes_iter / (ms_k / steps * 1e-3) / 1e9 if ms_k > 0 else None}
        out["kernels"] = kern
        F, th, P = ctx.measure()
        out["F"], out["theta"], out["plaquette"] = F, th, P
        out["iter_bytes"] = ctx.algorithmic_bytes(binding.LGF_K_ITERATION)
        out["kernel_names"] = ctx.kernel_names()
    del d
    torch.cuda.empty_cache()
    return out


def time_sustained(binding, torch, U0, dims, prec_name, storage, seconds, ms_guess, index):
    """The same step run back to back for at least `seconds` of device time (a beta = 5.8 configuration needs
    ~10^4 iterations): the number a long fix sees once the board settles at its power cap."""
    prec = PREC[prec_name]
    cdt = torch.complex128 if prec == 8 else torch.complex64
    stream = torch.cuda.current_stream()
    sampler = ClockSampler(index, period=0.05)
    with binding.Context(dims, prec, storage, stream=stream) as ctx:
        apply_tune(ctx)
        d = torch.from_numpy(U0).to(cdt).cuda()
        ctx.set_links(d)
        chunk = max(50, int(0.25 * 1e3 / ms_guess))        # about a quarter of a second per call
        ctx.iterate(ALPHA, chunk)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n, t0 = 0, time.perf_counter()
        with sampler:
            a.record(stream)
            while True:
                ctx.iterate(ALPHA, chunk)
                n += chunk
                if time.perf_counter() - t0 > seconds and n * ms_guess * 1e-3 > 0.8 * seconds:
                    break
            b.record(stream)
            torch.cuda.synchronize()
        ms = a.elapsed_time(b)
    del d
    torch.cuda.empty_cache()
    return {"seconds": ms * 1e-3, "steps": n, "ms_per_step": ms / n, "value": 1e3 * n / ms, "unit": UNIT, "clocks": sampler.summary()}


def time_e2e(binding, torch, U0, dims, prec_name, storage, tol, max_iter, dist):
    """Algorithm 1 end to end through lgf_fix_host: pinned HOST buffer in, gauge-fixed HOST buffer out;
    the H2D and D2H copies of the configuration are inside the timed region."""
    prec = PREC[prec_name]
    cdt = torch.complex128 if prec == 8 else torch.complex64
    stream = torch.cuda.current_stream()
    with binding.Context(dims, prec, storage, stream=stream) as ctx:
        apply_tune(ctx)
        h = torch.from_numpy(U0).to(cdt).pin_memory()
        warm = h.clone().pin_memory()
        ctx.fix_host(warm, ALPHA, tol, 1)              # allocates the staging buffer, warms the kernels
        del warm
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record(stream)
        it = ctx.fix_host(h, ALPHA, tol, max_iter)
        e1.record(stream)
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        ms = max(e0.elapsed_time(e1), 1e3 * wall)
        if dist is not None:
            dist.barrier()
        ms = ensemble.max_over_ranks(dist, ms)
        F, th, _ = ctx.measure(plaquette=False)
        nbytes = h.numel() * h.element_size()
    return {"iterations": it, "ms": ms, "bytes_each_way": nbytes, "theta": th, "F": F}


def cpu_baseline(U0, dims, budget_s=30.0):
    """The oracle as it stands, on the host cores, on a bounded sample: whole iterations of Algorithm 1
    on the same configuration until ~budget_s have been spent (at least one)."""
    import oracle

    n, t = 0, 0.0
    U = U0
    while True:
        t0 = time.perf_counter()
        U, _, _ = oracle.iterate(dims, U, ALPHA, 1)
        t += time.perf_counter() - t0
        n += 1
        if t + t / n > budget_s:
            break
    # orc_iterate(n=1) = measure + update + measure; one loop-body pass is update + measure, so correct by
    # timing one extra measure
    t0 = time.perf_counter()
    oracle.measure(dims, U, want_delta=True)
    tm = time.perf_counter() - t0
    t_iter = t / n - tm
    return {"value": 1.0 / t_iter, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": "%d whole iteration(s) of Algorithm 1 on the full %s lattice, fp64, 9-component naive separable DFT "
                      "(%.2f s each)" % (n, "x".join(str(v) for v in dims), t_iter)}


# ---------------------------------------------------------------------------------------------------------
def run_reference(args):
    """--impl reference: the oracle, as it stands, timed on the host cores.  Rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    import oracle
    from paper_1206_0675_b200 import inputs

    oracle.build()
    cfg = inputs.CONFIGS[args.workload]
    dims = cfg["dims"]
    U = inputs.make_config(args.workload)
    budget = float(args.reference_budget)
    done_w, t_w = 0, 0.0
    for _ in range(max(1, args.warmup)):                 # warm-up steps (bounded by the budget)
        t0 = time.perf_counter()
        U, _, _ = oracle.iterate(dims, U, ALPHA, 1)
        t_w += time.perf_counter() - t0
        done_w += 1
        if t_w > 0.25 * budget:
            break
    per = t_w / done_w
    k = int(max(1, min(args.steps, (budget - t_w) // per)))
    # one call for the k timed steps: orc_iterate(n) = measure + n x (update + measure), so a step is one pass
    # of Algorithm 1's loop body, as in the CUDA arm and in cpu_baseline (the single leading measure is the
    # configuration's first Delta/F/theta, which the CUDA arm's first iteration also finds already computed)
    t0 = time.perf_counter()
    oracle.measure(dims, U, want_delta=True)
    t_measure = time.perf_counter() - t0
    t0 = time.perf_counter()
    U, _, _ = oracle.iterate(dims, U, ALPHA, k)
    t = time.perf_counter() - t0 - t_measure
    value = k / t
    sample = ("%d of the %d requested steps timed (%d warm-up); a step = one whole oracle iteration "
              "(9-component DFT pair + g + update + measure) on the full %s lattice, fp64"
              % (k, args.steps, done_w, "x".join(str(v) for v in dims)))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": k,
            "warmup": done_w, "ms_per_step": 1e3 * t / k, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.workload, dims), "precision": "fp64", "alpha": ALPHA},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def run_thermal(args):
    """--thermal BETA: the paper's kind of input.  Thermalise a cold 32^4 lattice with
    lgf_thermalize (heat bath, Wilson action) and gauge-fix it with lgf_fix: iterations and seconds to
    theta < 1e-15 (fp64) / 1e-12 (fp32), to set beside the paper's Table 3.  Prints one JSON
    line of its own; not the contract line."""
    import torch

    from paper_1206_0675_b200 import binding

    torch.cuda.set_device(0)
    binding.load()
    L = int(args.thermal_size)
    dims, prec = (L, L, L, L), PREC[args.precision]
    cdt = torch.complex128 if prec == 8 else torch.complex64
    stream = torch.cuda.current_stream()
    with binding.Context(dims, prec, args.storage, stream=stream) as ctx:
        apply_tune(ctx)
        ctx.tune("reunit_every", args.reunit_every)
        cold = torch.zeros((L, L, L, L, 4, 3, 3), dtype=cdt, device="cuda")
        for i in range(3):
            cold[..., i, i] = 1
        ctx.set_links(cold)
        def cycles(n):                                   # one heat-bath sweep + K overrelaxation sweeps each
            for _ in range(n):
                ctx.thermalize(args.thermal, 1, args.thermal_seed)
                if args.thermal_overrelax > 0:
                    ctx.overrelax(args.thermal_overrelax)

        cycles(5)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        cycles(args.thermal_sweeps - 5)
        e1.record(stream)
        torch.cuda.synchronize()
        ms_sweep = e0.elapsed_time(e1) / ((args.thermal_sweeps - 5) * (1 + args.thermal_overrelax))
        _, theta0, P0 = ctx.measure()
        links = ctx.get_links(torch.empty_like(cold))
        ctx_thermalised = links.clone() if args.mixed else None
        dev0 = 0.0                                        # deviation from SU(3), one t slice at a time (64^4: 9.7 GB)
        eye = torch.eye(3, dtype=cdt, device="cuda")
        for t in range(L):
            sl = links[t]
            dev0 = max(dev0, float((sl @ sl.conj().transpose(-1, -2) - eye).abs().max()))
        tol = 1e-15 if prec == 8 else 1e-12
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        it = ctx.fix(links, args.alpha, tol, args.thermal_max_iter)
        torch.cuda.synchronize()
        sec = time.perf_counter() - t0
        F, theta, P1 = ctx.measure()
        Fh, _ = ctx.history()
        hb_bytes = ctx.algorithmic_bytes(binding.LGF_K_HEATBATH)
        thermalised = ctx_thermalised if args.mixed else None
    mixed = None
    if args.mixed:
        # NEXT-4 ablation, orbit-preserving: an fp32 context finds the accumulated transformation G (tracked, links
        # projected every 20 updates, theta < 1e-12); G is applied to the ORIGINAL fp64 links with
        # lgf_apply_transform (an exact gauge transformation: the plaquette is kept to fp64 rounding); lgf_fix
        # polishes in fp64 to 1e-15.  Timed against the fp64-only fix above.  The float -> double cast of G is a
        # dtype conversion of the exchange buffer.
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        with binding.Context(dims, binding.LGF_FP32, args.storage, stream=stream) as c32:
            c32.tune("reunit_every", 20)
            c32.track_transform(True)
            it32 = c32.fix(thermalised.to(torch.complex64), args.alpha, 1e-12, args.thermal_max_iter)
            G32 = c32.get_transform(torch.empty((L, L, L, L, 3, 3), dtype=torch.complex64, device="cuda"))
        with binding.Context(dims, binding.LGF_FP64, args.storage, stream=stream) as c64:
            c64.set_links(thermalised)
            c64.apply_transform(G32.to(torch.complex128))
            l64 = c64.get_links(torch.empty_like(thermalised))
            it64 = c64.fix(l64, args.alpha, 1e-15, args.thermal_max_iter)
            torch.cuda.synchronize()
            sec_mixed = time.perf_counter() - t0
            Fm, thm, Pm = c64.measure()
        mixed = {"iterations_fp32": it32, "iterations_fp64_polish": it64, "seconds": sec_mixed, "F_final": Fm,
                 "theta_final": thm, "plaquette_after": Pm, "plaquette_drift": abs(Pm - P0),
                 "speedup_vs_fp64_only": sec / sec_mixed}
    peak, _ = measured_peak()
    print(json.dumps({
        "mode": "thermal", "beta": args.thermal, "lattice": "x".join([str(L)] * 4), "precision": args.precision,
        "link_storage": args.storage, "tune": dict(TUNE), "alpha": args.alpha, "reunit_every": args.reunit_every,
        "heatbath_sweeps": args.thermal_sweeps, "overrelax_per_heatbath": args.thermal_overrelax,
        "seed": args.thermal_seed, "heatbath_ms_per_sweep": ms_sweep,
        "heatbath_algorithmic_gbs": hb_bytes / (ms_sweep * 1e-3) / 1e9, "heatbath_frac_of_peak": hb_bytes / (ms_sweep * 1e-3) / 1e9 / peak,
        "plaquette_thermalised": P0, "su3_deviation_thermalised": dev0, "theta_before": theta0,
        "iterations_to_tol": it, "tol": tol, "seconds_to_fix": sec, "ms_per_iteration": 1e3 * sec / max(it, 1),
        "F_final": F, "theta_final": theta, "plaquette_after_fix": P1, "plaquette_drift": abs(P1 - P0),
        "F_min_step": float(np.min(np.diff(Fh))) if len(Fh) > 1 else None, "mixed_precision": mixed,
        "paper_table3": "32^4 dp, C2070: 765-10427 iterations, 61.1 ms/iteration (12-real tex) -- other hardware, context"}),
        flush=True)
    return 0


def run_shard(args):
    """--shard K: ONE configuration sharded over ranks (t-slabs, paper_1206_0675_b200/slab.py).
    Under torchrun (WORLD_SIZE = N > 1) the ranks are the processes and the exchanges go over NCCL: strong scaling,
    value = iterations/s of the one configuration, max-over-ranks device time.  In a single process K ranks are
    emulated one after the other on the one GPU (exchanges = device copies): the time is then the SUM of the K
    ranks' kernel times plus the copies -- a per-rank cost figure, NOT a scaling measurement; the NVLink time is a
    model from the bytes each rank sends (stated as such).  Prints one JSON line of its own; not the contract line."""
    import torch

    from paper_1206_0675_b200 import binding, inputs, slab

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: liblgf has no CPU path")
    torch.cuda.set_device(local)
    binding.load()
    dist = None
    if world > 1:
        import torch.distributed as dist  # noqa: PLC0415

        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        ex, nranks, mode = slab.DistExchange(dist), world, "nccl"
    else:
        ex, nranks, mode = slab.LocalExchange(args.shard), args.shard, "emulated on one GPU, ranks in turn"
    cfg = inputs.CONFIGS[args.workload]
    dims = cfg["dims"]
    V = int(np.prod(dims))
    prec = PREC[args.precision]
    if cfg["kind"] == "hot":
        U0 = inputs.hot_config_torch(dims, cfg["seed"], device="cuda")
    else:
        U0 = torch.from_numpy(inputs.make_config(args.workload)).cuda()
    U0 = torch.view_as_real(U0.to(torch.complex128 if prec == 8 else torch.complex64)).contiguous()
    fx = slab.SlabFixer(dims, prec, args.storage, ex)
    fx.set_links_global(U0)
    del U0
    fx.iterate(ALPHA, args.warmup)
    n0 = fx.launch_count()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    fx.iterate(ALPHA, args.steps)
    b.record()
    torch.cuda.synchronize()
    ms = ensemble.max_over_ranks(dist, a.elapsed_time(b), torch.device("cuda", local)) / args.steps
    F, theta = fx.measure()
    sent = fx.exchanged_bytes / args.steps
    if rank == 0:
        line = {"metric": METRIC, "value": 1e3 / ms, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms, "higher_is_better": True, "scaling": "strong" if world > 1 else "none (emulation)",
                "dtype": "f64" if prec == 8 else "f32", "data": "synthetic",
                "config": {"workload": workload_name(args.workload, dims), "precision": args.precision,
                           "link_storage": args.storage, "alpha": ALPHA, "sites": V,
                           "parallelism": "one configuration in %d t-slabs (%s)" % (nranks, mode)},
                "slab": {"ranks": nranks, "sites_per_rank": V // nranks, "sent_bytes_per_rank_per_iteration": sent,
                         "ms_per_rank_kernels_and_copies": ms / (nranks if world == 1 else 1),
                         "launches_per_iteration": (fx.launch_count() - n0) / args.steps,
                         "nvlink_model_ms": sent / 900e9 * 1e3,
                         "nvlink_model": "sent bytes / 900 GB/s per direction per GPU (B200 NVLink 5); not measured"},
                "state_after_timing": {"F": F, "theta": theta}}
        print(json.dumps(line), flush=True)
    fx.destroy()
    if dist is not None:
        dist.destroy_process_group()
    return 0


def workload_name(key, dims):
    from paper_1206_0675_b200 import inputs

    c = inputs.CONFIGS[key]
    what = "hot start (Haar-random links)" if c["kind"] == "hot" else "smooth eps=%g with Haar h(x)" % c["eps"]
    return "%s: %s periodic SU(3) lattice, %s, seed %d" % (key, "x".join(str(v) for v in dims), what, c["seed"])


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="C3", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--precision", default="fp64", choices=["fp64", "fp32"])
    ap.add_argument("--storage", type=int, default=18, choices=[18, 12])
    ap.add_argument("--no-variants", action="store_true", help="time only the headline variant")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cpu-budget", type=float, default=20.0)
    ap.add_argument("--reference-budget", type=float, default=240.0)
    ap.add_argument("--tune", default="", metavar="KEY=VALUE[,KEY=VALUE]",
                    help="lgf_tune overrides for every context (ablations; the default line uses none)")
    ap.add_argument("--thermal", type=float, default=None, metavar="BETA",
                    help="thermalise a cold 32^4 lattice at BETA and gauge-fix it (own JSON line, not the contract line)")
    ap.add_argument("--thermal-size", type=int, default=32, choices=[8, 16, 32, 64], help="lattice extent L of --thermal (L^4)")
    ap.add_argument("--thermal-sweeps", type=int, default=300)
    ap.add_argument("--thermal-seed", type=int, default=1234)
    ap.add_argument("--thermal-overrelax", type=int, default=0, help="overrelaxation sweeps after each heat-bath sweep")
    ap.add_argument("--reunit-every", type=int, default=0)
    ap.add_argument("--alpha", type=float, default=ALPHA, help="step size of the --thermal fix (the paper uses 0.08)")
    ap.add_argument("--thermal-max-iter", type=int, default=200000)
    ap.add_argument("--shard", type=int, default=0, metavar="K",
                    help="ONE configuration sharded over t-slabs: K emulated ranks in a single process; under torchrun the "
                         "ranks are the processes (any K > 0)")
    ap.add_argument("--sustained-seconds", type=float, default=5.0,
                    help="also run the step back to back for this long (device time) and report it as `sustained` (0 = skip)")
    ap.add_argument("--reduce-ncu", default=None, metavar="CSV",
                    help="turn an ncu --csv launch list of this script (dram bytes + duration metrics) into profiles/*_traffic.csv rows")
    ap.add_argument("--mixed", action="store_true", help="--thermal (fp64 only): also time fp32 iterations + fp64 polish")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    for kv in [x for x in args.tune.split(",") if x]:
        k, v = kv.split("=")
        TUNE[k.strip()] = int(v)
    if args.reduce_ncu:
        return reduce_ncu(args)
    if args.impl == "reference":
        return run_reference(args)
    if args.thermal is not None:
        return run_thermal(args)
    if args.shard > 0:
        return run_shard(args)

    import torch

    from paper_1206_0675_b200 import binding, inputs

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: liblgf has no CPU path")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist  # noqa: PLC0415

        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    binding.load()

    cfg = inputs.CONFIGS[args.workload]
    dims = cfg["dims"]
    V = int(np.prod(dims))
    member = ensemble.member_indices(world, rank, world)[0]      # replicas: one ensemble member per GPU
    if cfg["kind"] == "hot":
        # 64^4 hot start: the torch back end of the same counter-based streams (seconds on the GPU instead of
        # minutes of numpy QR for 67 M links), brought to the host like every other input
        seed = cfg["seed"] + 7919 * ensemble.member_seed_offset(member)
        U0 = inputs.hot_config_torch(dims, seed, device="cuda").cpu().numpy()
        torch.cuda.empty_cache()
    else:
        U0 = inputs.make_config(args.workload, seed_offset=ensemble.member_seed_offset(member))

    sampler = ClockSampler(physical_gpu_index(local))
    head = time_variant(binding, torch, U0, dims, args.precision, args.storage, args.steps, args.warmup, dist, sampler)
    value = world * args.steps / (head["ms_total"] * 1e-3)
    peak, peak_src = measured_peak()

    # dominant kernel class of the iteration -> roofline object
    hot = {k: v for k, v in head["kernels"].items() if k in ("delta", "fft", "update", "gbuild")}
    dom = max(hot, key=lambda k: hot[k]["ms_per_step"])
    dk = hot[dom]
    bytes_per_launch = dk["algorithmic_bytes_per_step"] / dk["launches_per_step"]
    achieved = bytes_per_launch / (dk["avg_launch_us"] * 1e-6) / 1e9
    caps, stale = captured_traffic(args.workload, args.precision, args.storage, head["kernel_names"])
    cap = (caps.get(dom) or [None])[0]
    # whole iteration in REAL DRAM bytes: the ncu capture of every kernel of one iteration, summed
    dram_iter = sum(r["bytes"] * r["launches_per_step"] for k in hot for r in caps.get(k, [])) if caps else None
    complete = bool(caps) and all(k in caps for k in hot)
    yard = head["iter_bytes"] / (head["ms_per_step"] * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS,
                "traffic": cap["bytes"] if cap else None,
                "traffic_source": cap["source"] if cap else None, "traffic_kernel": cap["kernel"] if cap else None,
                "stale_captures_refused": stale[:8], "peak_source": peak_src,
                "algorithmic_bytes_per_launch": bytes_per_launch, "avg_launch_us": dk["avg_launch_us"],
                "launched_kernels": head["kernel_names"],
                "iteration": {"yardstick_bytes": head["iter_bytes"], "yardstick_rate": yard, "yardstick_frac": yard / peak,
                              "yardstick_note": "SURVEY 8(d) UNFUSED budget (12 n_l + 64 reals/site) / time: an effective rate, "
                                                "not DRAM traffic -- the fused path moves fewer bytes",
                              "dram_bytes": dram_iter if complete else None,
                              "dram_rate": dram_iter / (head["ms_per_step"] * 1e-3) / 1e9 if complete else None,
                              "dram_frac": dram_iter / (head["ms_per_step"] * 1e-3) / 1e9 / peak if complete else None,
                              "dram_frac_of_nominal_8TBs": dram_iter / (head["ms_per_step"] * 1e-3) / 1e9 / NOMINAL_HBM_GBS if complete else None,
                              "dram_note": "sum over the iteration's kernels of ncu dram__bytes_read + write per launch "
                                           "(committed capture, cold L2 per kernel) / this run's ms_per_step"},
                "kernels": {k: {"ms_per_step": round(v["ms_per_step"], 6), "launches_per_step": v["launches_per_step"],
                                "algorithmic_gbs": v["gbs"], "algorithmic_frac": v["gbs"] / peak,
                                "dram_bytes_per_step": (sum(r["bytes"] * r["launches_per_step"] for r in caps[k]) if k in caps else None)}
                            for k, v in hot.items()}}

    variants = {}
    if not args.no_variants:
        for pn in ("fp64", "fp32"):
            for st in (18, 12):
                if pn == args.precision and st == args.storage:
                    r = head
                else:
                    r = time_variant(binding, torch, U0, dims, pn, st, args.steps, args.warmup, dist)
                gbs = r["iter_bytes"] / (r["ms_per_step"] * 1e-3) / 1e9
                vcaps, _ = captured_traffic(args.workload, pn, st, r["kernel_names"])
                vhot = [k for k in r["kernels"] if k in ("delta", "fft", "update", "gbuild")]
                vdram = (sum(x["bytes"] * x["launches_per_step"] for k in vhot for x in vcaps[k])
                         if vcaps and all(k in vcaps for k in vhot) else None)
                variants["%s/%d" % (pn, st)] = {"iterations_per_s": world * 1e3 / r["ms_per_step"],
                                                "site_updates_per_s": world * V * 1e3 / r["ms_per_step"],
                                                "ms_per_step": r["ms_per_step"], "yardstick_gbs": gbs,
                                                "yardstick_frac": gbs / peak,
                                                "dram_bytes_per_step": vdram,
                                                "dram_frac": vdram / (r["ms_per_step"] * 1e-3) / 1e9 / peak if vdram else None,
                                                "update_ms": r["kernels"].get("update", {}).get("ms_per_step"),
                                                "fft_ms": r["kernels"].get("fft", {}).get("ms_per_step")}

    e2e = None
    if not args.no_e2e:
        tol = 1e-15 if args.precision == "fp64" else 1e-12
        # a hot start is not run to convergence: BASELINE.json's C5 is a fixed 200 iterations
        max_iter = 200 if cfg["kind"] == "hot" else 5000
        r = time_e2e(binding, torch, U0, dims, args.precision, args.storage, tol, max_iter, dist)
        its = max(1, r["iterations"])
        e2e = {"value": world * its / (r["ms"] * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": r["bytes_each_way"] / its, "d2h_bytes_per_step": r["bytes_each_way"] / its,
               "call": "lgf_fix_host(pinned host links, alpha=0.08, tol=%g, max_iter=%d): H2D + %d iterations + D2H in %.1f ms"
                       % (tol, max_iter, r["iterations"], r["ms"]), "final_theta": r["theta"]}

    sustained = None
    if world == 1 and args.sustained_seconds > 0:
        sustained = time_sustained(binding, torch, U0, dims, args.precision, args.storage, args.sustained_seconds,
                                   head["ms_per_step"], physical_gpu_index(local))
        if roofline["iteration"]["dram_bytes"]:
            sustained["dram_frac"] = roofline["iteration"]["dram_bytes"] / (sustained["ms_per_step"] * 1e-3) / 1e9 / peak

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(U0, dims, args.cpu_budget)

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": head["ms_per_step"], "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64" if args.precision == "fp64" else "f32", "data": "synthetic",
                "config": {"workload": workload_name(args.workload, dims), "precision": args.precision,
                           "tune": dict(TUNE), "link_storage": args.storage, "alpha": ALPHA, "sites": V, "parallelism": "replicas x%d" % world,
                           "l2": "inputs larger than L2: one step streams %.0f MB of links and fields"
                                 % (head["iter_bytes"] / 1e6)},
                "site_updates_per_s": value * V, "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e,
                "sustained": sustained,
                "gpu_launches": head["launches"], "clocks": sampler.summary(), "remeasured": head.get("remeasured"),
                "variants": variants,
                "state_after_timing": {"F": head["F"], "theta": head["theta"], "plaquette": head["plaquette"]}}
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
