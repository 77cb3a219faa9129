#!/usr/bin/env python
"""bench.py -- throughput of the StePS cylindrical hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--n 1048576] [--precision fp64|mixed] [--n-cut 5]

A "step" is one KDK leapfrog step of Eq. 11 over the whole particle set: background term,
kick + drift, pack + wrap, the all-pairs image sum (Eq. 8), reduction, background term, kick --
i.e. every row of the hot-path table, one force evaluation per step.  The workload is
BASELINE.json configs[3] (N = 1 048 576, LCDM comoving load, L = 100 Mpc/h, n_cut = 5), the
configuration the metric "pair interactions/s (N=1M, periodic-z, fp64)" is quoted on.

Prints ONE JSON line.  `value` = ordered pairs N(N-1) per second of whole-step time, inputs
resident in HBM.  `e2e` = the same through steps_cyl_kdk_step_host with pinned HOST buffers
(host->device and device->host copies inside the timed region).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "pair interactions/s (N=1M, periodic-z, fp64); % of B200 FP64 FMA peak"
NOMINAL_FP64_LANES_PER_SM = 64
NOMINAL_FP32_LANES_PER_SM = 128
NOMINAL_XU_LANES_PER_SM = 16
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "ncu_dram_traffic.csv")


def pipe_counts(kernel, n_cut):
    """Pipe instructions / flops per ORDERED pair interaction of `kernel`, from the SASS tally build.py wrote
    beside the library (paper_2602_20787_b200/sassmix.py); never a literal in this file."""
    from paper_2602_20787_b200 import build, sassmix
    return sassmix.per_interaction(sassmix.load(build.SASSMIX), kernel, n_cut)


def ncu_traffic(kernel, n, n_cut):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` at (n, n_cut), from the committed
    `ncu --set full` rows in profiles/ncu_dram_traffic.csv (None if that configuration was never captured)."""
    import csv
    if not os.path.exists(TRAFFIC_CSV):
        return None, None
    with open(TRAFFIC_CSV) as f:
        for row in csv.DictReader(l for l in f if not l.startswith("#")):
            if row["kernel"] == kernel and int(row["n"]) == n and int(row["n_cut"]) in (n_cut, -1):
                return float(row["dram_bytes_read"]) + float(row["dram_bytes_write"]), row["source"]
    return None, None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(prefix="steps_clocks_", suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in open(self.path):
            f = [t.strip() for t in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        os.unlink(self.path)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)),
                       power_w_max=float(max(pw)), reasons=sorted(reasons), samples=len(sm))
        return out


def max_over_ranks(seconds, dist=None, device=None):
    """Job time = the slowest rank's device time (all ranks call this; identity without a group)."""
    if dist is None:
        return float(seconds)
    import torch
    t = torch.tensor([float(seconds)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_throughput(pairs_per_rank_step, steps, world, seconds_max):
    """Replicas only: whole-job pair interactions/s = all ranks' units / slowest rank."""
    return world * pairs_per_rank_step * steps / seconds_max


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "sm_max_mhz": 1965.0}, "fallback"


def cosmo_schedule(w, n_steps_total):
    """(a_n, H_n, a_np1, H_np1) for consecutive KDK steps, from the library's own RK4."""
    from paper_2602_20787_b200 import binding as b
    c = w.cosmo
    a = c["a_init"]
    _, H = b.friedmann_step(a, 0.0, c["H0"], c["Om"], c["Or"], c["Ok"], c["OL"])
    sched = []
    for _ in range(n_steps_total):
        a1, H1 = b.friedmann_step(a, c["dt"], c["H0"], c["Om"], c["Or"], c["Ok"], c["OL"])
        sched.append((a, H, a1, H1))
        a, H = a1, H1
    return sched


def oracle_sample(w, seconds, n_cut):
    """Time the oracle, as it stands, on a bounded seeded sample of targets x all N sources."""
    import oracle
    from paper_2602_20787_b200 import workloads
    oracle.build()
    cores = oracle.max_threads()
    probe = workloads.sample_targets(w.n, 2 * cores, seed=99)
    t0 = time.perf_counter()
    oracle.accel(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, n_cut, targets=probe)
    per_target = (time.perf_counter() - t0) / len(probe)
    T = int(max(cores, min(w.n, seconds / max(per_target, 1e-9))))
    T -= T % cores or 0
    T = max(T, cores)
    idx = workloads.sample_targets(w.n, T, seed=100)
    return idx, cores


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores, same workload / metric / unit."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    from paper_2602_20787_b200 import workloads
    w = workloads.make(3, n=args.n)
    idx, cores = oracle_sample(w, args.ref_seconds, args.n_cut)
    times = []
    for s in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        oracle.accel(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, args.n_cut, targets=idx)
        dt = time.perf_counter() - t0
        if s >= args.warmup:
            times.append(dt)
    t = float(np.mean(times))
    value = len(idx) * (w.n - 1) / t
    sample = ("oracle.accel (force evaluation only) on %d seeded targets x all %d sources per step, "
              "n_cut=%d" % (len(idx), w.n, args.n_cut))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "pairs/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": "BASELINE configs[3]: N=%d LCDM comoving load, L=100, n_cut=%d, "
                               "bounded target sample" % (w.n, args.n_cut)},
        "image_terms_per_s": value * 2 * args.n_cut,
        "cpu_baseline": {"value": value, "unit": "pairs/s", "cores": cores, "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": "pairs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def make_ctx(b, w, local, args, precision, periodic, tab_fp32, interp, flags):
    table = periodic == "table"
    # table mode sums all images (N_cut -> inf), so its consistent background term is Eq. 10
    return b.StepsCyl(n=w.n, Lz=w.Lz, G=w.G, n_cut=args.n_cut,
                      precision=b.PREC_MIXED if precision == "mixed" else b.PREC_FP64,
                      background=b.BG_INFINITE if table else b.BG_FINITE,
                      R_sim=w.R_sim, rho0=w.rho0, device=local,
                      periodic_mode=b.PERIODIC_EWALD_TABLE if table else b.PERIODIC_IMAGES,
                      tab_fp32=1 if (table and tab_fp32) else 0,
                      interp=b.INTERP_TSC if (table and interp == "tsc") else b.INTERP_CIC, flags=flags)


def roofline_of(ctx, n, n_cut, t_pair, sm_count, sm_max, table):
    """Roofline record of the all-pairs kernel `ctx` launches: numerator from the SASS tally of the built
    library, duration from the CUDA events the library records around that launch."""
    kernel = ctx.pair_kernel_name()
    cnt, how = pipe_counts(kernel, n_cut)
    # the mixed image kernel runs two forms of its ring pass (pair_mixed_sym.cuh: SIMPLE where the Morton-ordered
    # groups are far apart); their tallies are weighted with the pass counts the kernel itself keeps
    simple_frac = None
    n_simple, n_pass = ctx.pass_stats()
    if n_pass > 0 and how == "counted":
        from paper_2602_20787_b200 import build, sassmix
        var = sassmix.load(build.SASSMIX)["kernels"][kernel]["variants"]
        if len(var) >= 2:
            simple_frac = n_simple / n_pass
            cnt = {k: simple_frac * var[1]["per_interaction"][k] + (1.0 - simple_frac) * var[0]["per_interaction"][k]
                   for k in cnt}
            how = "two loop forms weighted by the kernel's own pass counts"
    pairs = float(n) * float(n - 1)
    is_mixed = "mixed" in kernel
    lanes = NOMINAL_FP32_LANES_PER_SM if is_mixed else NOMINAL_FP64_LANES_PER_SM
    instr = cnt["fp32_ops"] if is_mixed else cnt["fp64_instr"]
    flops = cnt["fp32_flops"] if is_mixed else cnt["fp64_flops"]
    nominal_tflops = sm_count * lanes * 2 * sm_max * 1e6 / 1e12
    achieved_tflops = flops * pairs / t_pair / 1e12
    traffic, traffic_src = ncu_traffic(kernel, n, -1 if table else n_cut)
    r = {
        "bound": "alu", "kernel": kernel, "achieved": achieved_tflops, "peak": nominal_tflops,
        "unit": "TFLOP/s", "frac": achieved_tflops / nominal_tflops,
        "traffic": traffic, "traffic_source": traffic_src,
        "traffic_unit": "bytes per launch (ncu dram__bytes_read.sum + dram__bytes_write.sum); the bound is the "
                        "%s pipe, not HBM" % ("FP32" if is_mixed else "FP64"),
        "algorithmic_bytes": 72.0 * n,
        "peak_kind": "nominal %s FMA: %d SMs x %d lanes x 2 flop x %.0f MHz (DESIGN.md)"
                     % ("FP32" if is_mixed else "FP64", sm_count, lanes, sm_max),
        "counting": "SASS tally of the built library (sassmix.py, %s); FMA = 2 flop, ADD/MUL = 1" % how,
        "flops_per_pair_interaction": flops, "pipe_instr_per_pair_interaction": instr,
        "pipe_util_vs_nominal": instr * pairs / t_pair / (nominal_tflops * 1e12 / 2),
        "kernel_ms": 1e3 * t_pair,
    }
    if simple_frac is not None:
        r["simple_pass_fraction"] = simple_frac
    if is_mixed or cnt["fp32_ops"] > 0:
        xu_peak = sm_count * NOMINAL_XU_LANES_PER_SM * sm_max * 1e6
        r["xu_pipe_util_vs_nominal"] = (cnt["mufu"] + cnt["conv"]) * pairs / t_pair / xu_peak
    if not np.isfinite(t_pair):      # STEPS_FLAG_GRAPH: the kernel is not timed on its own inside the graph
        for key in ("achieved", "frac", "pipe_util_vs_nominal", "kernel_ms", "xu_pipe_util_vs_nominal"):
            if key in r:
                r[key] = None
    return r


def run_ours(args):
    import torch
    from paper_2602_20787_b200 import binding as b
    from paper_2602_20787_b200 import build, workloads
    build.build()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; there is no CPU fallback for the product path")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # replicas only: every rank integrates its own particle set
    w = workloads.make(3, n=args.n, seed=3 + rank)
    n = w.n
    table = args.periodic == "table"
    flags = ((b.FLAG_DETERMINISTIC if args.deterministic else 0) | (b.FLAG_ORDERED_PAIRS if args.ordered else 0)
             | (b.FLAG_FAR_ORDER2 if args.far_order2 else 0) | (b.FLAG_GRAPH if args.graph else 0))
    names = ("x", "y", "z", "vx", "vy", "vz", "m", "h")
    host0 = {k: np.ascontiguousarray(getattr(w, k), dtype=np.float64) for k in names}
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2
    pairs_per_step = float(n) * float(n - 1)
    sm_count = torch.cuda.get_device_properties(local).multi_processor_count
    peaks, peaks_kind = load_peaks()
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))

    def measure(precision, periodic, tab_fp32, interp, flags, steps, warmup, e2e_steps, sample_clocks):
        """One mode: fresh context and particle state; W warm-up + K timed KDK steps (device time, L2 flushed
        between steps), then the same step through the host-pointer entry point."""
        ctx = make_ctx(b, w, local, args, precision, periodic, tab_fp32, interp, flags)
        host = {k: torch.from_numpy(host0[k].copy()).pin_memory() for k in names}
        dev = {k: host[k].cuda(non_blocking=True) for k in names}
        g = [torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3)]
        ctx.accel(dev["x"], dev["y"], dev["z"], dev["m"], dev["h"], *g)       # g(x_0), untimed
        ctx.check()
        hg = [t.cpu().pin_memory() for t in g]
        sched = cosmo_schedule(w, warmup + steps + e2e_steps + 2)

        def step(k):
            flush.zero_()
            ctx.kdk_step(*[dev[q] for q in names], *g, *sched[k], w.cosmo["dt"])

        for k in range(warmup):
            step(k)
        barrier()
        sampler = ClockSampler(local)
        if rank == 0 and sample_clocks:
            sampler.start()
        # device time of each step: a CUDA event pair around the step on the launching stream, the L2 flush between
        # steps outside it.  Large N: the pair kernel's own events are read after every step (a host sync that costs
        # nothing against seconds of kernel); small N: no host sync inside the loop, the last step's pair time is read.
        graph = bool(flags & b.FLAG_GRAPH)
        sync_each = n >= 100000 and not graph
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        pair_ms = []
        launches0 = ctx.launch_count()                # kernels of this library launched inside the timed steps
        for k in range(steps):
            flush.zero_()
            evs[k][0].record()
            ctx.kdk_step(*[dev[q] for q in names], *g, *sched[warmup + k], w.cosmo["dt"])
            evs[k][1].record()
            if sync_each:
                pair_ms.append(ctx.last_pair_kernel_ms())          # waits for that launch's end event
        barrier()
        launches_per_step = (ctx.launch_count() - launches0) / max(steps, 1)
        if not sync_each and not graph:
            pair_ms.append(ctx.last_pair_kernel_ms())
        clocks = sampler.stop() if (rank == 0 and sample_clocks) else {}
        ctx.check()
        step_ms = [e0.elapsed_time(e1) for e0, e1 in evs]
        t_dev = max_over_ranks(float(np.sum(step_ms)) * 1e-3, dist, "cuda")
        if not pair_ms:
            pair_ms = [float("nan")]
        out = {"ctx": ctx, "t_dev": t_dev, "t_pair": float(np.mean(pair_ms)) * 1e-3, "clocks": clocks,
               "launches_per_step": launches_per_step, "value": replica_throughput(pairs_per_step, steps, world, t_dev),
               "e2e_value": None, "step_ms_min": float(np.min(step_ms)), "step_ms_median": float(np.median(step_ms))}
        if e2e_steps:
            # end to end: pinned host buffers through steps_cyl_kdk_step_host, copies inside the timing
            hs = [host[q] for q in names] + hg
            ctx.kdk_step_host(*hs, *sched[warmup + steps], w.cosmo["dt"])
            barrier()
            t0 = time.perf_counter()
            for k in range(e2e_steps):
                ctx.kdk_step_host(*hs, *sched[warmup + steps + 1 + k], w.cosmo["dt"])
            torch.cuda.synchronize()
            out["e2e_value"] = replica_throughput(pairs_per_step, e2e_steps, world,
                                                  max_over_ranks(time.perf_counter() - t0, dist, "cuda"))
            assert all(bool(torch.isfinite(t).all()) for t in hg)
        return out

    main = measure(args.precision, args.periodic, args.table_fp32, args.interp, flags, args.steps, args.warmup,
                   args.steps, True)
    ctx = main["ctx"]
    dfma_per_s = ctx.fp64_peak(200.0) if rank == 0 else 0.0

    # the other modes north_star names, in the same run (rank 0's line carries them; all ranks run them so that the
    # barriers match): mixed precision against the FP32 peak, and the Ewald-table mode of Eq. 12-17
    subs = {}
    default_line = (args.precision == "fp64" and not table and flags == 0)
    if default_line and not args.no_sub:
        k_sub, w_sub = min(args.steps, 3), 3
        for key, (prec, per, f32) in (("mixed", ("mixed", "images", False)),
                                      ("table", ("fp64", "table", False)),
                                      ("table_fp32", ("fp64", "table", True)),
                                      ("table_mixed", ("mixed", "table", True))):
            subs[key] = measure(prec, per, f32, "cic", 0, k_sub, w_sub, 0, True)
            subs[key]["steps"], subs[key]["warmup"] = k_sub, w_sub

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    t_dev, t_pair = main["t_dev"], main["t_pair"]
    roofline = roofline_of(ctx, n, args.n_cut, t_pair, sm_count, sm_max, table)
    roofline["kernel_share_of_step"] = t_pair * args.steps / t_dev if np.isfinite(t_pair) else None
    if "mixed" not in roofline["kernel"] and np.isfinite(t_pair):
        roofline["measured_dfma_tflops"] = 2 * dfma_per_s / 1e12
        roofline["pipe_util_vs_measured_dfma"] = (roofline["pipe_instr_per_pair_interaction"] * pairs_per_step
                                                  / t_pair / dfma_per_s)
    sub_records = {}
    for key, m in subs.items():
        is_tab = key.startswith("table")
        r = roofline_of(m["ctx"], n, args.n_cut, m["t_pair"], sm_count, sm_max, is_tab)
        sub_records[key] = {
            "value": m["value"], "unit": "pairs/s", "steps": m["steps"], "warmup": m["warmup"],
            "ms_per_step": 1e3 * m["t_dev"] / m["steps"], "seconds_per_force_evaluation": m["t_pair"],
            "dtype": {"mixed": "f32 pair terms, f64 accumulation", "table": "f64",
                      "table_fp32": "f64 pair terms, f32 table nodes and interpolation",
                      "table_mixed": "f32 pair terms and table, f64 accumulation"}[key],
            "periodic": "Ewald table 144x128 CIC, rho_max=5L, all images (Eq. 12-17)" if is_tab
                        else "n_cut=%d (%d images/pair)" % (args.n_cut, 2 * args.n_cut),
            "roofline": r, "clocks": m["clocks"], "gpu_launches": int(round(m["launches_per_step"] * m["steps"])),
        }
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        import oracle
        idx, cores = oracle_sample(w, args.ref_seconds, args.n_cut)
        t0 = time.perf_counter()
        oracle.accel(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, args.n_cut, targets=idx)
        tc = time.perf_counter() - t0
        cpu = {"value": len(idx) * (n - 1) / tc, "unit": "pairs/s", "cores": cores, "kind": "oracle",
               "sample": "oracle.accel on %d seeded targets x all %d sources (force evaluation only), "
                         "%.1f s" % (len(idx), n, tc)}
    mixed_prec = args.precision == "mixed"
    periodic_desc = ("Ewald table 144x128 %s%s, (n_max,m_max)=(5,12), rho_max=5L, background Eq. 10"
                     % (args.interp.upper(), " (float nodes in shared memory)" if (args.table_fp32 or mixed_prec) else "") if table
                     else "n_cut=%d (%d images/pair), background Eq. 9" % (args.n_cut, 2 * args.n_cut))
    if mixed_prec:
        dtype = "f32"            # pair terms in float (hi/lo separations), accumulation in double
    elif table and args.table_fp32:
        dtype = "f64+f32"        # pair terms in double, table nodes and their interpolation in float
    else:
        dtype = "f64"
    line = {
        "metric": METRIC, "value": main["value"], "unit": "pairs/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t_dev / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": dtype, "data": "synthetic",
        "config": {"workload": "BASELINE configs[3]: N=%d LCDM comoving KDK step (Om=0.3, OL=0.7, "
                               "a 0.02->0.025), L=100 Mpc/h, r_max=1000, %s" % (n, periodic_desc),
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": "256 MiB buffer written between steps (L2 flush), outside the per-step event pairs",
                   "graph": bool(args.graph)},
        "image_terms_per_s": None if table else main["value"] * 2 * args.n_cut,
        "seconds_per_force_evaluation": t_pair if np.isfinite(t_pair) else None, "step_ms_min": main["step_ms_min"],
        "step_ms_median": main["step_ms_median"],
        "roofline": roofline, "cpu_baseline": cpu, "clocks": main["clocks"],
        "e2e": {"value": main["e2e_value"], "unit": "pairs/s", "h2d_bytes_per_step": 11 * 8 * n,
                "d2h_bytes_per_step": 9 * 8 * n},
        "gpu_launches": int(round(main["launches_per_step"] * args.steps)),
        "peaks_file": peaks_kind,
    }
    line.update(sub_records)          # "mixed", "table", "table_fp32", "table_mixed" (default line only)
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=1048576)
    ap.add_argument("--n-cut", type=int, default=5)
    ap.add_argument("--precision", default="fp64", choices=["fp64", "mixed"])
    ap.add_argument("--periodic", default="images", choices=["images", "table"],
                    help="images: truncated image sum of Eq. 8 (the metric's mode); table: Eq. 12-17")
    ap.add_argument("--ref-seconds", type=float, default=12.0,
                    help="CPU seconds of oracle work per sample / reference step")
    ap.add_argument("--far-order2", action="store_true",
                    help="fp64 images mode: STEPS_FLAG_FAR_ORDER2 (far images refined to first order only)")
    ap.add_argument("--interp", default="cic", choices=["cic", "tsc"],
                    help="--periodic table: cloud-in-cell (4 nodes) or triangular-shaped cloud (9 nodes)")
    ap.add_argument("--table-fp32", action="store_true",
                    help="--periodic table: float table held in shared memory (tab_fp32 = 1)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sub", action="store_true",
                    help="default line only: skip the mixed / table sub-records measured in the same run")
    ap.add_argument("--graph", action="store_true",
                    help="STEPS_FLAG_GRAPH: the KDK step replayed as one captured CUDA graph")
    ap.add_argument("--deterministic", action="store_true",
                    help="STEPS_FLAG_DETERMINISTIC: bit-reproducible (fp64: round-scheduled symmetric kernel)")
    ap.add_argument("--ordered", action="store_true",
                    help="STEPS_FLAG_ORDERED_PAIRS: ordered-pair kernels with fixed-order reduction")
    args = ap.parse_args()
    if args.warmup < 3:
        print("bench.py: note: fewer than 3 warm-up steps", file=sys.stderr)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
