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

# Instruction mix of the pair kernels' inner loops at N_cut = 5 (10 image terms per pair), counted
# in the SASS of the shipped library (cuobjdump -sass).  "unit" says what one
# loop iteration covers: the symmetric kernel evaluates an UNORDERED pair (two interactions).
KERNEL_MIX = {
    # default fp64 kernel, pair_fp64_sym_kernel<5>: one unordered pair per iteration
    "fp64": dict(kernel="pair_fp64_sym_kernel<5>", interactions=2, dfma=53, dmul=33, dadd=22, dsetp=0,
                 per_image=(9.5, 14.0)),
    # STEPS_FLAG_DETERMINISTIC, pair_fp64_round_kernel<5>: the same loop, scheduled in conflict-free rounds
    "fp64_det": dict(kernel="pair_fp64_round_kernel<5>", interactions=2, dfma=53, dmul=33, dadd=22, dsetp=0,
                     per_image=(9.5, 14.0)),
    # STEPS_FLAG_ORDERED_PAIRS, pair_fp64_kernel<5,0>: one ordered pair per iteration
    "fp64_ord": dict(kernel="pair_fp64_kernel<5,0>", interactions=1, dfma=49, dmul=32, dadd=22, dsetp=0,
                     per_image=(9.5, 14.0)),
    # --periodic table: pair_table_sym_kernel<CIC, 4, false> (softened nearest image + 4 gathers of double2
    # nodes through L1), one unordered pair per iteration; independent of n_cut
    "table": dict(kernel="pair_table_sym_kernel<CIC>", interactions=2, dfma=23, dmul=13, dadd=17, dsetp=4,
                  per_image=(0.0, 0.0)),
    # --periodic table --table-fp32: pair_table_sym_kernel<CIC, 16, true> (float nodes in shared memory,
    # their weighted sum in fp32: 8 FADD + 6 FFMA per pair, not counted as FP64 work)
    "table_f32": dict(kernel="pair_table_sym_kernel<CIC,fp32 nodes>", interactions=2, dfma=17, dmul=13, dadd=11,
                      dsetp=3, per_image=(0.0, 0.0)),
    # --periodic table --precision mixed: pair_table_mixed_sym_kernel<CIC>, one unordered pair per iteration
    "mixed_table": dict(kernel="pair_table_mixed_sym_kernel<CIC>", interactions=2, ffma=19, fmul=10, fadd=23,
                        mufu=2, f2f=0, dadd=0),
    # default mixed kernel, pair_mixed_sym_kernel<5>: one unordered pair per iteration (FP32-pipe
    # instructions + 10 MUFU.RSQ; conversions and DADDs are outside the per-pair loop)
    # (main loop: 38 FFMA2 + 19 FMUL2 + 16 FADD2 + 20 MUFU per ring step of two unordered pairs; counted
    # here as scalar FP32 operations per unordered pair)
    "mixed": dict(kernel="pair_mixed_sym_kernel<5>", interactions=2, ffma=38, fmul=19, fadd=16, mufu=10,
                  f2f=0, dadd=0),
    # STEPS_FLAG_DETERMINISTIC, pair_mixed_round_kernel<5>: the same loop in conflict-free rounds
    "mixed_det": dict(kernel="pair_mixed_round_kernel<5>", interactions=2, ffma=38, fmul=19, fadd=16, mufu=10,
                      f2f=0, dadd=0),
    # STEPS_FLAG_ORDERED_PAIRS, pair_mixed_kernel<5>: one ordered pair per iteration
    "mixed_ord": dict(kernel="pair_mixed_kernel<5>", interactions=1, ffma=17, fmul=27, fadd=30, mufu=10,
                      f2f=4, dadd=4),
}
METRIC = "pair interactions/s (N=1M, periodic-z, fp64); % of B200 FP64 FMA peak"
NOMINAL_FP64_LANES_PER_SM = 64
NOMINAL_FP32_LANES_PER_SM = 128
NOMINAL_XU_LANES_PER_SM = 16
NCU_DRAM_BYTES_DEFAULT = 78.49e6 + 8.60e6     # pair_fp64_sym_kernel<5>, N = 1 048 576 (algorithmic: 42 MB + 34 MB)


def pipe_counts(mode, n_cut):
    """(pipe instructions, flops) per ORDERED pair interaction for the kernel of `mode`."""
    mix = KERNEL_MIX[mode]
    if mode.startswith("mixed"):
        instr = mix["ffma"] + mix["fmul"] + mix["fadd"]
        flops = 2 * mix["ffma"] + mix["fmul"] + mix["fadd"]
        d = 0 if mode == "mixed_table" else 2 * (n_cut - 5)
        return (instr + 7.5 * d) / mix["interactions"], (flops + 9.0 * d) / mix["interactions"]
    instr = mix["dfma"] + mix["dmul"] + mix["dadd"] + mix["dsetp"]
    flops = 2 * mix["dfma"] + mix["dmul"] + mix["dadd"]
    d = 0 if mode.startswith("table") else 2 * (n_cut - 5)   # extra image terms per pair evaluation
    instr += mix["per_image"][0] * d
    flops += mix["per_image"][1] * d
    return instr / mix["interactions"], flops / mix["interactions"]


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

    prec = b.PREC_MIXED if args.precision == "mixed" else b.PREC_FP64
    # replicas only: every rank integrates its own particle set
    w = workloads.make(3, n=args.n, seed=3 + rank)
    n = w.n
    table = args.periodic == "table"
    # table mode sums all images (N_cut -> inf), so its consistent background term is Eq. 10
    ctx = b.StepsCyl(n=n, Lz=w.Lz, G=w.G, n_cut=args.n_cut, precision=prec,
                     background=b.BG_INFINITE if table else b.BG_FINITE,
                     R_sim=w.R_sim, rho0=w.rho0, device=local,
                     periodic_mode=b.PERIODIC_EWALD_TABLE if table else b.PERIODIC_IMAGES,
                     tab_fp32=1 if (table and args.table_fp32) else 0,
                     interp=b.INTERP_TSC if (table and args.interp == "tsc") else b.INTERP_CIC,
                     flags=(b.FLAG_DETERMINISTIC if args.deterministic else 0)
                     | (b.FLAG_ORDERED_PAIRS if args.ordered else 0)
                     | (b.FLAG_FAR_ORDER2 if args.far_order2 else 0))
    names = ("x", "y", "z", "vx", "vy", "vz", "m", "h")
    host = {k: torch.from_numpy(np.ascontiguousarray(getattr(w, k), dtype=np.float64)).pin_memory()
            for k in names}
    dev = {k: host[k].cuda(non_blocking=True) for k in names}
    g = [torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3)]
    ctx.accel(dev["x"], dev["y"], dev["z"], dev["m"], dev["h"], *g)       # g(x_0), untimed
    ctx.check()
    hg = [t.cpu().pin_memory() for t in g]
    dfma_per_s = ctx.fp64_peak(200.0)
    sched = cosmo_schedule(w, 2 * (args.warmup + args.steps) + 2)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2

    def step(k):
        flush.zero_()
        ctx.kdk_step(*[dev[q] for q in names], *g, *sched[k], w.cosmo["dt"])

    launches0 = ctx.launch_count()
    for k in range(args.warmup):
        step(k)
    launches_per_step = (ctx.launch_count() - launches0) / max(args.warmup, 1)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    pair_ms = []
    ev[0].record()
    for k in range(args.steps):
        step(args.warmup + k)
        pair_ms.append(ctx.last_pair_kernel_ms())          # waits for that launch's end event
    ev[1].record()
    barrier()
    clocks = sampler.stop() if rank == 0 else {}
    ctx.check()
    t_dev = max_over_ranks(ev[0].elapsed_time(ev[1]) * 1e-3, dist, "cuda")
    pairs_per_step = float(n) * float(n - 1)
    value = replica_throughput(pairs_per_step, args.steps, world, t_dev)

    # end to end: pinned host buffers through steps_cyl_kdk_step_host, copies inside the timing
    hs = [host[q] for q in names] + hg
    for k in range(1):
        ctx.kdk_step_host(*hs, *sched[args.warmup + args.steps + k], w.cosmo["dt"])
    barrier()
    t0 = time.perf_counter()
    for k in range(args.steps):
        ctx.kdk_step_host(*hs, *sched[args.warmup + args.steps + 1 + k], w.cosmo["dt"])
    torch.cuda.synchronize()
    e2e_value = replica_throughput(pairs_per_step, args.steps, world,
                                   max_over_ranks(time.perf_counter() - t0, dist, "cuda"))
    assert all(bool(torch.isfinite(t).all()) for t in hg)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    peaks, peaks_kind = load_peaks()
    if table:
        mode = "mixed_table" if prec == b.PREC_MIXED else ("table_f32" if args.table_fp32 else "table")
    else:
        mode = ("mixed" if prec == b.PREC_MIXED else "fp64") + ("_det" if args.deterministic else "")
        if args.ordered:
            mode = "mixed_ord" if prec == b.PREC_MIXED else "fp64_ord"
    instr, flops = pipe_counts(mode, args.n_cut)
    if args.far_order2 and mode == "fp64":              # one DFMA less per far image
        instr -= (2 * args.n_cut - 1) / 2.0
        flops -= (2 * args.n_cut - 1)
    t_pair = float(np.mean(pair_ms)) * 1e-3
    sm_count = torch.cuda.get_device_properties(local).multi_processor_count
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    is_mixed = mode.startswith("mixed")
    lanes = NOMINAL_FP32_LANES_PER_SM if is_mixed else NOMINAL_FP64_LANES_PER_SM
    nominal_tflops = sm_count * lanes * 2 * sm_max * 1e6 / 1e12
    achieved_tflops = flops * pairs_per_step / t_pair / 1e12
    roofline = {
        "bound": "alu", "kernel": KERNEL_MIX[mode]["kernel"].replace("<5", "<%d" % args.n_cut),
        "achieved": achieved_tflops, "peak": nominal_tflops, "unit": "TFLOP/s",
        "frac": achieved_tflops / nominal_tflops,
        # dram__bytes_read.sum + dram__bytes_write.sum of this kernel, one `ncu --set full` capture of the
        # default configuration (profiles/r1_ncu_full_pair_kernels.md); other configurations: not captured
        "traffic": NCU_DRAM_BYTES_DEFAULT if (mode == "fp64" and n == 1048576 and args.n_cut == 5) else None,
        "traffic_unit": "bytes per launch (ncu); the bound is the FP64 pipe, not HBM",
        "peak_kind": "nominal %s FMA: %d SMs x %d lanes x 2 flop x %.0f MHz (DESIGN.md)"
                     % ("FP32" if is_mixed else "FP64", sm_count, lanes, sm_max),
        "flops_per_pair_interaction": flops, "pipe_instr_per_pair_interaction": instr,
        "pipe_util_vs_nominal": instr * pairs_per_step / t_pair / (nominal_tflops * 1e12 / 2),
        "kernel_ms": 1e3 * t_pair, "kernel_share_of_step": t_pair * args.steps / t_dev,
    }
    if table and args.deterministic:                       # same loops, scheduled in rounds (pair_table_round.cuh)
        roofline["kernel"] = roofline["kernel"].replace("sym_kernel", "round_kernel")
    if table and args.interp == "tsc":
        # the instruction tallies above are those of the CIC loops; the TSC loops (9 gathers) are not tallied
        roofline["kernel"] = roofline["kernel"].replace("CIC", "TSC")
        for key in ("achieved", "frac", "flops_per_pair_interaction", "pipe_instr_per_pair_interaction",
                    "pipe_util_vs_nominal"):
            roofline[key] = None
    if is_mixed:
        xu_peak = sm_count * NOMINAL_XU_LANES_PER_SM * sm_max * 1e6
        mufu = ((KERNEL_MIX[mode]["mufu"] if table else 2 * args.n_cut) + KERNEL_MIX[mode]["f2f"]) \
            / KERNEL_MIX[mode]["interactions"]
        roofline["xu_pipe_util_vs_nominal"] = mufu * pairs_per_step / t_pair / xu_peak
    else:
        roofline["measured_dfma_tflops"] = 2 * dfma_per_s / 1e12
        roofline["pipe_util_vs_measured_dfma"] = (None if roofline["frac"] is None
                                                  else instr * pairs_per_step / t_pair / dfma_per_s)
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
    periodic_desc = ("Ewald table 144x128 %s%s, (n_max,m_max)=(5,12), rho_max=5L, background Eq. 10"
                     % (args.interp.upper(), " (float nodes in shared memory)" if (args.table_fp32 or prec == b.PREC_MIXED) else "") if table
                     else "n_cut=%d (%d images/pair), background Eq. 9" % (args.n_cut, 2 * args.n_cut))
    line = {
        "metric": METRIC, "value": value, "unit": "pairs/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t_dev / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None,
        "dtype": "f64" if prec == b.PREC_FP64 else "f32",
        "data": "synthetic",
        "config": {"workload": "BASELINE configs[3]: N=%d LCDM comoving KDK step (Om=0.3, OL=0.7, "
                               "a 0.02->0.025), L=100 Mpc/h, r_max=1000, %s" % (n, periodic_desc),
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": "256 MiB buffer written between steps (L2 flush)"},
        "image_terms_per_s": None if table else value * 2 * args.n_cut,
        "seconds_per_force_evaluation": t_pair,
        "roofline": roofline, "cpu_baseline": cpu, "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": "pairs/s", "h2d_bytes_per_step": 11 * 8 * n,
                "d2h_bytes_per_step": 9 * 8 * n},
        "gpu_launches": int(round(launches_per_step * args.steps)),
        "peaks_file": peaks_kind,
    }
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
