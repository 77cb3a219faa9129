#!/usr/bin/env python
"""Full-size parity report: BASELINE.json configs 0-4 at their full particle counts, GPU (through
the C ABI) against the CPU oracle on seeded sampled targets x all sources, both precisions.

    python tests/fullsize_parity.py [--configs 1,2,3,4] [--targets 256] > gpurun_out/fullsize.md

Not collected by pytest (minutes of GPU time at N = 4 194 304); the default `-m gpu` suite covers
the same code at N <= 1 048 576.  Prints a markdown table (profiles/r1_fullsize_parity.md is its output).
"""
import argparse
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="0,1,2,3,4")
    ap.add_argument("--targets", type=int, default=256)
    ap.add_argument("--n", type=int, default=0, help="override N (debugging)")
    ap.add_argument("--table", action="store_true",
                    help="also EWALD_TABLE mode (144 x 128 CIC, rho_max = 5 L) against oracle.accel_table")
    args = ap.parse_args()
    import torch
    import oracle
    from paper_2602_20787_b200 import binding as b
    from paper_2602_20787_b200 import build, workloads
    build.build()
    oracle.build()
    assert torch.cuda.is_available()
    print("| config | N | mode | targets | max rel err | RMS rel err | GPU s / evaluation | "
          "sum m g / sum m abs(g) |")
    print("|---|---:|---|---:|---:|---:|---:|---:|")
    for cfg in [int(c) for c in args.configs.split(",")]:
        w = workloads.make(cfg, n=args.n or None)
        idx = workloads.sample_targets(w.n, args.targets, seed=cfg)
        if cfg == 4:        # half of the targets inside the Plummer spheres (softening branches)
            ncl = w.cosmo["n_clustered"]
            a = workloads.sample_targets(ncl, args.targets // 2, seed=40)
            c = ncl + workloads.sample_targets(w.n - ncl, args.targets - args.targets // 2, seed=41)
            idx = np.sort(np.concatenate([a, c]))
        ref = np.stack(oracle.accel(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, w.n_cut, targets=idx), 1)
        dev = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (w.x, w.y, w.z, w.m, w.h)]
        for name, prec, flags in (("fp64 (symmetric, default)", b.PREC_FP64, 0),
                                  ("fp64 deterministic (rounds)", b.PREC_FP64, b.FLAG_DETERMINISTIC),
                                  ("fp64 ordered pairs", b.PREC_FP64, b.FLAG_ORDERED_PAIRS),
                                  ("mixed", b.PREC_MIXED, 0)):
            ctx = b.StepsCyl(n=w.n, Lz=w.Lz, G=w.G, n_cut=w.n_cut, precision=prec, flags=flags)
            g = [torch.empty(w.n, dtype=torch.float64, device="cuda") for _ in range(3)]
            ctx.accel(*dev, *g)
            ctx.check()
            secs = ctx.last_pair_kernel_ms() * 1e-3
            got = np.stack([t.cpu().numpy() for t in g], 1)
            ctx.close()
            e = np.linalg.norm(got[idx] - ref, axis=1) / np.linalg.norm(ref, axis=1)
            mom = max(abs(np.sum(w.m * got[:, c])) / np.sum(w.m * np.abs(got[:, c])) for c in range(3))
            print("| %d | %d | %s | %d | %.2e | %.2e | %.4g | %.1e |"
                  % (cfg, w.n, name, len(idx), e.max(), np.sqrt(np.mean(e ** 2)), secs, mom), flush=True)
        if not args.table:
            continue
        # EWALD_TABLE mode: the oracle interpolates ITS table (double nodes, or the same nodes rounded to
        # float for the two shared-memory variants) in double
        rmax = 5.0 * w.Lz
        D = oracle.ewald_table(w.Lz, 2.0 / w.Lz, 5, 12, 144, 128, rmax)
        D32 = D.astype(np.float32).astype(np.float64)
        refs = {0: np.stack(oracle.accel_table(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, D, rmax, 0, targets=idx), 1),
                1: np.stack(oracle.accel_table(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, D32, rmax, 0, targets=idx), 1)}
        for name, prec, f32 in (("table, double nodes (global memory)", b.PREC_FP64, 0),
                                ("table, float nodes (shared memory)", b.PREC_FP64, 1),
                                ("table, mixed", b.PREC_MIXED, 1)):
            ctx = b.StepsCyl(n=w.n, Lz=w.Lz, G=w.G, precision=prec, periodic_mode=b.PERIODIC_EWALD_TABLE,
                             tab_fp32=f32)
            g = [torch.empty(w.n, dtype=torch.float64, device="cuda") for _ in range(3)]
            ctx.accel(*dev, *g)
            ctx.check()
            secs = ctx.last_pair_kernel_ms() * 1e-3
            got = np.stack([t.cpu().numpy() for t in g], 1)
            ctx.close()
            ref_t = refs[f32]
            e = np.linalg.norm(got[idx] - ref_t, axis=1) / np.linalg.norm(ref_t, axis=1)
            mom = max(abs(np.sum(w.m * got[:, c])) / np.sum(w.m * np.abs(got[:, c])) for c in range(3))
            print("| %d | %d | %s | %d | %.2e | %.2e | %.4g | %.1e |"
                  % (cfg, w.n, name, len(idx), e.max(), np.sqrt(np.mean(e ** 2)), secs, mom), flush=True)


if __name__ == "__main__":
    main()
