"""The paper's timing experiment on B200 (Figs. 6-9).

    python paper_timing.py [--N 55] [--sweeps 4000 --every 1000] [--out gpurun_out/paper_timing.md] [--reps 3]

Workload of the paper's timings: homopolymer N = 55, 4000 sweeps per replica, replicas exchanged
every 1000 sweeps, number of replicas n_r varied; GPU time includes the host<->device copies
(PAPER.md:257).  Here: one ensemble of n_r replicas on a geometric ladder 0.2..3.0, sequential
monomer order, widths 0.1 sqrt(T), fp64 and fp32; the exchange runs on the device (the paper's
ran on the host).  Reported per n_r: wall time of pt_init + pt_run + pt_read (the paper's
convention) and of pt_run alone (CUDA events), attempted moves per second, and the mapping the
planner chose.  The paper prints speed-ups only (no absolute times), so there is nothing to
compare against; the shape to look for is its staircase in n_r, whose
period is the number of chains resident per wave.
"""
from __future__ import annotations

import argparse
import time

import numpy as np

import sys
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

from paper_1107_3490_b200 import binding as pt   # noqa: E402
from paper_1107_3490_b200 import synth           # noqa: E402

# the paper's range (up to ~500 replicas) and beyond it, with points on both sides of every multiple of the
# 592 SM sub-partitions of a B200, where a uniform mapping would step, and of the 394 chains up to which the
# warp-specialised kernel is chosen for N = 55
NR = [1, 8, 64, 148, 296, 394, 395, 592, 593, 740, 888, 1036, 1184, 1185, 1480, 1776, 2072, 2368, 2369, 2664, 2960, 3256,
      3552, 3848, 4144, 4145, 4440, 4736, 4737, 6000, 8288, 9472]


def run_one(N: int, SWEEPS: int, EVERY: int, n_r: int, precision: int, reps: int):
    import torch
    T = synth.temperature_ladder(n_r, 0.2, 3.0)
    w = synth.move_halfwidths(T)
    conf = synth.random_walk_conformations(1, n_r, N, seed=55_000 + n_r)
    seeds = synth.seeds(6, 1)
    p = pt.make_params(N, n_r, 1, precision=precision, nbins=0)
    stream = torch.cuda.Stream()
    best_wall, best_dev = 1e30, 1e30
    with pt.ParallelTempering(p, T, w, stream=stream) as sim:
        info = sim.pt_launch_info()
        kern = sim.pt_sweep_kernel_name()
        for _ in range(reps + 1):          # first repetition is the warm-up
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            sim.pt_init(seeds, conf)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            sim.pt_run(SWEEPS, EVERY)
            b.record(stream)
            sim.pt_read(histograms=False, obs_moments=False)
            wall = time.perf_counter() - t0
            dev = a.elapsed_time(b) * 1e-3
            if _ > 0:
                best_wall, best_dev = min(best_wall, wall), min(best_dev, dev)
    return best_wall, best_dev, info, kern


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--N", default="55", help="chain lengths, comma separated (the paper's timings: 55)")
    ap.add_argument("--sweeps", type=int, default=4000)
    ap.add_argument("--every", type=int, default=1000)
    ap.add_argument("--out", default="")
    ap.add_argument("--reps", type=int, default=3)
    ap.add_argument("--precisions", default="f64,f32")
    args = ap.parse_args()
    lines = []
    for N in [int(x) for x in args.N.split(",")]:
        lines.append(f"\nN = {N}, {args.sweeps} sweeps per replica, exchange every {args.every}; best of {args.reps} after one warm-up\n")
        lines.append("| n_r | kernel | lanes / chains per CTA / grid | " +
                     " | ".join(f"{p} wall s | {p} run s | {p} moves/s | {p} ns per move and chain on the busiest sub-partition"
                                for p in args.precisions.split(",")) + " |")
        lines.append("|---|---|---|" + "---|---|---|---|" * len(args.precisions.split(",")))
        for n_r in NR:
            cols, kern, info = [], "", None
            for prec in args.precisions.split(","):
                wall, dev, info, kern = run_one(N, args.sweeps, args.every, n_r, pt.PT_F32 if prec == "f32" else pt.PT_F64,
                                                args.reps)
                moves = n_r * N * args.sweeps
                cols += [f"{wall:.4f}", f"{dev:.4f}", f"{moves / dev:.3e}", f"{dev / (N * args.sweeps) * 1e9:.0f}"]
            lines.append(f"| {n_r} | `{kern}` | {info['lanes']} / {info['chains_per_cta']} / {info['grid']} | " + " | ".join(cols) + " |")
            print(lines[-1], flush=True)
    text = "\n".join(lines) + "\n"
    if args.out:
        Path(args.out).write_text(text)


if __name__ == "__main__":
    main()
