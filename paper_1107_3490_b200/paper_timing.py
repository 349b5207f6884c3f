"""The paper's timing experiment on B200 (Figs. 6-9).

    python -m paper_1107_3490_b200.paper_timing [--out profiles/r01_paper_timing.md] [--reps 3]

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

from . import binding as pt
from . import synth

N, SWEEPS, EVERY = 55, 4000, 1000
NR = [1, 2, 4, 8, 16, 32, 64, 128, 148, 149, 256, 296, 297, 512, 592, 593, 1024, 1184, 1185, 2048, 2368, 2369, 4096]


def run_one(n_r: int, precision: int, reps: int):
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
    return best_wall, best_dev, info


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default="")
    ap.add_argument("--reps", type=int, default=3)
    args = ap.parse_args()
    rows = []
    for n_r in NR:
        r = {"n_r": n_r}
        for name, prec in (("f64", pt.PT_F64), ("f32", pt.PT_F32)):
            wall, dev, info = run_one(n_r, prec, args.reps)
            r[name] = (wall, dev, info)
        rows.append(r)
        print(n_r, {k: (round(v[0], 4), round(v[1], 4)) for k, v in r.items() if k != "n_r"}, flush=True)
    lines = ["| n_r | lanes / chains per CTA / grid | fp64 wall s (init+run+read) | fp64 run s | fp64 moves/s | fp32 wall s | fp32 run s | fp32 moves/s |",
             "|---|---|---|---|---|---|---|---|"]
    for r in rows:
        moves = r["n_r"] * N * SWEEPS
        i = r["f64"][2]
        lines.append(f"| {r['n_r']} | {i['lanes']} / {i['chains_per_cta']} / {i['grid']} | {r['f64'][0]:.4f} | {r['f64'][1]:.4f} | "
                     f"{moves / r['f64'][1]:.3e} | {r['f32'][0]:.4f} | {r['f32'][1]:.4f} | {moves / r['f32'][1]:.3e} |")
    text = "\n".join(lines)
    print(text)
    if args.out:
        with open(args.out, "w") as f:
            f.write(text + "\n")


if __name__ == "__main__":
    main()
