#!/usr/bin/env python
"""Two small experiments from the paper run on the B200 library.

    python paper_physics.py --what literal [--out gpurun_out/paper_literal.md]
    python paper_physics.py --what cv      [--out gpurun_out/paper_cv_N13.md] [--N 13]

literal  The paper's move exactly as printed: "a random monomer of the chain is picked" and its
         coordinates are shifted by a vector with components uniform in [-0.01, 0.01], the same at every
         temperature (PT_RANDOM_PICK + synth.paper_halfwidths), on BASELINE configs 1 and 3: acceptance rate of
         the moves and of the swaps per temperature, beside the configs' own 0.1 sqrt(T) width.
cv       Thermodynamics of the N = 13 chain (Figs. 4 and 5): C_V(T)/N from Eq. (7) and
         d<r_gyr^2>/dT / N from the fluctuation formula under Eq. (8) per temperature, with the standard error
         over independent ensembles, plus C_V between the ladder points by single-histogram reweighting
         (paper_1107_3490_b200.analysis).  An eyeball against Fig. 4 -- the paper gives no numbers, no
         temperature set and no run lengths -- whose freezing peak it places at T ~ 0.33.

Nothing here is on the hot path or in the timed region; the arithmetic of the method runs in the CUDA kernels.
"""
from __future__ import annotations

import argparse
import sys
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

import paper_1107_3490_b200 as pt                      # noqa: E402
from paper_1107_3490_b200 import analysis, synth       # noqa: E402


def literal(out: str):
    lines = ["Acceptance rates of the paper-literal move (random monomer pick, components uniform in [-0.01, 0.01] at",
             "every temperature, PAPER.md:95) beside the BASELINE.json move (sequential order, half-width 0.1 sqrt(T)).",
             "Full length of each configuration, fp64, measured after discarding the first 20 % of the sweeps.", ""]
    for cid in (1, 3):
        inp = synth.make_inputs(cid)
        wl = inp.workload
        res = {}
        for name, mode, w in (("paper", pt.PT_RANDOM_PICK, synth.paper_halfwidths(wl.M)),
                              ("baseline", pt.PT_SEQUENTIAL, inp.widths)):
            p = pt.make_params(wl.N, wl.M, wl.E, select_mode=mode, nbins=0)
            with pt.ParallelTempering(p, inp.temperatures, w) as sim:
                sim.pt_init(inp.seeds, inp.conformations)
                sim.pt_run(wl.n_sweeps // 5, wl.exchange_every)
                sim.pt_reset_stats()
                sim.pt_run(wl.n_sweeps - wl.n_sweeps // 5, wl.exchange_every)
                o = sim.pt_read(histograms=False, conformations=False)
            mc, sc = o["move_counts"][0].astype(float), o["swap_counts"][0].astype(float)
            res[name] = (mc[:, 1] / mc[:, 0], mc[:, 2] / mc[:, 0], sc[:, 1] / np.maximum(sc[:, 0], 1),
                         o["moments"][0, :, 1] / o["moments"][0, :, 0])
        lines += [f"### {wl.name}: N = {wl.N}, M = {wl.M}, {wl.n_sweeps} sweeps, exchange every {wl.exchange_every}", "",
                  "| i | T | paper: move acc. | paper: swap acc. (i, i+1) | paper: <E> | baseline: move acc. | baseline: bond-range rej. | baseline: swap acc. | baseline: <E> |",
                  "|---|---|---|---|---|---|---|---|---|"]
        step = max(1, wl.M // 16)
        for i in range(0, wl.M, step):
            a, b = res["paper"], res["baseline"]
            sw = lambda r: f"{r[2][i]:.3f}" if i < wl.M - 1 else "-"
            lines.append(f"| {i} | {inp.temperatures[i]:.4f} | {a[0][i]:.4f} | {sw(a)} | {a[3][i]:.3f} | {b[0][i]:.4f} | "
                         f"{b[1][i]:.2e} | {sw(b)} | {b[3][i]:.3f} |")
        a, b = res["paper"], res["baseline"]
        lines += ["", f"Move acceptance over all temperatures: paper-literal {a[0].min():.3f} .. {a[0].max():.3f}, "
                      f"baseline width {b[0].min():.3f} .. {b[0].max():.3f}.  With steps of 0.01 (1.4 % of the bond length) "
                      f"nearly every move is accepted and the chain diffuses slowly: after the same number of sweeps the "
                      f"cold replicas of the paper-literal run are still {np.max(a[3][:4] - b[3][:4]):.1f} above the baseline's energies.", ""]
    text = "\n".join(lines) + "\n"
    print(text)
    if out:
        Path(out).write_text(text)


def cv(out: str, N: int, E: int, M: int, n_therm: int, n_meas: int):
    T = synth.temperature_ladder(M, 0.15, 3.0)
    w = synth.move_halfwidths(T)
    conf = synth.random_walk_conformations(E, M, N, seed=1107349013)
    seeds = synth.seeds(13, E)
    nbins, hr = 2048, (-5.0 * N, 3.0 * N)
    p = pt.make_params(N, M, E, nbins=nbins, observables=1, hist_emin=hr[0], hist_emax=hr[1])
    with pt.ParallelTempering(p, T, w) as sim:
        sim.pt_init(seeds, conf)
        sim.pt_run(n_therm, 10)
        sim.pt_reset_stats()
        sim.pt_run(n_meas, 10)
        o = sim.pt_read(conformations=False)
        kernel = sim.pt_sweep_kernel_name()
    mom, obs = o["moments"], o["obs_moments"]
    e = analysis.mean_energy(mom) / N
    c = analysis.specific_heat(mom, T) / N
    g = analysis.mean_rgyr2(mom, obs)
    dg = analysis.d_rgyr2_dT(mom, obs, T) / N
    se = lambda a: a.std(0, ddof=1) / np.sqrt(E)
    acc = (o["move_counts"][..., 1] / o["move_counts"][..., 0]).mean(0)
    sacc = (o["swap_counts"][..., 1] / np.maximum(o["swap_counts"][..., 0], 1)).mean(0)
    lines = [f"N = {N} homopolymer, {E} independent ensembles x {M} temperatures (geometric 0.15 .. 3.0), half-width 0.1 sqrt(T),",
             f"exchange every 10 sweeps; {n_therm} sweeps discarded, {n_meas} measured; fp64; kernel `{kernel}`.",
             "Mean over ensembles +- standard error.  C_V = (<E^2> - <E>^2)/T^2 (Eq. 7, PAPER.md:232);",
             "d<r_gyr^2>/dT = (<E r_gyr^2> - <E><r_gyr^2>)/T^2 (PAPER.md:238-249).", "",
             "| i | T | <E>/N | C_V/N | <r_gyr^2> | (d<r_gyr^2>/dT)/N | move acc. | swap acc. (i, i+1) |", "|---|---|---|---|---|---|---|---|"]
    for i in range(M):
        lines.append(f"| {i} | {T[i]:.4f} | {e.mean(0)[i]:.4f} +- {se(e)[i]:.4f} | {c.mean(0)[i]:.4f} +- {se(c)[i]:.4f} | "
                     f"{g.mean(0)[i]:.4f} +- {se(g)[i]:.4f} | {dg.mean(0)[i]:.5f} +- {se(dg)[i]:.5f} | {acc[i]:.3f} | "
                     + (f"{sacc[i]:.3f}" if i < M - 1 else "-") + " |")
    # C_V between the ladder points: reweight the pooled histogram of each temperature to +-4 % around it
    centres = analysis.bin_centres(nbins, *hr)
    hist = o["histograms"][..., :nbins].sum(0)
    lo = int(np.searchsorted(T, 0.2)); hi = int(np.searchsorted(T, 0.6))
    curve = []
    for i in range(max(lo - 1, 0), min(hi + 1, M)):
        Tt = T[i] * np.linspace(0.96, 1.04, 9)
        _, cvt = analysis.reweight(hist[i], centres, T[i], Tt)
        curve += list(zip(Tt, cvt / N))
    curve.sort()
    tt, cc = np.array([x for x, _ in curve]), np.array([y for _, y in curve])
    win = (tt > 0.2) & (tt < 0.6)
    t_peak = tt[win][np.argmax(cc[win])]
    lines += ["", "C_V/N between the ladder points (single-histogram reweighting of each temperature's pooled histogram to +-4 %):", "",
              "| T | C_V/N |", "|---|---|"]
    lines += [f"| {x:.4f} | {y:.4f} |" for x, y in curve[::3]]
    imax = int(np.argmax(np.where((T > 0.2) & (T < 0.6), c.mean(0), -np.inf)))
    lines += ["", f"Low-temperature maximum of C_V/N: ladder point T = {T[imax]:.3f} ({c.mean(0)[imax]:.3f} +- {se(c)[imax]:.3f}); "
                  f"reweighted curve T = {t_peak:.3f}.  The paper reads T ~ 0.33 for N = 13 off its Fig. 4 (PAPER.md:236); "
                  f"no numbers, temperature set or run lengths are given there, so this is an eyeball, not a pin.", ""]
    text = "\n".join(lines) + "\n"
    print(text)
    if out:
        Path(out).write_text(text)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--what", required=True, choices=["literal", "cv"])
    ap.add_argument("--out", default="")
    ap.add_argument("--N", type=int, default=13)
    ap.add_argument("--E", type=int, default=64)
    ap.add_argument("--M", type=int, default=32)
    ap.add_argument("--therm", type=int, default=20000)
    ap.add_argument("--meas", type=int, default=200000)
    args = ap.parse_args()
    if args.what == "literal":
        literal(args.out)
    else:
        cv(args.out, args.N, args.E, args.M, args.therm, args.meas)


if __name__ == "__main__":
    main()
