"""Helpers of the GPU-vs-oracle parity tests: run both sides on the same seeded inputs and
compare decision for decision (SURVEY.md 8(c) acceptance criteria, BASELINE.json north_star).

The CUDA path is reached only through the C ABI (paper_1107_3490_b200.binding); the oracle only
through oracle/.  Nothing here computes any of the method's arithmetic.
"""
from __future__ import annotations

import numpy as np

import oracle
import paper_1107_3490_b200 as pt

REL_TOL = 1e-9   # north_star: per-step energies within 1e-9 relative; |dE| <= 1e-9 max(1, |E|)


def hist_range(N):
    return (-5.0 * N, 3.0 * N)


def run_oracle(N, M, E, T, widths, seeds, conf, n_sweeps, exchange_every, *, select_mode=0, nbins=64,
               hist=None, trace_sweeps=None, threads=None, e_offset=0):
    hist = hist or hist_range(N)
    p = oracle.make_params(N, M, E, select_mode=select_mode, nbins=nbins, hist_emin=hist[0],
                           hist_emax=hist[1], e_offset=e_offset)
    o = oracle.Oracle(p, T, widths, threads=threads)
    o.init(seeds, conf)
    cap = n_sweeps if trace_sweeps is None else trace_sweeps
    n_events = (n_sweeps // exchange_every) if exchange_every > 0 else 0
    tr = o.enable_trace(cap, n_events) if cap > 0 else {}
    o.run(n_sweeps, exchange_every)
    out = o.read()
    o.close()
    return out, tr


def run_gpu(N, M, E, T, widths, seeds, conf, n_sweeps, exchange_every, *, select_mode=0, nbins=64,
            hist=None, trace_sweeps=None, precision=pt.PT_F64, lanes=0, observables=1, stepwise=False,
            recompute=True):
    hist = hist or hist_range(N)
    p = pt.make_params(N, M, E, precision=precision, select_mode=select_mode, nbins=nbins,
                       observables=observables, lanes=lanes, hist_emin=hist[0], hist_emax=hist[1])
    with pt.ParallelTempering(p, T, widths) as sim:
        sim.pt_init(seeds, conf)
        cap = n_sweeps if trace_sweeps is None else trace_sweeps
        n_events = (n_sweeps // exchange_every) if exchange_every > 0 else 0
        if cap > 0:
            sim.pt_set_trace(cap, n_events)
        if stepwise:
            # the five calls of north_star used one by one instead of pt_run
            done = 0
            while done < n_sweeps:
                n = exchange_every if 0 < exchange_every <= n_sweeps - done else n_sweeps - done
                sim.pt_sweeps(n)
                done += n
                if exchange_every > 0 and n == exchange_every:
                    sim.pt_exchange()
        else:
            sim.pt_run(n_sweeps, exchange_every)
        out = sim.pt_read()
        if recompute:
            out["energies_full"] = sim.pt_recompute_energy()
        out["launch_info"] = sim.pt_launch_info()
        out["counters"] = sim.pt_counters()
        tr = sim.trace() if cap > 0 else {}
    return out, tr


def energy_close(a, b, tol=REL_TOL, floor=1.0):
    """|a - b| <= tol max(floor, |b|).  floor > 1 only where a chain started from an energy far
    above its current one: the running energy then carries the rounding of the large values it
    passed through."""
    a, b = np.asarray(a), np.asarray(b)
    return np.abs(a - b) <= tol * np.maximum(floor, np.abs(b))


def compare(gout, gtr, oout, otr, *, N, nbins, hist, label="", floor=1.0):
    """Asserts the fp64 acceptance criteria; returns a small report dict."""
    rep = {}
    if "move" in otr:
        div = int(np.count_nonzero(gtr["move"] != otr["move"]))
        rep["divergent_moves"] = div
        assert div == 0, f"{label}: {div} divergent move decisions (first at {np.argwhere(gtr['move'] != otr['move'])[0]})"
    if "swap" in otr:
        div = int(np.count_nonzero(gtr["swap"] != otr["swap"]))
        rep["divergent_swaps"] = div
        assert div == 0, f"{label}: {div} divergent swap decisions"
    if "energy" in otr:
        fl = np.asarray(floor)[..., None] if np.ndim(floor) else floor
        ok = energy_close(gtr["energy"], otr["energy"], floor=fl)
        rep["max_rel_energy_err"] = float(np.max(np.abs(gtr["energy"] - otr["energy"]) /
                                                 np.maximum(fl, np.abs(otr["energy"]))))
        assert ok.all(), f"{label}: per-sweep energy differs by {rep['max_rel_energy_err']:.3e} relative"
    # coordinates are bit-identical while decisions agree (proposals are exactly rounded on both sides)
    gc, oc = gout["conformations"], oout["conformations"]
    assert np.array_equal(gc.view(np.uint64), oc.view(np.uint64)), f"{label}: final conformations differ bitwise"
    assert energy_close(gout["energies"], oout["energies"], floor=floor).all(), f"{label}: final energies differ"
    if "energies_full" in gout:
        assert energy_close(gout["energies"], gout["energies_full"], floor=floor).all(), \
            f"{label}: running energy left the O(N^2) recompute"
    assert np.array_equal(gout["move_counts"], oout["move_counts"]), f"{label}: move counters differ"
    assert np.array_equal(gout["swap_counts"], oout["swap_counts"]), f"{label}: swap counters differ"
    gm, om = gout["moments"], oout["moments"]
    assert np.array_equal(gm[..., 0], om[..., 0]), f"{label}: n_meas differs"
    assert np.allclose(gm[..., 1:], om[..., 1:], rtol=1e-9, atol=1e-9 * float(np.max(floor)) ** 2), \
        f"{label}: energy moments differ"
    if "obs_moments" in gout and gout["obs_moments"].any():
        assert np.allclose(gout["obs_moments"], oout["obs_moments"], rtol=1e-9, atol=1e-12), \
            f"{label}: R_ee / R_gyr moments differ"
    if nbins > 0:
        gh, oh = gout["histograms"], oout["histograms"]
        assert gh.sum() == oh.sum(), f"{label}: histogram totals differ"
        l1 = int(np.abs(gh.astype(np.int64) - oh.astype(np.int64)).sum())
        allowed = 0
        if l1 and "energy" in otr:
            # a sample may land in the neighbouring bin only if it lies within 1e-9 relative of an edge
            e = otr["energy"]
            scale = nbins / (hist[1] - hist[0])
            lo = np.floor((e - REL_TOL * np.maximum(1, np.abs(e)) - hist[0]) * scale)
            hi = np.floor((e + REL_TOL * np.maximum(1, np.abs(e)) - hist[0]) * scale)
            allowed = 2 * int(np.count_nonzero(lo != hi))
        rep["hist_l1"] = l1
        assert l1 <= allowed, f"{label}: histograms differ (L1 = {l1}, allowed {allowed})"
    return rep
