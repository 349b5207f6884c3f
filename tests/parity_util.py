"""Helpers of the GPU-vs-oracle parity tests: run both sides on the same seeded inputs and
compare decision for decision (SURVEY.md 8(c) acceptance criteria, BASELINE.json north_star).

The CUDA path is reached only through the C ABI (paper_1107_3490_b200.binding); the oracle only
through oracle/.  Nothing here computes any of the method's arithmetic.

Two kinds of GPU run are compared with the same oracle run:
  trace_moves=True   pt_set_trace with a move-decision buffer: the TRACE=true instantiations of the sweep
                     kernels run, and the first divergent decision can be named;
  trace_moves=False  no move buffer: the kernels are the ones an untraced run (bench.py) launches; the
                     per-sweep energies and the swap decisions are still recorded (they are written outside
                     the step loop), and the final conformations are compared bitwise -- proposals are
                     exactly rounded on both sides, so equal final coordinates mean equal decisions.
"""
from __future__ import annotations

import numpy as np

import oracle
import paper_1107_3490_b200 as pt

REL_TOL = 1e-9   # north_star: per-step energies within 1e-9 relative; |dE| <= 1e-9 max(1, |E|)


def hist_range(N):
    return (-5.0 * N, 3.0 * N)


def run_oracle(N, M, E, T, widths, seeds, conf, n_sweeps, exchange_every, *, select_mode=0, nbins=64,
               hist=None, trace_sweeps=None, threads=None, e_offset=0, trace_moves=True):
    hist = hist or hist_range(N)
    p = oracle.make_params(N, M, E, select_mode=select_mode, nbins=nbins, hist_emin=hist[0],
                           hist_emax=hist[1], e_offset=e_offset)
    o = oracle.Oracle(p, T, widths, threads=threads)
    o.init(seeds, conf)
    cap = n_sweeps if trace_sweeps is None else trace_sweeps
    n_events = (n_sweeps // exchange_every) if exchange_every > 0 else 0
    tr = o.enable_trace(cap, n_events, moves=trace_moves) if cap > 0 else {}
    o.run(n_sweeps, exchange_every)
    out = o.read()
    o.close()
    return out, tr


def run_gpu(N, M, E, T, widths, seeds, conf, n_sweeps, exchange_every, *, select_mode=0, nbins=64,
            hist=None, trace_sweeps=None, precision=pt.PT_F64, lanes=0, observables=1, stepwise=False,
            recompute=True, trace_moves=True, trace_ensembles=None):
    hist = hist or hist_range(N)
    p = pt.make_params(N, M, E, precision=precision, select_mode=select_mode, nbins=nbins,
                       observables=observables, lanes=lanes, hist_emin=hist[0], hist_emax=hist[1])
    with pt.ParallelTempering(p, T, widths) as sim:
        sim.pt_init(seeds, conf)
        cap = n_sweeps if trace_sweeps is None else trace_sweeps
        n_events = (n_sweeps // exchange_every) if exchange_every > 0 else 0
        if cap > 0:
            sim.pt_set_trace(cap, n_events, moves=trace_moves)
        kernel = sim.pt_sweep_kernel_name()
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
        out["kernel"] = kernel
        tr = sim.trace(trace_ensembles) if cap > 0 else {}
    return out, tr


def energy_close(a, b, tol=REL_TOL, floor=1.0):
    """|a - b| <= tol max(floor, |b|).  floor > 1 only where a chain started from an energy far
    above its current one: the running energy then carries the rounding of the large values it
    passed through."""
    a, b = np.asarray(a), np.asarray(b)
    return np.abs(a - b) <= tol * np.maximum(floor, np.abs(b))


def rebased_floor(e_trace, e0, exchange_every):
    """Energy scale the 1e-9 relative criterion refers to, per (ensemble, temperature, sweep), for runs that
    start far above their equilibrium energy.  E_run += dE keeps the absolute rounding of the largest energy
    held since the running energy was last re-based on Eq. (4): at pt_init, and before the exchange events
    x = 2^k - 1 (R22), i.e. after sweep S 2^k - 1.  Conformations migrate between temperatures, so
    the scale is the largest |E| of the whole ensemble since that point.  e_trace [E][M][T] is the ORACLE's."""
    E, M, T = e_trace.shape
    a = np.abs(e_trace).max(axis=1)                       # [E][T]
    fl = np.empty((E, T))
    run = np.full(E, float(e0))
    nxt = exchange_every if exchange_every > 0 else T + 1  # first sweep index after a re-basing
    for t in range(T):
        if t == nxt:
            run = a[:, t - 1].copy()                       # the energies the re-basing recomputed
            nxt *= 2
        run = np.maximum(run, a[:, t])
        fl[:, t] = run
    return np.maximum(1.0, fl)[:, None, :].repeat(M, axis=1)


def compare(gout, gtr, oout, otr, *, N, nbins, hist, label="", floor=1.0):
    """Asserts the fp64 acceptance criteria; returns a small report dict.  `floor`: scalar, or [E][M][T]
    (rebased_floor) for starts with huge energies."""
    rep = {"kernel": gout.get("kernel")}
    floor_t = None
    if np.ndim(floor) == 3:
        floor_t = np.asarray(floor)
        floor = floor_t[:, :, -1]                          # scale of the final state
    if "move" in otr and "move" in gtr:
        div = int(np.count_nonzero(gtr["move"] != otr["move"]))
        rep["divergent_moves"] = div
        assert div == 0, f"{label}: {div} divergent move decisions (first at {np.argwhere(gtr['move'] != otr['move'])[0]})"
    if "swap" in otr:
        div = int(np.count_nonzero(gtr["swap"] != otr["swap"]))
        rep["divergent_swaps"] = div
        assert div == 0, f"{label}: {div} divergent swap decisions"
    if "energy" in otr:
        fl = floor_t if floor_t is not None else (np.asarray(floor)[..., None] if np.ndim(floor) else floor)
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
    if floor_t is not None and "energy" in otr:
        tol = REL_TOL * np.maximum(floor_t, np.abs(otr["energy"]))
        assert (np.abs(gm[..., 1] - om[..., 1]) <= tol.sum(-1) + 1e-9 * np.abs(om[..., 1])).all(), f"{label}: sum E differs"
        tol2 = (2 * np.abs(otr["energy"]) * tol + tol * tol).sum(-1)
        assert (np.abs(gm[..., 2] - om[..., 2]) <= tol2 + 1e-9 * np.abs(om[..., 2])).all(), f"{label}: sum E^2 differs"
    else:
        assert np.allclose(gm[..., 1:], om[..., 1:], rtol=1e-9, atol=1e-9 * float(np.max(floor)) ** 2), \
            f"{label}: energy moments differ"
    if "obs_moments" in gout and gout["obs_moments"].any():
        go, oo = gout["obs_moments"], oout["obs_moments"]
        assert np.allclose(go[..., :4], oo[..., :4], rtol=1e-9, atol=1e-12), f"{label}: R_ee / R_gyr moments differ"
        # sum E r_gyr^2 inherits the energy tolerance
        scale = float(np.max(floor_t)) if floor_t is not None else float(np.max(floor))
        assert np.allclose(go[..., 4], oo[..., 4], rtol=1e-9, atol=1e-9 * scale * float(oo[..., 1].max())), \
            f"{label}: E r_gyr^2 cross moment differs"
    if nbins > 0:
        gh, oh = gout["histograms"], oout["histograms"]
        assert gh.sum() == oh.sum(), f"{label}: histogram totals differ"
        l1 = int(np.abs(gh.astype(np.int64) - oh.astype(np.int64)).sum())
        allowed = 0
        if l1 and "energy" in otr:
            # a sample may land in the neighbouring bin only if it lies within the energy tolerance of an edge
            e = otr["energy"]
            fl = floor_t if floor_t is not None else (np.asarray(floor)[..., None] if np.ndim(floor) else floor)
            scale = nbins / (hist[1] - hist[0])
            lo = np.floor((e - REL_TOL * np.maximum(fl, np.abs(e)) - hist[0]) * scale)
            hi = np.floor((e + REL_TOL * np.maximum(fl, np.abs(e)) - hist[0]) * scale)
            allowed = 2 * int(np.count_nonzero(lo != hi))
        rep["hist_l1"] = l1
        assert l1 <= allowed, f"{label}: histograms differ (L1 = {l1}, allowed {allowed})"
    return rep


def both(N, M, E, T, widths, seeds, conf, n_sweeps, exchange_every, *, lanes=0, select_mode=0, nbins=64,
         stepwise=False, threads=None, floor=1.0, label="", traces=(True, False), expect_kernel=None,
         start_energy=None):
    """One oracle run, then one GPU run per entry of `traces` (move-decision trace on / off), each compared
    with it.  With both settings the two GPU runs must have used different sweep-kernel instantiations
    (...trace=1> and ...trace=0>).  Returns ({trace_moves: report}, {trace_moves: (gout, gtr)}, (oout, otr))."""
    hist = hist_range(N)
    kw = dict(select_mode=select_mode, nbins=nbins, hist=hist)
    o = run_oracle(N, M, E, T, widths, seeds, conf, n_sweeps, exchange_every, threads=threads, **kw)
    if start_energy is not None:      # a start far above equilibrium: the energy scale follows the re-basings
        floor = rebased_floor(o[1]["energy"], start_energy, exchange_every)
    reps, runs = {}, {}
    for tm in traces:
        g = run_gpu(N, M, E, T, widths, seeds, conf, n_sweeps, exchange_every, lanes=lanes, stepwise=stepwise,
                    trace_moves=tm, **kw)
        reps[tm] = compare(g[0], g[1], o[0], o[1], N=N, nbins=nbins, hist=hist, floor=floor,
                           label=f"{label} lanes={lanes} move-trace={'on' if tm else 'off'} [{g[0]['kernel']}]")
        runs[tm] = g
        if n_sweeps > 0:
            assert g[0]["kernel"].endswith(f"trace={1 if tm else 0}>"), g[0]["kernel"]
        if expect_kernel is not None:
            assert g[0]["kernel"].startswith(expect_kernel), (g[0]["kernel"], expect_kernel)
    if True in runs and False in runs and n_sweeps > 0:
        assert runs[True][0]["kernel"] != runs[False][0]["kernel"]
        # the two instantiations agree with each other bit for bit as well
        assert np.array_equal(runs[True][0]["energies"], runs[False][0]["energies"])
    return reps, runs, o
