"""GPU-vs-oracle parity (fp64): the CUDA path, called through the C ABI, must reproduce the
oracle's trajectory decision for decision on the same seeded inputs (BASELINE.json north_star;
SURVEY.md 8(c)): 0 divergent accept/reject decisions, 0 divergent swap decisions, per-sweep
running energies within 1e-9 max(1,|E|), final conformations bit-identical, equal counters and
histograms.  The GPU swaps temperature labels, the oracle swaps conformations (PAPER.md:105 vs
:267): their agreement is itself the test of that equivalence.
"""
import numpy as np
import pytest

import paper_1107_3490_b200 as pt
from paper_1107_3490_b200 import synth
from parity_util import compare, energy_close, hist_range, run_gpu, run_oracle

pytestmark = pytest.mark.gpu


def _both(inp, n_sweeps, *, lanes=0, select_mode=0, widths=None, nbins=64, stepwise=False, threads=None,
          exchange_every=None, floor=1.0):
    wl = inp.workload
    w = inp.widths if widths is None else widths
    S = wl.exchange_every if exchange_every is None else exchange_every
    hist = hist_range(wl.N)
    kw = dict(select_mode=select_mode, nbins=nbins, hist=hist)
    o = run_oracle(wl.N, wl.M, wl.E, inp.temperatures, w, inp.seeds, inp.conformations, n_sweeps, S,
                   threads=threads, **kw)
    g = run_gpu(wl.N, wl.M, wl.E, inp.temperatures, w, inp.seeds, inp.conformations, n_sweeps, S,
                lanes=lanes, stepwise=stepwise, **kw)
    return compare(g[0], g[1], o[0], o[1], N=wl.N, nbins=nbins, hist=hist, floor=floor,
                   label=f"{wl.name} lanes={lanes}"), g, o


# ---- the five BASELINE.json configurations --------------------------------------------------

def test_config1_full_run():
    """N=13, M=8, 2000 sweeps, exchange every 10: the whole job, default mapping."""
    rep, g, _ = _both(synth.make_inputs(1), 2000)
    assert rep["divergent_moves"] == 0 and rep["divergent_swaps"] == 0
    assert g[0]["counters"] == (2000, 200)


@pytest.mark.parametrize("lanes", [8, 16, 32, 64, 128])
def test_config1_every_mapping(lanes):
    """All lane mappings (sub-warp groups, one warp, one CTA per replica) give the same trajectory."""
    _both(synth.make_inputs(1), 300, lanes=lanes)


def test_config1_stepwise_calls_equal_pt_run():
    """pt_sweeps / pt_exchange called one by one = pt_run."""
    _both(synth.make_inputs(1), 200, stepwise=True)


def test_config2_full_run():
    """N=30, M=32, 10^4 sweeps, 4096-bin histograms."""
    rep, g, _ = _both(synth.make_inputs(2), 10000, nbins=4096)
    assert g[0]["histograms"].sum() == 32 * 10000


def test_config3_fp64():
    """N=55, M=64, exchange every 20; 2000 of the 10^4 sweeps (the oracle's share of the time)."""
    _both(synth.make_inputs(3), 2000, nbins=4096)


@pytest.mark.parametrize("lanes", [0, 128, 256])
def test_config4_long_chain(lanes):
    """N=309, M=128: the long Delta-E reduction: one warp per replica (default), one CTA per replica."""
    rep, g, _ = _both(synth.make_inputs(4), 60 if lanes else 100, lanes=lanes)
    if lanes == 0:
        assert g[0]["launch_info"]["lanes"] == 32, "config 4 maps one warp per replica (10 unrolled iterations)"


def test_config5_sampled_ensembles_of_the_full_batch():
    """64 ensembles x 64 replicas, N=100: the GPU runs the FULL batch in bench.py's launch
    configuration; the oracle recomputes sampled ensembles one by one (first, middle, last)."""
    inp = synth.make_inputs(5)
    wl = inp.workload
    n_sweeps, S, nbins = 100, wl.exchange_every, 4096
    hist = hist_range(wl.N)
    g, gtr = run_gpu(wl.N, wl.M, wl.E, inp.temperatures, inp.widths, inp.seeds, inp.conformations,
                     n_sweeps, S, nbins=nbins, hist=hist)
    assert energy_close(g["energies"], g["energies_full"]).all()
    for e in (0, 31, 63):
        o, otr = run_oracle(wl.N, wl.M, 1, inp.temperatures, inp.widths, inp.seeds[e:e + 1],
                            inp.conformations[e:e + 1], n_sweeps, S, nbins=nbins, hist=hist, e_offset=e)
        ge = {k: v[e:e + 1] for k, v in g.items() if isinstance(v, np.ndarray)}
        gte = {k: v[e:e + 1] for k, v in gtr.items()}
        compare(ge, gte, o, otr, N=wl.N, nbins=nbins, hist=hist, label=f"config5 ensemble {e}")


def test_mixed_mapping_at_the_papers_chain_length():
    """N = 55, 40 ensembles x 64 replicas = 2560 chains: between 4 and 7 chains per SM sub-partition, so
    the planner maps 4 chains x 8 lanes + 3 chains x 10 lanes on every one (k_sweep_mixed<7, 6>).  Sampled
    ensembles against the oracle; they cover both kinds of warp."""
    N, M, E = 55, 64, 40
    T = synth.temperature_ladder(M, 0.15, 3.0)
    w = synth.move_halfwidths(T)
    conf = synth.random_walk_conformations(E, M, N, seed=5564)
    seeds = synth.seeds(3, E, rank=3)
    hist = hist_range(N)
    g, gtr = run_gpu(N, M, E, T, w, seeds, conf, 30, 10, nbins=64, hist=hist)
    assert g["launch_info"]["chains_per_cta"] == 28 and g["launch_info"]["lanes"] == 8
    assert energy_close(g["energies"], g["energies_full"]).all()
    for e in (0, 17, 39):
        o, otr = run_oracle(N, M, 1, T, w, seeds[e:e + 1], conf[e:e + 1], 30, 10, nbins=64, hist=hist, e_offset=e)
        ge = {k: v[e:e + 1] for k, v in g.items() if isinstance(v, np.ndarray)}
        gte = {k: v[e:e + 1] for k, v in gtr.items()}
        compare(ge, gte, o, otr, N=N, nbins=64, hist=hist, label=f"mixed N=55 ensemble {e}")


def test_config5_full_length_invariants():
    """Config 5 at full size and length (10^3 sweeps) as bench.py times it: properties that hold at
    any size -- E_run equals the oracle's Eq.-4 energy of the returned conformation for sampled
    chains, counters add up, every bond inside the FENE range, label permutation intact."""
    import oracle
    inp = synth.make_inputs(5)
    wl = inp.workload
    p = pt.make_params(wl.N, wl.M, wl.E, nbins=4096, hist_emin=-5.0 * wl.N, hist_emax=3.0 * wl.N)
    with pt.ParallelTempering(p, inp.temperatures, inp.widths) as sim:
        sim.pt_init(inp.seeds, inp.conformations)
        sim.pt_run(wl.n_sweeps, wl.exchange_every)
        out = sim.pt_read()
        efull = sim.pt_recompute_energy()
    assert energy_close(out["energies"], efull).all()
    rng = np.random.default_rng(5)
    op = oracle.make_params(wl.N)
    for e, i in zip(rng.integers(0, wl.E, 48), rng.integers(0, wl.M, 48)):
        eo = oracle.total_energy(out["conformations"][e, i], op)
        assert energy_close(out["energies"][e, i], eo), (e, i)
    mc = out["move_counts"]
    assert (mc[..., 0] == wl.N * wl.n_sweeps).all() and (mc[..., 1] <= mc[..., 0]).all()
    assert (out["moments"][..., 0] == wl.n_sweeps).all()
    assert (out["histograms"].sum(-1) == wl.n_sweeps).all()
    sc = out["swap_counts"]
    n_events = wl.n_sweeps // wl.exchange_every
    assert (sc[:, 0::2, 0] == (n_events + 1) // 2).all() and (sc[:, 1::2, 0] == n_events // 2).all()
    b = np.linalg.norm(np.diff(out["conformations"], axis=2), axis=-1)
    assert (np.abs(b - 0.7) < 0.3).all()
    # colder replicas end with lower mean energy than hotter ones
    em = out["moments"][..., 1].mean(0) / wl.n_sweeps
    assert em[0] < em[-1]


# ---- variants and edge cases ----------------------------------------------------------------

def test_random_pick_mode():
    """Paper-literal monomer choice in every mapping family."""
    for lanes in (8, 32, 64):
        _both(synth.make_inputs(1), 200, lanes=lanes, select_mode=1)


def test_paper_literal_width():
    """Components uniform in [-0.01, 0.01] at every temperature."""
    _both(synth.make_inputs(1), 300, widths=synth.paper_halfwidths(8))


def test_overlapping_start_large_energies():
    """Plain random walks with overlaps: huge initial energies, Delta E = -1e6...+inf, bond-range
    rejections.  Decisions and coordinates must still agree; energies within 1e-9 relative."""
    wl = synth.CONFIGS[1]
    T = synth.temperature_ladder(wl.M, wl.T_min, wl.T_max)
    conf = synth.random_walk_conformations(1, wl.M, wl.N, seed=99, d_min=0.0)
    inp = synth.Inputs(wl, T, synth.move_halfwidths(T, 0.6), synth.seeds(9, 1), conf)
    import oracle
    e0 = max(abs(oracle.total_energy(c)) for c in conf[0])
    assert e0 > 1e3
    # the running energy carries the rounding of the large values it came down from; conformations
    # can swap between temperatures, so the largest initial energy is the floor for all of them
    rep, g, _ = _both(inp, 150, nbins=0, floor=e0)
    assert g[0]["move_counts"][..., 2].sum() > 0, "the wide moves should have produced bond-range rejections"


@pytest.mark.parametrize("N,M,E", [(2, 1, 1), (2, 3, 5), (3, 2, 7), (5, 1, 3), (17, 5, 3), (33, 7, 2),
                                    (64, 4, 2), (65, 3, 1), (128, 2, 1), (129, 2, 1), (257, 2, 1), (481, 2, 1)])
def test_ragged_shapes(N, M, E):
    """Degenerate and ragged sizes: the dimer, M=1 (no exchange partner), odd M, chain lengths
    around the lane-count multiples, chain counts that leave partly empty warps."""
    T = synth.temperature_ladder(M, 0.4, 2.5)
    wl = synth.Workload(f"ragged_{N}_{M}_{E}", N, M, E, 0.4, 2.5, 3, 40)
    inp = synth.Inputs(wl, T, synth.move_halfwidths(T), synth.seeds(7, E),
                       synth.random_walk_conformations(E, M, N, seed=N * 1000 + M * 10 + E))
    for lanes in (0, 8, 32, 64):
        _both(inp, 40, lanes=lanes, nbins=16)


def test_zero_sweeps_and_no_exchange():
    inp = synth.make_inputs(1)
    _both(inp, 0)
    _both(inp, 25, exchange_every=0)
    _both(inp, 25, exchange_every=7)    # a trailing partial block is not followed by an exchange


def test_reset_stats_and_resume():
    """pt_reset_stats keeps the trajectory: 100 + reset + 100 sweeps ends in the same state as 200."""
    inp = synth.make_inputs(1)
    wl = inp.workload
    p = pt.make_params(wl.N, wl.M, wl.E, nbins=32, hist_emin=-65, hist_emax=39)
    outs = []
    for split in (False, True):
        with pt.ParallelTempering(p, inp.temperatures, inp.widths) as sim:
            sim.pt_init(inp.seeds, inp.conformations)
            if split:
                sim.pt_run(100, 10)
                sim.pt_reset_stats()
                sim.pt_run(100, 10)
            else:
                sim.pt_run(200, 10)
            outs.append(sim.pt_read())
    a, b = outs
    assert np.array_equal(a["conformations"], b["conformations"])
    assert np.array_equal(a["energies"], b["energies"])
    assert (b["moments"][..., 0] == 100).all() and (a["moments"][..., 0] == 200).all()
    assert (b["move_counts"][..., 0] == 100 * wl.N).all()


def test_exact_resume_from_read_state():
    """pt_read at a break + pt_init + pt_set_counters on a fresh handle continues
    the run bit for bit (coordinates, decisions, swap decisions), across an odd exchange parity."""
    inp = synth.make_inputs(2)
    wl = inp.workload
    S = wl.exchange_every
    p = pt.make_params(wl.N, wl.M, wl.E, nbins=0)
    n1, n2 = 70, 50      # break after 7 exchange events: the next event has odd parity
    with pt.ParallelTempering(p, inp.temperatures, inp.widths) as a:
        a.pt_init(inp.seeds, inp.conformations)
        a.pt_set_trace(n1 + n2, (n1 + n2) // S)
        a.pt_run(n1 + n2, S)
        full, ftr = a.pt_read(), a.trace()
    with pt.ParallelTempering(p, inp.temperatures, inp.widths) as b:
        b.pt_init(inp.seeds, inp.conformations)
        b.pt_run(n1, S)
        mid = b.pt_read()
        t, x = b.pt_counters()
    assert (t, x) == (n1, n1 // S)
    with pt.ParallelTempering(p, inp.temperatures, inp.widths) as c:
        c.pt_init(inp.seeds, mid["conformations"])
        c.pt_set_counters(t, x)
        c.pt_set_trace(n1 + n2, (n1 + n2) // S)
        c.pt_run(n2, S)
        res, rtr = c.pt_read(), c.trace()
        assert c.pt_counters() == (n1 + n2, (n1 + n2) // S)
    assert np.array_equal(res["conformations"].view(np.uint64), full["conformations"].view(np.uint64))
    assert np.array_equal(rtr["move"][:, :, n1:], ftr["move"][:, :, n1:])
    assert np.array_equal(rtr["swap"][:, n1 // S:], ftr["swap"][:, n1 // S:])
    assert energy_close(res["energies"], full["energies"]).all()
    with pytest.raises(pt.PtError):
        with pt.ParallelTempering(p, inp.temperatures, inp.widths) as e:
            e.pt_set_counters(1, 1)          # before pt_init


def test_determinism_and_seed_locality():
    """Same seeds -> identical output; changing one ensemble's seed changes only that ensemble."""
    inp = synth.make_inputs(5, E=4)
    wl = inp.workload
    p = pt.make_params(wl.N, wl.M, wl.E)

    def run(seeds):
        with pt.ParallelTempering(p, inp.temperatures, inp.widths) as sim:
            sim.pt_init(seeds, inp.conformations)
            sim.pt_run(30, 10)
            return sim.pt_read()
    a, b = run(inp.seeds), run(inp.seeds)
    assert all(np.array_equal(a[k], b[k]) for k in a)
    s2 = inp.seeds.copy()
    s2[2] += np.uint64(12345)
    c = run(s2)
    for e in range(4):
        same = np.array_equal(a["conformations"][e], c["conformations"][e])
        assert same == (e != 2)


def test_error_paths_on_device():
    inp = synth.make_inputs(1)
    wl = inp.workload
    p = pt.make_params(wl.N, wl.M, wl.E)
    with pt.ParallelTempering(p, inp.temperatures, inp.widths) as sim:
        with pytest.raises(pt.PtError) as ei:
            sim.pt_sweeps(1)
        assert ei.value.code == pt.binding.PT_ESTATE
        bad = inp.conformations.copy()
        bad[0, 3, 5] = bad[0, 3, 4] + np.array([1.2, 0.0, 0.0])     # a bond of length 1.2 > r0 + R
        with pytest.raises(pt.PtError) as ei:
            sim.pt_init(inp.seeds, bad)
        assert ei.value.code == pt.binding.PT_EBOND
        bad = inp.conformations.copy()
        bad[0, 0, 0, 0] = np.nan
        with pytest.raises(pt.PtError) as ei:
            sim.pt_init(inp.seeds, bad)
        assert ei.value.code == pt.binding.PT_EBOND
        sim.pt_init(inp.seeds, inp.conformations)
        sim.pt_sweeps(3)
        with pytest.raises(pt.PtError) as ei:
            sim.pt_sweeps(2 ** 32)
        assert ei.value.code == pt.binding.PT_ERANGE
    # library-owned memory (cudaMalloc) instead of a torch workspace gives the same result
    outs = []
    for tw in (True, False):
        with pt.ParallelTempering(p, inp.temperatures, inp.widths, torch_workspace=tw) as sim:
            sim.pt_init(inp.seeds, inp.conformations)
            sim.pt_run(20, 10)
            outs.append(sim.pt_read())
    assert all(np.array_equal(outs[0][k], outs[1][k]) for k in outs[0])


def test_non_default_stream():
    import torch
    inp = synth.make_inputs(1)
    wl = inp.workload
    p = pt.make_params(wl.N, wl.M, wl.E)
    st = torch.cuda.Stream()
    with pt.ParallelTempering(p, inp.temperatures, inp.widths, stream=st) as sim:
        sim.pt_init(inp.seeds, inp.conformations)
        sim.pt_run(50, 10)
        a = sim.pt_read()
    with pt.ParallelTempering(p, inp.temperatures, inp.widths) as sim:
        sim.pt_init(inp.seeds, inp.conformations)
        sim.pt_run(50, 10)
        b = sim.pt_read()
    assert all(np.array_equal(a[k], b[k]) for k in a)
