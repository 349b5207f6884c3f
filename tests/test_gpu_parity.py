"""GPU-vs-oracle parity (fp64): the CUDA path, called through the C ABI, must reproduce the
oracle's trajectory decision for decision on the same seeded inputs (BASELINE.json north_star;
SURVEY.md 8(c)): 0 divergent accept/reject decisions, 0 divergent swap decisions, per-sweep
running energies within 1e-9 max(1,|E|), final conformations bit-identical, equal counters and
histograms.  The GPU swaps temperature labels, the oracle swaps conformations (PAPER.md:105 vs
:267): their agreement is itself the test of that equivalence.

Every case runs the GPU twice against one oracle run: with the move-decision trace (the TRACE=true
instantiation of the sweep kernel) and without it (the instantiation bench.py times); parity_util.both
asserts that the two really are different kernels.  The five BASELINE.json configurations run at their
full length, config 5 with all 64 ensembles.
"""
import numpy as np
import pytest

import paper_1107_3490_b200 as pt
from paper_1107_3490_b200 import synth
from parity_util import both, compare, energy_close, hist_range, run_gpu, run_oracle

pytestmark = pytest.mark.gpu


def _both(inp, n_sweeps, *, widths=None, exchange_every=None, **kw):
    """parity_util.both on an Inputs bundle; returns (report of the untraced run, its GPU output, oracle)."""
    wl = inp.workload
    w = inp.widths if widths is None else widths
    S = wl.exchange_every if exchange_every is None else exchange_every
    kw.setdefault("label", wl.name)
    reps, runs, o = both(wl.N, wl.M, wl.E, inp.temperatures, w, inp.seeds, inp.conformations, n_sweeps, S, **kw)
    last = False if False in runs else True
    if True in reps:
        assert reps[True].get("divergent_moves", 0) == 0
    return reps[last], runs[last], o


# ---- the five BASELINE.json configurations, full length, both instantiations --------------------

def test_config1_full_run():
    """N=13, M=8, 2000 sweeps, exchange every 10: the whole job, default mapping."""
    rep, g, _ = _both(synth.make_inputs(1), 2000)
    assert rep["divergent_swaps"] == 0
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


def test_config3_full_run():
    """N=55, M=64, exchange every 20, all 10^4 sweeps."""
    rep, g, _ = _both(synth.make_inputs(3), 10000, nbins=4096)
    assert g[0]["counters"] == (10000, 500)


def test_config4_full_run():
    """N=309, M=128, all 2000 sweeps, default mapping: one CTA per replica, two pair warps (5 partner iterations
    each) and two stream warps (k_sweep_ws)."""
    rep, g, _ = _both(synth.make_inputs(4), 2000, nbins=4096, expect_kernel="k_sweep_ws<double,2,5,")
    assert g[0]["launch_info"]["lanes"] == 64 and g[0]["counters"] == (2000, 100)


def test_config4_one_warp_per_replica():
    """Config 4 on the mapping that was the default before k_sweep_ws: one warp per replica, 10 unrolled partner
    iterations with the bond stream interleaved (lanes = 32), 200 sweeps."""
    _both(synth.make_inputs(4), 200, lanes=32, expect_kernel="k_sweep_group<double,32,10,")


@pytest.mark.parametrize("config_id, kernel", [(1, "k_sweep_ws<double,1,1,"), (2, "k_sweep_ws<double,1,1,"),
                                               (3, "k_sweep_ws<double,1,2,")])
def test_small_configs_default_to_the_warp_specialised_kernel(config_id, kernel):
    """Configs 1-3 (8, 32, 64 chains): the planner's default is k_sweep_ws, one pair warp and two stream warps per
    chain; 300 sweeps here, the full runs above go through the same kernel."""
    _both(synth.make_inputs(config_id), 300, expect_kernel=kernel)


@pytest.mark.parametrize("lanes", [128, 256])
def test_config4_one_cta_per_replica(lanes):
    """BASELINE.json's wording of config 4, "one CTA per replica": the long Delta-E reduction across warps
    (k_sweep_cta; slower than one warp per replica, so not the default), 60 sweeps."""
    _both(synth.make_inputs(4), 60, lanes=lanes, expect_kernel="k_sweep_cta<double")


def test_config5_full_run_all_64_ensembles():
    """The throughput batch exactly as bench.py times it: 64 ensembles x 64 replicas, N=100, 10^3 sweeps,
    exchange every 10, default mapping (k_sweep_seven<double,13,10>: 7 chains per SM sub-partition as 4 x 8 + 3 x 10
    lanes, 147 CTAs of 28 chains; the last CTA is partly filled -- chains 4088..4095 = the tail of ensemble 63 --
    and its inactive lanes clone chain C-1).
    One oracle run of all 64 ensembles; the GPU runs twice, untraced (the timed kernel) and traced; every
    decision of all 4096 chains is compared."""
    rep, g, _ = _both(synth.make_inputs(5), 1000, nbins=4096, expect_kernel="k_sweep_seven<double,13,10,")
    info = g[0]["launch_info"]
    assert info["chains_per_cta"] == 28 and info["grid"] == 147
    assert g[0]["counters"] == (1000, 100)
    assert (g[0]["histograms"].sum(-1) == 1000).all()


def test_config5_sampled_ensembles_of_the_full_batch():
    """The oracle recomputes single ensembles of the batch on their own (first, middle, last; e_offset puts
    the ensemble index into the Philox counter): the per-ensemble streams are independent of the batch."""
    inp = synth.make_inputs(5)
    wl = inp.workload
    n_sweeps, S, nbins = 100, wl.exchange_every, 4096
    hist = hist_range(wl.N)
    g, gtr = run_gpu(wl.N, wl.M, wl.E, inp.temperatures, inp.widths, inp.seeds, inp.conformations,
                     n_sweeps, S, nbins=nbins, hist=hist, trace_moves=False)
    assert energy_close(g["energies"], g["energies_full"]).all()
    for e in (0, 31, 63):
        o, otr = run_oracle(wl.N, wl.M, 1, inp.temperatures, inp.widths, inp.seeds[e:e + 1],
                            inp.conformations[e:e + 1], n_sweeps, S, nbins=nbins, hist=hist, e_offset=e)
        ge = {k: v[e:e + 1] for k, v in g.items() if isinstance(v, np.ndarray)}
        gte = {k: v[e:e + 1] for k, v in gtr.items()}
        compare(ge, gte, o, otr, N=wl.N, nbins=nbins, hist=hist, label=f"config5 ensemble {e}")


def test_mixed_mapping_at_the_papers_chain_length():
    """N = 55, 40 ensembles x 64 replicas = 2560 chains: between 4 and 7 chains per SM sub-partition, so
    the planner spreads 18 chains over every SM: sub-partition loads 5, 5, 4, 4 (k_sweep_comp<7,4,2>)."""
    N, M, E = 55, 64, 40
    T = synth.temperature_ladder(M, 0.15, 3.0)
    reps, runs, _ = both(N, M, E, T, synth.move_halfwidths(T), synth.seeds(3, E, rank=3),
                         synth.random_walk_conformations(E, M, N, seed=5564), 100, 10, label="mixed N=55",
                         expect_kernel="k_sweep_comp<double,7,4,2,")
    assert runs[False][0]["launch_info"]["chains_per_cta"] == 18


# ---- variants and edge cases ----------------------------------------------------------------

# (N, chains) -> chains per CTA and the sub-partition loads the planner must produce on 148 SMs
COMPOSED = [(40, 600, 5), (55, 4144, 28), (30, 1336, 10), (30, 2000, 14), (30, 2960, 20), (30, 3400, 23), (30, 3848, 26),
            (30, 4440, 30), (30, 4736, 32), (30, 5000, 17), (17, 1200, 9), (64, 2400, 17), (80, 3000, 21),
            (104, 1480, 10), (128, 1000, 7), (100, 2376, 17)]


@pytest.mark.parametrize("N,C,q", COMPOSED, ids=[f"N{n}_C{c}" for n, c, _ in COMPOSED])
def test_composed_ctas(N, C, q):
    """Every composition of k_sweep_comp (SM sub-partition loads 1..8 as warps of 32, 16 and 8 lanes per chain, some
    with an idle chain slot; two waves beyond 4736 chains) and of k_sweep_seven, chain lengths around the table's N,
    both instantiations:
    chains spread evenly over the SMs, so the time has no staircase in the number of replicas
    beyond the one of the most loaded sub-partition."""
    M = 8
    E = C // M
    T = synth.temperature_ladder(M, 0.3, 2.5)
    reps, runs, _ = both(N, M, E, T, synth.move_halfwidths(T), synth.seeds(8, E, rank=N),
                         synth.random_walk_conformations(E, M, N, seed=77000 + N + C), 20, 10, nbins=16,
                         label=f"composed N={N} C={C}", expect_kernel="k_sweep_seven<double,7,6," if q == 28 else "k_sweep_comp<double,")
    assert runs[False][0]["launch_info"]["chains_per_cta"] == q


def test_random_pick_mode():
    """Paper-literal monomer choice in every mapping family."""
    for lanes in (8, 32, 64):
        _both(synth.make_inputs(1), 200, lanes=lanes, select_mode=1)


def test_paper_literal_width():
    """Components uniform in [-0.01, 0.01] at every temperature."""
    _both(synth.make_inputs(1), 300, widths=synth.paper_halfwidths(8))


@pytest.mark.parametrize("config_id,n_sweeps", [(1, 2000), (3, 1000)])
def test_paper_literal_mode(config_id, n_sweeps):
    """the paper's move as one mode -- "a random monomer of the chain is picked" AND
    components uniform in [-0.01, 0.01] at every temperature -- on configs 1 and 3."""
    inp = synth.make_inputs(config_id)
    rep, g, o = _both(inp, n_sweeps, select_mode=1, widths=synth.paper_halfwidths(inp.workload.M))
    acc = g[0]["move_counts"][..., 1] / g[0]["move_counts"][..., 0]
    assert (acc > 0.5).all(), "a 0.01 cube is accepted most of the time at every temperature"


def _max_abs_energy(conf):
    import oracle
    return max(abs(oracle.total_energy(c)) for e in conf for c in e)


# (label, N, M, E, lanes, kernel the planner must pick, sweeps, exchange_every)
OVERLAP_CASES = [
    ("config1_shape", 13, 8, 1, 0, "k_sweep_ws<double,1,1,", 150, 10),
    ("config1_shape_lanes16", 13, 8, 1, 16, "k_sweep_group<double,16,1,", 150, 10),
    ("comp_13_7_4", 100, 64, 40, 0, "k_sweep_comp<double,13,7,4,", 40, 10),
    ("comp_7_4_2", 55, 64, 40, 0, "k_sweep_comp<double,7,4,2,", 60, 10),
    ("seven_13_10_partly_filled", 100, 64, 60, 0, "k_sweep_seven<double,13,10,", 30, 10),
    ("config4_shape", 309, 128, 1, 0, "k_sweep_ws<double,2,5,", 40, 20),
    ("ws_three_pair_warps", 400, 8, 1, 0, "k_sweep_ws<double,3,5,", 30, 10),
    ("config4_shape_lanes32", 309, 128, 1, 32, "k_sweep_group<double,32,10,", 40, 20),
    ("ws_1_4", 100, 16, 2, 0, "k_sweep_ws<double,1,4,", 60, 10),
    ("ws_odd_length_wrap", 37, 8, 3, 0, "k_sweep_ws<double,1,2,", 80, 7),
    ("wsg_four_chains_per_cta", 37, 8, 60, 0, "k_sweep_wsg<double,2,chains=4,", 40, 7),
    ("N100_lanes8", 100, 16, 2, 8, "k_sweep_group<double,8,13,", 60, 10),
    ("N100_lanes16", 100, 16, 2, 16, "k_sweep_group<double,16,7,", 60, 10),
    ("N100_lanes32", 100, 16, 2, 32, "k_sweep_group<double,32,4,", 60, 10),
    ("N200_lanes8_runtime_loop", 200, 8, 1, 8, "k_sweep_group<double,8,0,", 30, 10),
    ("cta128", 100, 16, 1, 128, "k_sweep_cta<double", 40, 10),
]


@pytest.mark.parametrize("case", OVERLAP_CASES, ids=[c[0] for c in OVERLAP_CASES])
def test_overlapping_start_large_energies(case):
    """Plain random walks (d_min = 0: overlaps allowed, the start of SURVEY.md 8(d)) and wide moves in front
    of every kernel family, both instantiations: huge initial energies, Delta E from -1e6 to +1e6 and beyond,
    bond-range rejections (E_new = +inf).  Decisions, coordinates, counters and histograms must agree exactly.
    The running energy keeps the rounding of the largest value held since it was last re-based on Eq. (4)
    (pt_init; exchange events 2^k - 1, R22), so the 1e-9 energy criterion refers to that scale
    (parity_util.rebased_floor): the largest |E| of the ensemble since the last re-basing."""
    label, N, M, E, lanes, kernel, n_sweeps, S = case
    T = synth.temperature_ladder(M, 0.2, 3.0)
    conf = synth.random_walk_conformations(E, M, N, seed=9900 + N + M + E, d_min=0.0)
    e0 = _max_abs_energy(conf)
    assert e0 > 1e3, "the start must contain overlaps"
    reps, runs, _ = both(N, M, E, T, synth.move_halfwidths(T, 0.6), synth.seeds(9, E), conf, n_sweeps, S,
                         lanes=lanes, nbins=64, start_energy=e0, label=label, expect_kernel=kernel)
    assert runs[False][0]["move_counts"][..., 2].sum() > 0, "the wide moves should have produced bond-range rejections"


@pytest.mark.parametrize("config_id", [1, 2, 3, 4, 5])
def test_every_config_from_the_plain_walk(config_id):
    """SURVEY.md 8(d) input recipe taken literally: each of the five configurations started from plain random
    walks with overlaps, 200 sweeps at its own widths and exchange cadence, both instantiations.  Energy scale:
    parity_util.rebased_floor -- the initial energies (1e10 ... 1e33 for the big batches) until the first
    re-basing of E_run, the energies at the last re-basing afterwards; the last 40 sweeps follow the re-basing
    at sweep 160 and must meet the plain criterion 1e-9 max(1e3, |E|)."""
    wl = synth.CONFIGS[config_id]
    T = synth.temperature_ladder(wl.M, wl.T_min, wl.T_max)
    conf = synth.random_walk_conformations(wl.E, wl.M, wl.N, seed=8800 + config_id, d_min=0.0)
    e0 = _max_abs_energy(conf)
    assert e0 > 1e3
    reps, runs, o = both(wl.N, wl.M, wl.E, T, synth.move_halfwidths(T), synth.seeds(config_id, wl.E, rank=5), conf, 200,
                         wl.exchange_every, nbins=64, start_energy=e0, label=f"{wl.name} plain walk (start {e0:.3g})")
    tail_g, tail_o = runs[False][1]["energy"][..., 160:], o[1]["energy"][..., 160:]
    assert energy_close(tail_g, tail_o, floor=1e3).all(), float(np.abs(tail_g - tail_o).max())


def test_library_random_walk_start():
    """pt_init(seeds, NULL): the library's own seeded walk: bonds of length r0 in
    directions z = s(w0), phi = 2 pi u(w1) from Philox tag INIT.  Restated here in NumPy from the recipe with
    the oracle's generator; equal up to the last bits of the host's sin / cos."""
    import oracle
    N, M, E = 30, 4, 3
    T = synth.temperature_ladder(M, 0.5, 2.0)
    seeds = synth.seeds(2, E, rank=9)
    p = pt.make_params(N, M, E)
    with pt.ParallelTempering(p, T, synth.move_halfwidths(T)) as sim:
        sim.pt_init(seeds, None)
        a = sim.pt_read()
        sim.pt_init(seeds, None)
        b = sim.pt_read()
        sim.pt_run(20, 10)
        assert energy_close(sim.pt_read()["energies"], sim.pt_recompute_energy(), floor=np.abs(a["energies"]).max()).all()
    x = a["conformations"]
    assert np.array_equal(x, b["conformations"])
    assert np.allclose(np.linalg.norm(np.diff(x, axis=2), axis=-1), 0.7, atol=1e-13)
    ref = np.zeros_like(x)
    for e in range(E):
        key = [int(seeds[e]) & 0xFFFFFFFF, int(seeds[e]) >> 32]
        for i in range(M):
            for n in range(1, N):
                w = oracle.philox([n, 0, e, (3 << 24) | i], key)
                z = (2 * w[0] + 1 - 2 ** 32) / 2.0 ** 32
                phi = 2 * np.pi * (w[1] + 0.5) / 2.0 ** 32
                sxy = np.sqrt(1 - z * z)
                ref[e, i, n] = ref[e, i, n - 1] + 0.7 * np.array([sxy * np.cos(phi), sxy * np.sin(phi), z])
    assert np.allclose(x, ref, rtol=0, atol=1e-12)
    for e in range(E):
        for i in range(M):
            assert a["energies"][e, i] == pytest.approx(oracle.total_energy(x[e, i]), rel=1e-12)


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


# (N, M, E, kernel the planner must pick): the classes of the warp-specialised kernel and its limits
WS_CASES = [
    (6, 8, 1, "k_sweep_ws<double,1,1,"),           # the shortest chain it takes
    (5, 8, 1, "k_sweep_group<double,"),            # below: the stream warps' table reads would meet commits
    (64, 8, 2, "k_sweep_ws<double,1,2,"),
    (65, 16, 1, "k_sweep_ws<double,1,3,"),
    (129, 16, 1, "k_sweep_ws<double,2,3,"),
    (200, 8, 1, "k_sweep_ws<double,2,4,"),
    (330, 6, 1, "k_sweep_ws<double,3,4,"),
    (200, 100, 3, "k_sweep_ws<double,1,7,"),       # 300 chains: one pair warp each
    (480, 4, 1, "k_sweep_ws<double,3,5,"),
    (600, 4, 1, "k_sweep_ws<double,3,7,"),         # beyond the unrolled one-warp kernels: before, one CTA per replica
    (1000, 2, 1, "k_sweep_ws<double,3,15,"),
    (55, 394, 1, "k_sweep_ws<double,1,2,"),        # the last chain count with a CTA per chain (N = 55) ...
    (55, 395, 1, "k_sweep_wsg<double,2,chains=4,"),   # ... beyond: four chains per CTA share the stream warps (397: a partly filled CTA)
    (55, 397, 1, "k_sweep_wsg<double,2,chains=4,"),
    (20, 5, 100, "k_sweep_wsg<double,1,chains=4,"),    # the chains of a CTA belong to different ensembles; fused exchange
    (30, 148, 5, "k_sweep_wsg<double,1,chains=4,"),    # 740 chains: two such CTAs per SM
    (55, 593, 1, "k_sweep_comp<double,7,4,2,"),        # N > 32 beyond 592 chains: composed CTAs
    (100, 500, 1, "k_sweep_wsg<double,4,chains=4,"),   # up to N = 128 between 395 and 592 chains
    (150, 500, 1, "k_sweep_group<double,32,7,"),       # longer chains there: one warp per chain
]


@pytest.mark.parametrize("N,M,E,kernel", WS_CASES, ids=[f"N{c[0]}_C{c[1] * c[2]}" for c in WS_CASES])
def test_warp_specialised_classes(N, M, E, kernel):
    """k_sweep_ws for one, two and three pair warps, short and long partner loops, chain counts up to where the planner
    leaves it, 60 sweeps with exchanges, both instantiations (pt_sweep_ws.cuh)."""
    T = synth.temperature_ladder(M, 0.3, 2.5)
    reps, runs, _ = both(N, M, E, T, synth.move_halfwidths(T), synth.seeds(11, E),
                         synth.random_walk_conformations(E, M, N, seed=7000 + N + M), 60, 10, nbins=32,
                         label=f"ws N={N} C={M * E}", expect_kernel=kernel)
    assert reps[False]["divergent_swaps"] == 0


@pytest.mark.parametrize("N,M,E,S", [(20, 5, 3, 3), (37, 8, 2, 1), (100, 7, 2, 4)])
def test_fused_exchange_equals_separate_calls(N, M, E, S):
    """Under pt_run the warp-specialised kernel does the exchange event at the end of the sweep launch (the last CTA of
    every ensemble to finish); pt_sweeps + pt_exchange called one by one use the exchange kernel.  Both against the
    oracle: odd and even numbers of temperatures, several ensembles, exchange after every S sweeps (the events before
    which E_run is re-based, 0, 1, 3, 7, ..., take the separate path in both)."""
    T = synth.temperature_ladder(M, 0.3, 2.5)
    args = (N, M, E, T, synth.move_halfwidths(T), synth.seeds(13, E), synth.random_walk_conformations(E, M, N, seed=8100 + N))
    for stepwise in (False, True):
        reps, runs, _ = both(*args, 40 * S, S, nbins=32, stepwise=stepwise, label=f"fused exchange N={N} M={M} stepwise={stepwise}",
                             expect_kernel="k_sweep_ws<double,")
        assert reps[False]["divergent_swaps"] == 0 and runs[False][0]["counters"] == (40 * S, 40)


@pytest.mark.parametrize("N,M,E,n,S", [(30, 32, 1, 40000, 10), (40, 16, 8, 10000, 7), (150, 12, 2, 3000, 5), (24, 8, 60, 3000, 5)])
def test_warp_specialised_long_runs(N, M, E, n, S):
    """Long untraced runs of k_sweep_ws (one, one and two pair warps; 3.8e7, 5.1e7, 1.1e7 decisions; thousands of fused
    exchange events): a rare ordering fault between pair warps, stream warps and the committing thread would surface as
    one divergent decision, and every later coordinate would differ.  Final coordinates bitwise, counters, histograms."""
    T = synth.temperature_ladder(M, 0.3, 3.0)
    args = (N, M, E, T, synth.move_halfwidths(T), synth.seeds(21, E), synth.random_walk_conformations(E, M, N, seed=N + M), n, S)
    g, _ = run_gpu(*args, trace_sweeps=0, recompute=False)
    o, _ = run_oracle(*args, trace_sweeps=0)
    assert g["kernel"].startswith(("k_sweep_ws<double,", "k_sweep_wsg<double,")) and g["kernel"].endswith("trace=0>"), g["kernel"]
    assert np.array_equal(g["conformations"].view(np.uint64), o["conformations"].view(np.uint64))
    assert np.array_equal(g["move_counts"], o["move_counts"]) and np.array_equal(g["swap_counts"], o["swap_counts"])
    assert np.array_equal(g["histograms"], o["histograms"])


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
