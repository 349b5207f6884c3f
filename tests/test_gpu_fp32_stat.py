"""fp32 path (north_star (d)): per-temperature <E> and C_V = beta^2 (<E^2> - <E>^2)
(Eq. 7) within 3 sigma of the fp64 run.  Config 5: sigma = standard error over the 64
independent ensembles.  Config 3 (N = 55, M = 64): 32 independent ensembles of that shape.  Both precisions start from the same seeds, so their trajectories coincide
until the first rounding-induced decision flip and are independent samples afterwards.

With 64 temperatures x 2 observables = 128 comparisons, a 3-sigma excursion is expected in ~1 of 3
honest runs; the criterion is therefore: no |z| above 4, at most 2 of the 128 above 3, and the
z-scores unbiased (|mean z| < 0.5) -- a systematic precision effect would shift all of them.
Sigma is always the standard error across INDEPENDENT ensembles (64 for config 5, 32 for the config-3
shape): no autocorrelation model enters the criterion."""
import numpy as np
import pytest

import paper_1107_3490_b200 as pt
from paper_1107_3490_b200 import synth

pytestmark = pytest.mark.gpu


def _run_blocks(inp, precision, n_discard, n_blocks, block_sweeps, E=None):
    """Returns per-block (mean E, mean E^2) arrays of shape [n_blocks][E][M]."""
    wl = inp.workload
    p = pt.make_params(wl.N, wl.M, wl.E, precision=precision, nbins=0)
    S = wl.exchange_every
    m1, m2 = [], []
    with pt.ParallelTempering(p, inp.temperatures, inp.widths) as sim:
        sim.pt_init(inp.seeds, inp.conformations)
        sim.pt_run(n_discard, S)
        for _ in range(n_blocks):
            sim.pt_reset_stats()
            sim.pt_run(block_sweeps, S)
            mom = sim.pt_read(energies=False, histograms=False, move_counts=False, swap_counts=False,
                              conformations=False, obs_moments=False)["moments"]
            assert (mom[..., 0] == block_sweeps).all()
            m1.append(mom[..., 1] / block_sweeps)
            m2.append(mom[..., 2] / block_sweeps)
        info = sim.pt_launch_info()
    return np.array(m1), np.array(m2), info


def _zscores(a, sa, b, sb):
    return (a - b) / np.sqrt(sa * sa + sb * sb)


def _check(z, label):
    z = np.asarray(z).ravel()
    assert np.isfinite(z).all(), label
    assert np.abs(z).max() < 4.0, (label, float(np.abs(z).max()))
    assert int((np.abs(z) > 3.0).sum()) <= 2, (label, int((np.abs(z) > 3.0).sum()))
    assert abs(z.mean()) < 0.5, (label, float(z.mean()))


def test_config5_fp32_matches_fp64_over_64_ensembles():
    inp = synth.make_inputs(5)
    wl = inp.workload
    beta2 = (1.0 / inp.temperatures) ** 2
    res = {}
    for prec in (pt.PT_F64, pt.PT_F32):
        # one block = sweeps 200..999 of the 10^3-sweep job; the 64 ensembles are the samples
        m1, m2, info = _run_blocks(inp, prec, 200, 1, 800)
        e = m1[0]                                  # [E][M]
        cv = beta2 * (m2[0] - m1[0] ** 2)          # [E][M]
        res[prec] = (e.mean(0), e.std(0, ddof=1) / np.sqrt(wl.E), cv.mean(0), cv.std(0, ddof=1) / np.sqrt(wl.E))
    a, b = res[pt.PT_F64], res[pt.PT_F32]
    _check(np.concatenate([_zscores(a[0], a[1], b[0], b[1]), _zscores(a[2], a[3], b[2], b[3])]), "config 5")
    # the two precisions are not the same trajectory (the comparison is not vacuous) ...
    assert not np.allclose(a[0], b[0], rtol=1e-12, atol=0)
    # ... and agree physically: <E> rises with T
    assert b[0][0] < b[0][-1]


def test_config3_fp32_full_length_is_sane():
    """Config 3 as BASELINE.json states it (ONE ensemble, 10^4 sweeps), fp32 beside fp64.  A single ensemble has
    no honest error bar at this length: block means of 400 sweeps are correlated with rho ~ 0.8 (the replicas
    share slow modes through the exchange), so the 3-sigma criterion of record for this shape is the
    32-ensemble test below.  Here: the run completes, E_run stays on the Eq.-4 energy of
    the fp32 conformation, and <E>(T) agrees with fp64 to a few per cent of the energy scale at every T."""
    inp = synth.make_inputs(3)
    wl = inp.workload
    res = {}
    for prec in (pt.PT_F64, pt.PT_F32):
        p = pt.make_params(wl.N, wl.M, wl.E, precision=prec, nbins=0)
        with pt.ParallelTempering(p, inp.temperatures, inp.widths) as sim:
            sim.pt_init(inp.seeds, inp.conformations)
            sim.pt_run(2000, wl.exchange_every)
            sim.pt_reset_stats()
            sim.pt_run(8000, wl.exchange_every)
            out = sim.pt_read()
            efull = sim.pt_recompute_energy()
        assert np.abs(out["energies"] - efull).max() < (1e-9 * wl.N if prec == pt.PT_F64 else 5e-3)
        res[prec] = out["moments"][0, :, 1] / out["moments"][0, :, 0]
    a, b = res[pt.PT_F64], res[pt.PT_F32]
    assert not np.allclose(a, b, rtol=1e-12, atol=0)
    assert np.abs(a - b).max() < 0.06 * np.abs(a).max(), float(np.abs(a - b).max())
    assert b[0] < b[-1]


def test_config3_shape_fp32_matches_fp64_over_32_ensembles():
    """The statistically sound version of the config-3 check: the same N, M, ladder and exchange
    cadence, 32 independent ensembles (sigma = standard error across them), every fp32 mapping."""
    N, M, E = 55, 64, 32
    T = synth.temperature_ladder(M, 0.15, 3.0)
    w = synth.move_halfwidths(T)
    conf = synth.random_walk_conformations(E, M, N, seed=1107349003)
    seeds = synth.seeds(3, E, rank=7)
    beta2 = (1.0 / T) ** 2
    res = {}
    for prec, lanes in ((pt.PT_F64, 0), (pt.PT_F32, 0), (pt.PT_F32, 8), (pt.PT_F32, 16), (pt.PT_F32, 128)):
        p = pt.make_params(N, M, E, precision=prec, nbins=0, lanes=lanes)
        with pt.ParallelTempering(p, T, w) as sim:
            sim.pt_init(seeds, conf)
            sim.pt_run(1000, 20)
            sim.pt_reset_stats()
            sim.pt_run(3000, 20)
            mom = sim.pt_read(energies=False, histograms=False, move_counts=False, swap_counts=False,
                              conformations=False, obs_moments=False)["moments"]
        e = mom[..., 1] / 3000
        cv = beta2 * (mom[..., 2] / 3000 - e ** 2)
        res[(prec, lanes)] = (e.mean(0), e.std(0, ddof=1) / np.sqrt(E), cv.mean(0), cv.std(0, ddof=1) / np.sqrt(E))
    a = res[(pt.PT_F64, 0)]
    for key, b in res.items():
        if key[0] == pt.PT_F32:
            _check(np.concatenate([_zscores(a[0], a[1], b[0], b[1]), _zscores(a[2], a[3], b[2], b[3])]),
                   f"config-3 shape, fp32 lanes={key[1]}")


@pytest.mark.parametrize("lanes", [8, 16, 32, 128])
def test_fp32_every_mapping_is_sane(lanes):
    """Every lane mapping of the fp32 kernels: running energy equals the fp64 full recompute of the
    fp32 conformation to fp32 accuracy, bonds stay in range, counters add up."""
    inp = synth.make_inputs(2)
    wl = inp.workload
    p = pt.make_params(wl.N, wl.M, wl.E, precision=pt.PT_F32, nbins=64, lanes=lanes,
                       hist_emin=-5.0 * wl.N, hist_emax=3.0 * wl.N)
    with pt.ParallelTempering(p, inp.temperatures, inp.widths) as sim:
        sim.pt_init(inp.seeds, inp.conformations)
        sim.pt_run(500, wl.exchange_every)
        out = sim.pt_read()
        efull = sim.pt_recompute_energy()
    # E_run accumulates fp32-accurate dE in fp64: drift ~ sqrt(steps) * 1e-6 * |dE|
    assert np.abs(out["energies"] - efull).max() < 2e-2, float(np.abs(out["energies"] - efull).max())
    b = np.linalg.norm(np.diff(out["conformations"], axis=2), axis=-1)
    assert (np.abs(b - 0.7) < 0.3 + 1e-6).all()
    assert (out["move_counts"][..., 0] == wl.N * 500).all()
    assert (out["histograms"].sum(-1) == 500).all()
    acc = out["move_counts"][..., 1] / out["move_counts"][..., 0]
    assert (acc > 0.05).all() and (acc < 0.99).all()


def test_fp32_running_energy_does_not_drift():
    """E_run collects fp32-accurate increments; the library replaces it by the Eq.-4 sum every 8th exchange
    event (the paper's kernel recomputed the energy every sweep), so the distance to the full
    recompute stays bounded however long the run is."""
    inp = synth.make_inputs(2)
    wl = inp.workload
    p = pt.make_params(wl.N, wl.M, wl.E, precision=pt.PT_F32, nbins=0)
    worst = 0.0
    with pt.ParallelTempering(p, inp.temperatures, inp.widths) as sim:
        sim.pt_init(inp.seeds, inp.conformations)
        for _ in range(10):
            sim.pt_run(3000, wl.exchange_every)
            worst = max(worst, float(np.abs(sim.pt_read()["energies"] - sim.pt_recompute_energy()).max()))
    assert worst < 5e-3, worst
