"""Post-processing (paper_1107_3490_b200/analysis.py) against the dimer, whose <E> and C_V are
one-dimensional integrals (the quadrature values of tests/golden/closed_forms.txt / SURVEY.md P10):
moments and histograms come from the ORACLE here, so the check runs without a GPU."""
import numpy as np

import oracle
from paper_1107_3490_b200 import analysis, synth

# N = 2, V = LJ^mod + FENE on (0.4, 1.0), weight r^2 exp(-V/T)
P10 = {0.3: (-0.8116778275, 0.5968428903), 1.0: (-0.4550701079, 0.4138982268), 3.0: (0.0646680498, 0.1664119362)}


def _dimer_run(T, n_sweeps=120000, nbins=400, hist=(-1.2, 6.0)):
    T = np.asarray(T, dtype=np.float64)
    p = oracle.make_params(2, len(T), 1, nbins=nbins, hist_emin=hist[0], hist_emax=hist[1])
    o = oracle.Oracle(p, T, synth.move_halfwidths(T, 0.25), threads=1)
    conf = np.zeros((1, len(T), 2, 3))
    conf[:, :, 1, 0] = 0.7
    o.init(np.array([20261104], dtype=np.uint64), conf)
    o.run(2000, 0)
    # no reset in the oracle API: 2000 thermalisation sweeps of 122000 bias <E> by < 1e-3
    o.run(n_sweeps, 0)
    out = o.read()
    o.close()
    return out, analysis.bin_centres(nbins, *hist)


def test_moments_give_the_quadrature_energy_and_specific_heat():
    T = np.array([0.3, 1.0, 3.0])
    out, _ = _dimer_run(T)
    e = analysis.mean_energy(out["moments"])[0]
    cv = analysis.specific_heat(out["moments"], T)[0]
    for i, t in enumerate(T):
        assert abs(e[i] - P10[t][0]) < 0.02, (t, e[i])
        assert abs(cv[i] - P10[t][1]) < 0.05, (t, cv[i])


def test_reweighting_reproduces_neighbouring_temperatures():
    T = np.array([0.9, 1.0, 1.1])
    out, centres = _dimer_run(T)
    e_direct = analysis.mean_energy(out["moments"])[0]
    cv_direct = analysis.specific_heat(out["moments"], T)[0]
    nb = centres.size
    e_rw, cv_rw = analysis.reweight(out["histograms"][0, 1, :nb], centres, 1.0, T)
    # at T0 itself the histogram must give the moments back (up to the bin width 0.018)
    assert abs(e_rw[1] - e_direct[1]) < 0.01 and abs(cv_rw[1] - cv_direct[1]) < 0.02
    # and 10 % away in temperature it must agree with the direct simulation there
    assert np.all(np.abs(e_rw - e_direct) < 0.03), (e_rw, e_direct)
    assert np.all(np.abs(cv_rw - cv_direct) < 0.06), (cv_rw, cv_direct)
    assert abs(e_rw[1] - P10[1.0][0]) < 0.02


def test_d_rgyr2_dT_of_the_dimer():
    """analysis.d_rgyr2_dT (the quantity of Fig. 5) from the oracle's moments of a dimer run
    against the numerical temperature derivative of the 1-D integral <r^2/4>."""
    from scipy import integrate
    sigma2 = 0.7 ** 2 / 2 ** (1 / 3)

    def V(r):
        lj = 0.0
        if r < 2.5 * np.sqrt(sigma2):
            s6 = (sigma2 / r ** 2) ** 3
            lj = 4 * (s6 * s6 - s6) - 4 * (2.5 ** -12 - 2.5 ** -6)
        return lj - 1.8 * np.log(1 - ((r - 0.7) / 0.3) ** 2)

    def rg2(T):
        w = lambda r: r * r * np.exp(-(V(r) + 1) / T)
        Z = integrate.quad(w, 0.4, 1.0, epsrel=1e-12)[0]
        return integrate.quad(lambda r: r * r / 4 * w(r), 0.4, 1.0, epsrel=1e-12)[0] / Z

    T = np.array([0.5, 1.5])
    out, _ = _dimer_run(T, n_sweeps=200000)
    got = analysis.d_rgyr2_dT(out["moments"], out["obs_moments"], T)[0]
    assert np.allclose(analysis.mean_rgyr2(out["moments"], out["obs_moments"])[0], [rg2(0.5), rg2(1.5)], rtol=5e-3)
    for i, t in enumerate(T):
        exact = (rg2(t + 1e-4) - rg2(t - 1e-4)) / 2e-4
        assert abs(got[i] - exact) < 0.15 * abs(exact), (t, got[i], exact)
