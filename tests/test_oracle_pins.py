"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these tests touches the CUDA path.  Expected values are either the paper's
constants worked out by hand (tests/golden/closed_forms.txt), published known answers of
Philox4x32-10 (tests/golden/philox4x32_10_kat.txt), numerical quadrature of the Boltzmann
weight done here with SciPy/NumPy, or exact invariants.
"""
from pathlib import Path

import numpy as np
import pytest
from scipy import integrate

import oracle
from paper_1107_3490_b200 import synth

GOLD = Path(__file__).parent / "golden"

# the paper's constants, typed here independently of the oracle
EPS, R0, RFENE, K, RCS = 1.0, 0.7, 0.3, 40.0, 2.5
SIGMA = R0 / 2.0 ** (1.0 / 6.0)
RC = RCS * SIGMA


def _closed_forms():
    out = {}
    for line in (GOLD / "closed_forms.txt").read_text().splitlines():
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split()
            out[k] = float(v)
    return out


CF = _closed_forms()


# ---- independent NumPy statement of Eq. (1)-(3), used only as the integrand of the quadratures
def V_lj_mod(r):
    r = np.asarray(r, dtype=np.float64)
    rr = np.minimum(r, RC)
    f = lambda x: 4.0 * EPS * ((SIGMA / x) ** 12 - (SIGMA / x) ** 6)
    return f(rr) - f(RC)


def V_fene(r):
    r = np.asarray(r, dtype=np.float64)
    return -0.5 * K * RFENE ** 2 * np.log(1.0 - ((r - R0) / RFENE) ** 2)


# ------------------------------------------------------------------ P7: random stream
def test_philox_known_answers():
    n = 0
    for line in (GOLD / "philox4x32_10_kat.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        w = [int(t, 16) for t in line.split()]
        assert oracle.philox(w[0:4], w[4:6]) == w[6:10]
        n += 1
    assert n == 3


def test_philox_is_a_bijection_of_the_counter_and_sensitive_to_every_input_word():
    base = oracle.philox([1, 2, 3, 4], [5, 6])
    seen = {tuple(base)}
    for pos in range(4):
        c = [1, 2, 3, 4]; c[pos] ^= 1
        seen.add(tuple(oracle.philox(c, [5, 6])))
    for pos in range(2):
        k = [5, 6]; k[pos] ^= 1
        seen.add(tuple(oracle.philox([1, 2, 3, 4], k)))
    assert len(seen) == 7
    # avalanche: one flipped counter bit changes about half of the 128 output bits
    flips = []
    for bit in range(32):
        o = oracle.philox([1 ^ (1 << bit), 2, 3, 4], [5, 6])
        flips.append(sum(bin(a ^ b).count("1") for a, b in zip(o, base)))
    assert 48 < np.mean(flips) < 80


def test_word_to_number_maps():
    L = oracle.lib()
    assert L.orc_word_to_u01(0) == 2.0 ** -33
    assert L.orc_word_to_u01(0xFFFFFFFF) == 1.0 - 2.0 ** -33
    assert L.orc_word_to_sym(0) == -1.0 + 2.0 ** -32
    assert L.orc_word_to_sym(0xFFFFFFFF) == 1.0 - 2.0 ** -32
    assert L.orc_word_to_sym(0x7FFFFFFF) == -(2.0 ** -32) and L.orc_word_to_sym(0x80000000) == 2.0 ** -32
    for w in [0, 1, 12345, 0x7FFFFFFF, 0x80000000, 0xDEADBEEF]:
        assert L.orc_word_to_sym(w) == -L.orc_word_to_sym(0xFFFFFFFF - w)   # symmetric, never 0
        assert 0.0 < L.orc_word_to_u01(w) < 1.0
    # moments of the stream the moves use: counter (k, t, e, i), key = seed
    ws = np.array([oracle.philox([k, 0, 0, 0], [1, 0]) for k in range(25000)], dtype=np.uint64)
    u = (ws.astype(np.float64).ravel() + 0.5) / 2.0 ** 32
    assert abs(u.mean() - 0.5) < 4 * np.sqrt(1 / 12 / u.size)
    assert abs(u.var() - 1 / 12) < 4 * np.sqrt(1 / 180 / u.size)
    assert abs(np.corrcoef(u[:-1], u[1:])[0, 1]) < 4 / np.sqrt(u.size)


# ------------------------------------------------------------------ P1-P4: closed forms
def test_constants():
    assert CF["sigma"] == pytest.approx(SIGMA, rel=1e-15)
    assert CF["rc2"] == pytest.approx(RC * RC, rel=1e-15)
    # E_LJ(r_c) via the oracle: E_mod(r) - E_LJ(r) is the constant -E_LJ(r_c) inside the cutoff
    r = 0.9
    e_plain = 4 * ((SIGMA / r) ** 12 - (SIGMA / r) ** 6)
    assert oracle.lj_mod(r * r) - e_plain == pytest.approx(-CF["E_LJ_rc"], abs=1e-14)


@pytest.mark.parametrize("key,r", [("lj_mod_r0.5", 0.5), ("lj_mod_rsigma", SIGMA), ("lj_mod_r0.7", 0.7),
                                   ("lj_mod_r1.0", 1.0), ("lj_mod_r1.4", 1.4)])
def test_lj_mod_closed_forms(key, r):
    assert oracle.lj_mod(r * r) == pytest.approx(CF[key], rel=2e-12, abs=2e-12)


def test_lj_mod_cutoff_minimum_and_continuity():
    assert oracle.lj_mod(RC * RC) == 0.0
    assert oracle.lj_mod(1.0000001 * RC * RC) == 0.0
    assert oracle.lj_mod(100.0) == 0.0
    assert abs(oracle.lj_mod((RC * (1 - 1e-9)) ** 2)) < 1e-9            # continuous at r_c
    assert oracle.lj_mod((RC * 0.999) ** 2) < 0.0                       # attractive just inside
    h = 1e-5                                                            # "minimum of the potential is at r0"
    e0, em, ep = oracle.lj_mod(R0 ** 2), oracle.lj_mod((R0 - h) ** 2), oracle.lj_mod((R0 + h) ** 2)
    assert em > e0 and ep > e0 and abs(ep - em) / (2 * h) < 1e-3
    assert oracle.lj_mod(1e-60) == np.inf                               # nearly overlapping monomers
    assert not np.isfinite(oracle.lj_mod(0.0))                          # coincident: inf - inf = NaN, never accepted


@pytest.mark.parametrize("key,r", [("fene_r0.7", 0.7), ("fene_r0.85", 0.85), ("fene_r0.55", 0.55),
                                   ("fene_r0.99", 0.99), ("fene_r0.41", 0.41)])
def test_fene_closed_forms(key, r):
    assert oracle.fene(r * r) == pytest.approx(CF[key], rel=1e-11, abs=1e-13)


def test_fene_range_minimum_and_divergence():
    # "has its minimum also at r0 and diverges for r -> r0 +- R"
    assert oracle.fene(1.0) == np.inf and oracle.fene(1.21) == np.inf and oracle.fene(0.39 ** 2) == np.inf
    assert oracle.fene(0.0) == np.inf
    assert oracle.fene(0.999999 ** 2) > 20.0 and oracle.fene(0.400001 ** 2) > 20.0
    h = 1e-5
    assert oracle.fene((R0 + h) ** 2) > 0 and oracle.fene((R0 - h) ** 2) > 0
    assert oracle.fene((R0 + h) ** 2) == pytest.approx(oracle.fene((R0 - h) ** 2), rel=1e-4)


def _line(n, a=R0):
    x = np.zeros((n, 3)); x[:, 0] = a * np.arange(n); return x


def test_total_energy_of_hand_placed_chains():
    a = R0
    tri = np.array([[0, 0, 0], [a, 0, 0], [a / 2, a * np.sqrt(3) / 2, 0]])
    tet = np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], dtype=float) * (a / (2 * np.sqrt(2)))
    assert oracle.total_energy(_line(2)) == pytest.approx(CF["E_dimer_r0"], abs=1e-12)
    assert oracle.total_energy(tri) == pytest.approx(CF["E_triangle_r0"], abs=1e-12)
    assert oracle.total_energy(tet) == pytest.approx(CF["E_tetrahedron_r0"], abs=1e-12)
    assert oracle.total_energy(_line(4)) == pytest.approx(CF["E_line4_r0"], abs=1e-11)
    assert oracle.total_energy(_line(5)) == pytest.approx(CF["E_line5_r0"], abs=1e-11)
    # bonded pairs carry LJ *and* FENE: a stretched trimer, spacing 0.8
    e = 2 * (float(V_lj_mod(0.8)) + float(V_fene(0.8))) + float(V_lj_mod(1.6))
    assert oracle.total_energy(_line(3, 0.8)) == pytest.approx(e, rel=1e-13)
    assert float(V_lj_mod(1.6)) == 0.0


# ------------------------------------------------------------------ P5, P6: symmetry, pair enumeration
def _random_chain(rng, n):
    return synth.random_walk_conformations(1, 1, n, int(rng.integers(1 << 30)))[0, 0]


def test_energy_symmetries():
    rng = np.random.default_rng(5)
    for n in (2, 3, 13, 30, 55):
        x = _random_chain(rng, n)
        e = oracle.total_energy(x)
        q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
        for y in (x + rng.normal(size=3), x @ q.T, x * np.array([1, 1, -1.0]), x[::-1].copy()):
            assert oracle.total_energy(y) == pytest.approx(e, rel=1e-12, abs=1e-12)


def _listing4_pairs(N):
    """The pair-index map of the paper's Listing 4: N threads x floor(N/2)
    iterations; the guard i != N-2-i keeps row N/2-1 from being visited twice for even N."""
    pairs = []
    for i in range(N // 2):
        for tx in range(N):
            if tx > i:
                i1, i2 = i, tx
            else:
                i1 = N - 2 - i
                i2 = i1 + 1 + tx
                if i == N - 2 - i:
                    continue
            pairs.append((i1, i2))
    return pairs


@pytest.mark.parametrize("N", [2, 3, 4, 13, 30, 55, 100, 309])
def test_listing4_pair_map_equals_plain_double_loop(N):
    pairs = _listing4_pairs(N)
    assert len(pairs) == N * (N - 1) // 2
    assert set(pairs) == {(i, j) for i in range(N) for j in range(i + 1, N)}


def test_total_energy_equals_sum_over_listing4_pairs():
    rng = np.random.default_rng(6)
    for n in (13, 30):
        x = _random_chain(rng, n)
        d = lambda i, j: np.linalg.norm(x[i] - x[j])
        e = sum(float(V_lj_mod(d(i, j))) for i, j in _listing4_pairs(n))
        e += sum(float(V_fene(d(i, i + 1))) for i in range(n - 1))
        assert oracle.total_energy(x) == pytest.approx(e, rel=1e-12)


# ------------------------------------------------------------------ P8: local Delta E = E(C') - E(C)
def test_delta_energy_equals_full_difference():
    rng = np.random.default_rng(8)
    n_ok = n_broken = 0
    for n in (2, 3, 13, 55):
        for _ in range(60):
            x = _random_chain(rng, n)
            m = int(rng.integers(n))
            xn = x[m] + rng.uniform(-1.0, 1.0, size=3) * (0.15 if _ % 2 else 0.45)
            dE, ok = oracle.delta_energy(x, m, xn)
            y = x.copy(); y[m] = xn
            full = oracle.total_energy(y) - oracle.total_energy(x)
            if ok:
                n_ok += 1
                assert dE == pytest.approx(full, rel=1e-10, abs=1e-10 * max(1.0, abs(oracle.total_energy(x))))
            else:
                n_broken += 1
                assert dE == np.inf and full == np.inf
    assert n_ok > 50 and n_broken > 20


# ------------------------------------------------------------------ helpers for the sampling pins
def _run(N, T, widths, E, n_sweeps, exchange_every=0, select_mode=0, seed0=77, threads=4):
    T = np.asarray(T, dtype=np.float64)
    M = T.size
    p = oracle.make_params(N, M, E, select_mode=select_mode, nbins=64, hist_emin=-5.0 * N, hist_emax=3.0 * N)
    o = oracle.Oracle(p, T, widths, threads=threads)
    conf = synth.random_walk_conformations(E, M, N, seed0)
    o.init(np.arange(E, dtype=np.uint64) + np.uint64(seed0 * 1000), conf)
    tr = o.enable_trace(n_sweeps, (n_sweeps // exchange_every) if exchange_every else 0, moves=False,
                        swaps=False, energy=True, obs=True)
    o.run(n_sweeps, exchange_every)
    return o, tr


def _mean_se(per_ensemble):
    a = np.asarray(per_ensemble)
    return a.mean(0), a.std(0, ddof=1) / np.sqrt(a.shape[0])


def _dimer_exact(T):
    """<r>, <E>, C_V of the dimer from the 1-D integral of r^2 exp(-V(r)/T) over (0.4, 1.0)."""
    V = lambda r: float(V_lj_mod(r) + V_fene(r))
    lo, hi = R0 - RFENE, R0 + RFENE
    w = lambda r: r * r * np.exp(-(V(r) + 1.0) / T)
    Z = integrate.quad(w, lo, hi, epsabs=0, epsrel=1e-12, limit=400)[0]
    avg = lambda f: integrate.quad(lambda r: f(r) * w(r), lo, hi, epsabs=0, epsrel=1e-12, limit=400)[0] / Z
    r1, e1, e2 = avg(lambda r: r), avg(V), avg(lambda r: V(r) ** 2)
    return r1, e1, (e2 - e1 * e1) / T ** 2


DIMER_T = [0.3, 1.0, 3.0]
# SURVEY.md pin P10 quotes these quadrature values; they are recomputed here and must agree
DIMER_QUOTED = {0.3: (0.7238755708, -0.8116778275, 0.5968428903),
                1.0: (0.7599508697, -0.4550701079, 0.4138982268),
                3.0: (0.7924920977, 0.0646680498, 0.1664119362)}


def test_dimer_quadrature_matches_quoted_values():
    for T in DIMER_T:
        assert _dimer_exact(T) == pytest.approx(DIMER_QUOTED[T], rel=2e-8)


@pytest.mark.parametrize("select_mode", [0, 1])
def test_dimer_sampling_matches_boltzmann_integral(select_mode):
    """P10: for N = 2 the sampled bond length follows r^2 exp(-beta V(r)).  A wrong sign, a
    dropped term, a biased proposal or a wrong acceptance rule moves <E>, <r>, C_V or the
    histogram."""
    T = np.array(DIMER_T)
    E, n_sweeps, burn = 48, 24000, 2000
    o, tr = _run(2, T, 0.1 * np.sqrt(T), E, n_sweeps, select_mode=select_mode)
    en = tr["energy"][:, :, burn:]
    r = np.sqrt(tr["ree2"][:, :, burn:])
    for i, Ti in enumerate(T):
        r_ex, e_ex, cv_ex = _dimer_exact(Ti)
        m, se = _mean_se(en[:, i].mean(-1))
        assert se < 0.01 and abs(m - e_ex) < 4.0 * se
        m, se = _mean_se(r[:, i].mean(-1))
        assert se < 0.002 and abs(m - r_ex) < 4.0 * se
        m, se = _mean_se(en[:, i].var(-1) / Ti ** 2)
        assert se < 0.03 * cv_ex + 0.01 and abs(m - cv_ex) < 4.0 * se + 0.002 * cv_ex
        # bond-length histogram in 8 coarse bins: per-bin probability vs the integral
        edges = np.linspace(0.4, 1.0, 9)
        V = lambda x: float(V_lj_mod(x) + V_fene(x))
        w = lambda x: x * x * np.exp(-(V(x) + 1.0) / Ti)
        Z = integrate.quad(w, 0.4, 1.0, epsrel=1e-11, limit=400)[0]
        for b in range(8):
            p_ex = integrate.quad(w, edges[b], edges[b + 1], epsrel=1e-10, limit=400)[0] / Z
            frac = ((r[:, i] >= edges[b]) & (r[:, i] < edges[b + 1])).mean(-1)
            m, se = _mean_se(frac)
            assert abs(m - p_ex) < 4.5 * se + 1e-5, (Ti, b, m, p_ex, se)
    # energy moments and the E_run invariant come out of read() consistently with the trace
    out = o.read()
    assert np.allclose(out["moments"][:, :, 0], n_sweeps)
    assert np.allclose(out["moments"][:, :, 1], tr["energy"].sum(-1), rtol=1e-12)
    assert out["histograms"].sum(-1).min() == n_sweeps


def _trimer_exact(T, n=96):
    """<E>, C_V, <r13> of the trimer: 3-D Gauss-Legendre over (r12, r23, cos theta)."""
    g, wg = np.polynomial.legendre.leggauss(n)
    r = R0 + RFENE * g                       # (0.4, 1.0)
    wr = RFENE * wg
    c, wc = g, wg                            # cos(theta) in (-1, 1)
    r12, r23, ct = np.meshgrid(r, r, c, indexing="ij")
    W = wr[:, None, None] * wr[None, :, None] * wc[None, None, :]
    r13 = np.sqrt(r12 ** 2 + r23 ** 2 - 2 * r12 * r23 * ct)
    En = (V_lj_mod(r12) + V_fene(r12) + V_lj_mod(r23) + V_fene(r23) + V_lj_mod(r13))
    w = W * r12 ** 2 * r23 ** 2 * np.exp(-(En - En.min()) / T)
    Z = w.sum()
    e1, e2 = (w * En).sum() / Z, (w * En ** 2).sum() / Z
    return e1, (e2 - e1 ** 2) / T ** 2, (w * r13).sum() / Z


def test_trimer_sampling_matches_3d_quadrature():
    """P11: N = 3 adds the angle-dependent non-bonded 1-3 LJ term and its cutoff."""
    T = np.array([0.3, 1.0])
    quoted = {0.3: (-2.270079, 2.503378, 0.847209), 1.0: (-1.220114, 0.996405, 1.060322)}
    E, n_sweeps, burn = 48, 24000, 2000
    o, tr = _run(3, T, 0.1 * np.sqrt(T), E, n_sweeps)
    en = tr["energy"][:, :, burn:]
    r13 = np.sqrt(tr["ree2"][:, :, burn:])
    for i, Ti in enumerate(T):
        e_ex, cv_ex, r_ex = _trimer_exact(Ti)
        assert (e_ex, cv_ex, r_ex) == pytest.approx(quoted[Ti], rel=3e-4)
        m, se = _mean_se(en[:, i].mean(-1))
        assert se < 0.02 and abs(m - e_ex) < 4.0 * se
        m, se = _mean_se(r13[:, i].mean(-1))
        assert se < 0.01 and abs(m - r_ex) < 4.0 * se
        m, se = _mean_se(en[:, i].var(-1) / Ti ** 2)
        assert abs(m - cv_ex) < 4.0 * se + 0.01 * cv_ex


# ------------------------------------------------------------------ P12: exchange step
def _dimer_conf(E, rs):
    conf = np.zeros((E, len(rs), 2, 3))
    for i, r in enumerate(rs):
        conf[:, i, 1, 0] = r
    return conf


@pytest.mark.parametrize("T,rs,expect", [
    ((0.5, 1.0), (0.70, 0.85), "exp"),     # colder replica has the lower energy: Delta < 0, p = exp(Delta)
    ((0.5, 1.0), (0.85, 0.70), "one"),     # colder replica has the higher energy: always swap (Eq. 6 sign)
    ((1.0, 1.0), (0.70, 0.85), "one"),     # equal temperatures: Delta = 0, always swap
])
def test_exchange_acceptance_frequency(T, rs, expect):
    E = 20000
    p = oracle.make_params(2, 2, E)
    o = oracle.Oracle(p, np.array(T), np.array([0.05, 0.05]), threads=1)
    conf = _dimer_conf(E, rs)
    o.init(np.arange(E, dtype=np.uint64) + np.uint64(991), conf)
    e0 = float(V_lj_mod(rs[0]) + V_fene(rs[0])); e1 = float(V_lj_mod(rs[1]) + V_fene(rs[1]))
    before = o.read()
    assert np.allclose(before["energies"], [[e0, e1]], rtol=1e-12)
    o.exchange()
    out = o.read()
    att, acc = out["swap_counts"][:, 0, 0], out["swap_counts"][:, 0, 1]
    assert (att == 1).all()
    delta = (1 / T[0] - 1 / T[1]) * (e0 - e1)
    p_ex = 1.0 if expect == "one" else float(np.exp(delta))
    frac = acc.mean()
    if expect == "one":
        assert frac == 1.0
    else:
        assert 0.05 < p_ex < 0.95 and abs(frac - p_ex) < 4.0 * np.sqrt(p_ex * (1 - p_ex) / E)
    # an accepted swap exchanges conformations and running energies; a rejected one changes nothing
    sw = acc == 1
    assert np.array_equal(out["conformations"][sw][:, 0], conf[sw][:, 1])
    assert np.array_equal(out["conformations"][sw][:, 1], conf[sw][:, 0])
    assert np.array_equal(out["conformations"][~sw], conf[~sw])
    assert np.array_equal(out["energies"][sw], before["energies"][sw][:, ::-1])
    assert np.array_equal(out["energies"][~sw], before["energies"][~sw])


def test_exchange_pair_schedule_alternates_parity():
    M, E = 5, 3
    T = synth.temperature_ladder(M, 0.5, 2.0)
    p = oracle.make_params(4, M, E)
    o = oracle.Oracle(p, T, synth.move_halfwidths(T), threads=1)
    o.init(np.arange(E, dtype=np.uint64), synth.random_walk_conformations(E, M, 4, 3))
    tr = o.enable_trace(0, 4, moves=False, energy=False)
    for _ in range(4):
        o.exchange()
    tried = tr["swap"] > 0
    assert np.array_equal(tried[:, 0], np.tile([True, False, True, False], (E, 1)))   # pairs (0,1),(2,3)
    assert np.array_equal(tried[:, 1], np.tile([False, True, False, True], (E, 1)))   # pairs (1,2),(3,4)
    assert np.array_equal(tried[:, 2], tried[:, 0]) and np.array_equal(tried[:, 3], tried[:, 1])
    sc = o.read()["swap_counts"]
    assert np.array_equal(sc[:, :, 0], np.full((E, M - 1), 2))
    assert np.array_equal(sc[:, :, 1], (tr["swap"] == 2).sum(1))


def _swap_rate_exact(T0, T1, n=400):
    """Closed-form double integral of min(1, exp[(b0-b1)(E0-E1)]) over the two dimer Boltzmann
    distributions."""
    g, wg = np.polynomial.legendre.leggauss(n)
    r = R0 + RFENE * g
    V = V_lj_mod(r) + V_fene(r)
    w0 = RFENE * wg * r * r * np.exp(-(V - V.min()) / T0)
    w1 = RFENE * wg * r * r * np.exp(-(V - V.min()) / T1)
    d = (1 / T0 - 1 / T1) * (V[:, None] - V[None, :])
    return float((w0[:, None] * w1[None, :] * np.minimum(1.0, np.exp(np.minimum(d, 0.0)))).sum() / (w0.sum() * w1.sum()))


def test_swap_rate_quadrature_matches_quoted_values():
    # SURVEY.md pin P12(ii)
    assert _swap_rate_exact(0.5, 1.0) == pytest.approx(0.77188742, abs=2e-4)
    assert _swap_rate_exact(0.3, 3.0) == pytest.approx(0.40100022, abs=2e-4)
    assert _swap_rate_exact(1.0, 1.1) == pytest.approx(0.97066666, abs=2e-4)


@pytest.mark.parametrize("T", [(0.5, 1.0), (0.3, 3.0)])
def test_two_replica_dimer_detailed_balance(T):
    """P12(ii): with exchanges on, each temperature still samples its own Boltzmann
    distribution and the measured swap acceptance equals the double integral."""
    T = np.array(T)
    E, n_sweeps, burn, every = 48, 20000, 2000, 5
    o, tr = _run(2, T, 0.1 * np.sqrt(T), E, n_sweeps, exchange_every=every)
    en = tr["energy"][:, :, burn:]
    for i, Ti in enumerate(T):
        _, e_ex, _ = _dimer_exact(Ti)
        m, se = _mean_se(en[:, i].mean(-1))
        assert se < 0.01 and abs(m - e_ex) < 4.0 * se
    sc = o.read()["swap_counts"][:, 0, :].astype(np.float64)
    assert (sc[:, 0] == n_sweeps // every // 2).all()        # pair (0,1) is tried on even events only
    m, se = _mean_se(sc[:, 1] / sc[:, 0])
    assert abs(m - _swap_rate_exact(*T)) < 4.0 * se + 2e-4


# ------------------------------------------------------------------ P9, P14, P15 on config 1
def _config1(threads=1, seeds=None, select_mode=0, widths=None, n_sweeps=None, trace=True, d_min=0.6):
    inp = synth.make_inputs(1)
    wl = inp.workload
    p = oracle.make_params(wl.N, wl.M, wl.E, select_mode=select_mode, nbins=wl.nbins,
                           hist_emin=wl.hist_range[0], hist_emax=wl.hist_range[1])
    o = oracle.Oracle(p, inp.temperatures, inp.widths if widths is None else widths, threads=threads)
    conf = inp.conformations if d_min > 0 else synth.random_walk_conformations(wl.E, wl.M, wl.N, 4242, d_min=0.0)
    o.init(inp.seeds if seeds is None else seeds, conf)
    n = wl.n_sweeps if n_sweeps is None else n_sweeps
    tr = o.enable_trace(n, n // wl.exchange_every) if trace else None
    o.run(n, wl.exchange_every)
    return o, tr, wl


def test_running_energy_equals_full_recompute_and_counters_are_consistent():
    o, tr, wl = _config1()
    out = o.read()
    for i in range(wl.M):
        full = oracle.total_energy(out["conformations"][0, i])
        assert abs(out["energies"][0, i] - full) <= 1e-9 * max(1.0, abs(full))          # P9
    mc = out["move_counts"][0]
    assert (mc[:, 0] == wl.N * wl.n_sweeps).all()
    assert np.array_equal(mc[:, 1], tr["move"][0].reshape(wl.M, -1).sum(-1))
    assert (mc[:, 1] + mc[:, 2] <= mc[:, 0]).all() and mc[-1, 2] > mc[0, 2]           # hot chains break bonds more
    assert (out["histograms"].sum(-1) == wl.n_sweeps).all()
    # the run ends with an exchange event, which only permutes the energies of the last sweep
    assert np.array_equal(np.sort(out["energies"][0]), np.sort(tr["energy"][0, :, -1]))
    # bonds never leave the FENE range
    b = np.linalg.norm(np.diff(out["conformations"][0], axis=1), axis=-1)
    assert (abs(b - R0) < RFENE).all()


def test_large_overlap_start_is_relaxed_and_rejects_infinite_moves():
    """Plain random walks with overlaps (initial energies >> 1): large positive Delta E is
    rejected, large negative accepted; the run ends with finite, negative energies."""
    o, tr, wl = _config1(d_min=0.0, n_sweeps=400)
    e = o.read()["energies"][0]
    assert np.isfinite(e).all() and (e < 10.0).all() and e[0] < -20.0
    inp = synth.make_inputs(1)
    e0 = [oracle.total_energy(c) for c in synth.random_walk_conformations(1, wl.M, wl.N, 4242, d_min=0.0)[0]]
    assert max(e0) > 1e4                                   # the start really had overlaps
    out = o.read()
    for i in range(wl.M):                                  # E_run keeps ~ulp(E_start) of cancellation error
        full = oracle.total_energy(out["conformations"][0, i])
        assert abs(out["energies"][0, i] - full) <= 1e-16 * 64 * max(e0) + 1e-9


def test_determinism_across_threads_and_seed_locality():
    o1, tr1, _ = _config1(threads=1, n_sweeps=300)
    o4, tr4, _ = _config1(threads=4, n_sweeps=300)
    a, b = o1.read(), o4.read()
    for k in a:
        assert np.array_equal(a[k], b[k]), k
    assert np.array_equal(tr1["move"], tr4["move"]) and np.array_equal(tr1["swap"], tr4["swap"])
    # two ensembles: changing the seed of ensemble 1 changes only ensemble 1
    inp = synth.make_inputs(1)
    wl = inp.workload
    conf = np.concatenate([inp.conformations, inp.conformations], axis=0)
    outs = []
    for s1 in (11, 12):
        p = oracle.make_params(wl.N, wl.M, 2)
        o = oracle.Oracle(p, inp.temperatures, inp.widths, threads=2)
        o.init(np.array([7, s1], dtype=np.uint64), conf)
        o.run(100, 10)
        outs.append(o.read())
    assert np.array_equal(outs[0]["conformations"][0], outs[1]["conformations"][0])
    assert not np.array_equal(outs[0]["conformations"][1], outs[1]["conformations"][1])


def test_limits_of_the_move_width():
    inp = synth.make_inputs(1)
    M = inp.workload.M
    o, _, wl = _config1(widths=np.full(M, 1e-7), n_sweeps=50, trace=False)       # width -> 0: acceptance -> 1
    mc = o.read()["move_counts"][0]
    assert (mc[:, 1] / mc[:, 0] > 0.99).all()
    o, _, wl = _config1(widths=np.full(M, 50.0), n_sweeps=50, trace=False)       # huge width: only bond-range rejections
    mc = o.read()["move_counts"][0]
    assert (mc[:, 1] == 0).all() and (mc[:, 2] == mc[:, 0]).all()
    o, _, wl = _config1(widths=synth.paper_halfwidths(M), n_sweeps=50, trace=False)   # the paper's +-0.01
    mc = o.read()["move_counts"][0]
    assert (mc[:, 1] / mc[:, 0] > 0.6).all()


def test_random_pick_mode_picks_all_monomers_uniformly():
    o, tr, wl = _config1(select_mode=1, n_sweeps=200)
    out = o.read()
    for i in range(wl.M):
        full = oracle.total_energy(out["conformations"][0, i])
        assert abs(out["energies"][0, i] - full) <= 1e-9 * max(1.0, abs(full))
    # the pick word: m = floor(w0 * N / 2^32) over tag-1 draws is uniform on 0..N-1
    seed = int(synth.seeds(1, 1)[0])
    key = [seed & 0xFFFFFFFF, seed >> 32]
    picks = [(oracle.philox([k, t, 0, (1 << 24) | 3], key)[0] * wl.N) >> 32 for t in range(300) for k in range(wl.N)]
    cnt = np.bincount(picks, minlength=wl.N)
    assert cnt.min() > 0 and max(picks) == wl.N - 1
    exp = len(picks) / wl.N
    assert ((cnt - exp) ** 2 / exp).sum() < 40.0            # chi^2, 12 dof


def test_observables_rgyr_and_ree():
    x = _line(4, 1.0)                                      # 0,1,2,3 on a line: mean 1.5, r_gyr^2 = 1.25, R_ee^2 = 9
    assert oracle.rgyr2(x) == pytest.approx(1.25, rel=1e-15)
    assert oracle.ree2(x) == pytest.approx(9.0, rel=1e-15)
    rng = np.random.default_rng(1)
    y = rng.normal(size=(20, 3))
    assert oracle.rgyr2(y) == pytest.approx(((y - y.mean(0)) ** 2).sum() / 20, rel=1e-13)


def test_create_rejects_bad_parameters():
    T, w = np.array([1.0]), np.array([0.1])
    for kw in (dict(N=1), dict(M=0), dict(E=0), dict(nbins=-1), dict(nbins=4, hist_emin=1.0, hist_emax=1.0)):
        args = dict(N=4, M=1, E=1); args.update(kw)
        with pytest.raises((ValueError, AssertionError)):
            oracle.Oracle(oracle.make_params(**args), T[: max(args["M"], 0)] if args["M"] != 1 else T,
                          w[: max(args["M"], 0)] if args["M"] != 1 else w)
    with pytest.raises(ValueError):
        oracle.Oracle(oracle.make_params(4), np.array([-1.0]), w)
    o = oracle.Oracle(oracle.make_params(3), T, w)
    with pytest.raises(ValueError):                         # a bond outside the FENE range: infinite energy
        o.init(np.array([1], dtype=np.uint64), _line(3, 1.2)[None, None])


# ------------------------------------------------------------------ measurement: bins, under/overflow, observables
def _frozen_dimers(rs, hist, nbins, n_sweeps=7):
    """Dimers at hand-set bond lengths, moved with a half-width of 1e-13: the energy stays where it
    was put (to ~1e-10), so what the measurement writes can be typed in by hand."""
    M = len(rs)
    p = oracle.make_params(2, M, 1, nbins=nbins, hist_emin=hist[0], hist_emax=hist[1])
    o = oracle.Oracle(p, np.full(M, 1.0), np.full(M, 1e-13), threads=1)
    o.init(np.array([5], dtype=np.uint64), _dimer_conf(1, rs))
    o.run(n_sweeps, 0)
    return o.read()


def test_histogram_bins_underflow_overflow_by_hand():
    """Reading R18: nbins interior bins over [emin, emax), bin = floor((E - emin) nbins /
    (emax - emin)), then one underflow and one overflow bin.  Energies by hand (closed_forms.txt):
    dimer at r0: -0.983683108864; at 0.85: LJ^mod(0.85) + 0.517827730413206; at 0.5: 41.65 + FENE."""
    e07 = -0.983683108864
    s6 = 0.117649 / (2.0 * 0.85 ** 6)
    e085 = 4.0 * (s6 * s6 - s6) + 0.016316891136 + 0.517827730413206      # = +0.00758...
    assert 0.007 < e085 < 0.008
    e05 = 41.6511572664319 - 1.8 * np.log(1.0 - (0.2 / 0.3) ** 2)         # = 42.709...
    n = 7
    # (a) range [-2, 0.2), 11 bins of width 0.2: E(r0) -> bin floor(1.0163 * 5) = 5; E(0.85) -> floor(2.0076 * 5) = 10;
    #     E(0.5) = 42.7 -> overflow (index nbins + 1)
    out = _frozen_dimers([0.7, 0.85, 0.5], (-2.0, 0.2), 11, n)
    h = out["histograms"][0]
    assert out["energies"][0] == pytest.approx([e07, e085, e05], abs=1e-9)
    exp = np.zeros((3, 13), dtype=np.uint64)
    exp[0, 5] = n; exp[1, 10] = n; exp[2, 12] = n
    assert np.array_equal(h, exp)
    # (b) range [-0.5, 0.5), 4 bins of width 0.25: E(r0) -> underflow (index nbins); E(0.85) = 0.0076 -> bin 2
    out = _frozen_dimers([0.7, 0.85], (-0.5, 0.5), 4, n)
    exp = np.zeros((2, 6), dtype=np.uint64)
    exp[0, 4] = n; exp[1, 2] = n
    assert np.array_equal(out["histograms"][0], exp)
    # (c) an energy that sits on a bin edge belongs to the upper bin (half-open bins): emin = E exactly
    out = _frozen_dimers([0.7], (out["energies"][0, 0], 1.0), 8, 1)
    assert out["histograms"][0, 0, 0] + out["histograms"][0, 0, 8] == 1      # bin 0, or underflow by one ulp of drift
    # moments: n, n E, n E^2
    out = _frozen_dimers([0.7, 0.85], (-2.0, 0.0), 10, n)
    assert out["moments"][0, :, 0].tolist() == [n, n]
    assert out["moments"][0, :, 1] == pytest.approx([n * e07, n * e085], rel=1e-9)
    assert out["moments"][0, :, 2] == pytest.approx([n * e07 ** 2, n * e085 ** 2], rel=1e-9)


def test_observable_sums_by_hand():
    """obs = sums over sweeps of R_ee^2, r_gyr^2, r_gyr^4, R_ee^4, E r_gyr^2 (Eq. 8).
    Dimer at distance r: R_ee^2 = r^2, r_gyr^2 = r^2/4.  Trimer on a line with spacing 0.7: R_ee^2 = 1.96,
    r_gyr^2 = 2 * 0.49 / 3."""
    n = 5
    out = _frozen_dimers([0.7, 0.85], (-2.0, 0.0), 10, n)
    for i, (r, e) in enumerate(((0.7, -0.983683108864), (0.85, out["energies"][0, 1]))):
        assert out["obs_moments"][0, i] == pytest.approx(
            [n * r * r, n * r * r / 4, n * (r * r / 4) ** 2, n * r ** 4, n * e * r * r / 4], rel=1e-9)
    p = oracle.make_params(3, 1, 1)
    o = oracle.Oracle(p, np.array([1.0]), np.array([1e-13]), threads=1)
    o.init(np.array([1], dtype=np.uint64), _line(3)[None, None])
    o.run(n, 0)
    ob = o.read()["obs_moments"][0, 0]
    rg2 = 2 * 0.49 / 3
    e3 = 2 * -0.983683108864 - 0.014688968239          # two pairs at r0, one at 2 r0 (closed_forms.txt)
    assert ob == pytest.approx([n * 1.96, n * rg2, n * rg2 ** 2, n * 1.96 ** 2, n * e3 * rg2], rel=1e-9)


def test_dimer_cross_moment_gives_the_thermal_derivative_of_rgyr():
    """d<r_gyr^2>/dT = beta^2 (<E r_gyr^2> - <E><r_gyr^2>) (the quantity of Fig. 5).
    For the dimer r_gyr^2 = r^2/4 and all three averages are 1-D integrals of r^2 exp(-V/T); the same
    number must also come out as the numerical T-derivative of <r^2/4>."""
    V = lambda r: float(V_lj_mod(r) + V_fene(r))

    def avgs(T):
        w = lambda r: r * r * np.exp(-(V(r) + 1.0) / T)
        Z = integrate.quad(w, 0.4, 1.0, epsabs=0, epsrel=1e-12, limit=400)[0]
        av = lambda f: integrate.quad(lambda r: f(r) * w(r), 0.4, 1.0, epsabs=0, epsrel=1e-12, limit=400)[0] / Z
        return av(V), av(lambda r: r * r / 4), av(lambda r: V(r) * r * r / 4)

    T = np.array([0.5, 1.5])
    E, n_sweeps, burn = 48, 20000, 2000
    o, tr = _run(2, T, 0.1 * np.sqrt(T), E, n_sweeps)
    out = o.read()
    # the accumulated cross moment is the sum over sweeps of E_t rg2_t
    assert np.allclose(out["obs_moments"][..., 4], (tr["energy"] * tr["rg2"]).sum(-1), rtol=1e-11)
    assert np.allclose(out["obs_moments"][..., 1], tr["rg2"].sum(-1), rtol=1e-12)
    for i, Ti in enumerate(T):
        e1, g1, eg = avgs(Ti)
        exact = (eg - e1 * g1) / Ti ** 2
        h = 1e-4
        assert exact == pytest.approx((avgs(Ti + h)[1] - avgs(Ti - h)[1]) / (2 * h), rel=1e-5)
        en, rg = tr["energy"][:, i, burn:], tr["rg2"][:, i, burn:]
        est = ((en * rg).mean(-1) - en.mean(-1) * rg.mean(-1)) / Ti ** 2
        m, se = _mean_se(est)
        assert se < 0.1 * abs(exact) and abs(m - exact) < 4.0 * se, (Ti, m, exact, se)


def test_running_energy_is_rebased_on_eq4_before_events_2k_minus_1():
    """Reading R22: the paper's kernel recomputes the energy by Eq. (4) after every sweep
    (PAPER.md:146); the oracle keeps E_run += Delta E and replaces it by the Eq.-4 sum before the exchange
    events x = 0, 1, 3, 7, ...  With M = 1 an event has no pair to try, so after such an event E_run IS
    orc_total_energy of the conformation, bit for bit; after the other events it is the accumulated value."""
    N = 13
    conf = synth.random_walk_conformations(1, 1, N, 4242, d_min=0.0)
    p = oracle.make_params(N, 1, 1)
    o = oracle.Oracle(p, np.array([1.0]), np.array([0.1]), threads=1)
    o.init(np.array([3], dtype=np.uint64), conf)
    exact, n_inexact = [], 0
    for x in range(9):
        o.sweeps(5)
        o.exchange()
        out = o.read()
        same = out["energies"][0, 0] == oracle.total_energy(out["conformations"][0, 0])
        if x in (0, 1, 3, 7):
            assert same, x
        else:
            n_inexact += not same
    assert n_inexact >= 3            # 5 sweeps of accepted moves leave last-bit differences


def test_overlap_start_meets_the_invariant_after_rebasing():
    """P9 with the survey's own start (plain walk, overlaps): |E_run - E_full| <= 1e-9 max(1, |E_full|) once an
    event 2^k - 1 has re-based the energies after the relaxation (here event 31, sweep 320 of 400)."""
    o, tr, wl = _config1(d_min=0.0, n_sweeps=400)
    out = o.read()
    for i in range(wl.M):
        full = oracle.total_energy(out["conformations"][0, i])
        assert abs(out["energies"][0, i] - full) <= 1e-9 * max(1.0, abs(full))
