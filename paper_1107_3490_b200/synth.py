"""Seeded synthetic inputs shaped like the paper's workloads.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of
the method's arithmetic: no potentials, no Philox, no Metropolis rule.  It only
produces the arrays a caller hands to ``pt_create`` / ``pt_init``:

  * temperature ladders  T_i = T_min (T_max/T_min)^(i/(M-1))      (BASELINE.json configs)
  * move half-widths     d_i = 0.1 sqrt(T_i)                      (BASELINE.json configs)
  * Philox seeds         one 64-bit key per ensemble
  * initial conformations: random walks of bond length r0 from a NumPy PCG64 stream

The paper uses no public data set: its inputs are self-generated chains (PAPER.md:228,
:267), N = 13 and 55 for the physics, N = 55 with a varying number of replicas for the
timings.  The five BASELINE.json configurations stand in for those workloads.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

R0 = 0.7  # bond length of the initial random walk = position of both potential minima


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json configuration made concrete."""
    name: str
    N: int                 # monomers per chain
    M: int                 # replicas (temperatures) per ensemble
    E: int                 # independent ensembles
    T_min: float
    T_max: float
    exchange_every: int    # sweeps between exchange events
    n_sweeps: int
    nbins: int = 4096
    config_id: int = 0
    precisions: tuple = ("f64",)

    @property
    def chains(self) -> int:
        return self.E * self.M

    @property
    def moves(self) -> int:
        """attempted monomer moves of the whole job"""
        return self.chains * self.N * self.n_sweeps

    @property
    def pair_evals(self) -> int:
        """moves * 2(N-1): old and new position against every other monomer"""
        return self.moves * 2 * (self.N - 1)

    @property
    def hist_range(self) -> tuple:
        """energy-histogram range (inputs of the method; the paper has no histogram)"""
        return (-5.0 * self.N, 3.0 * self.N)


CONFIGS = {
    1: Workload("config1_N13_M8", 13, 8, 1, 0.3, 3.0, 10, 2000, config_id=1),
    2: Workload("config2_N30_M32", 30, 32, 1, 0.2, 3.0, 10, 10000, config_id=2),
    3: Workload("config3_N55_M64", 55, 64, 1, 0.15, 3.0, 20, 10000, config_id=3,
                precisions=("f64", "f32")),
    4: Workload("config4_N309_M128", 309, 128, 1, 0.2, 4.0, 20, 2000, config_id=4),
    5: Workload("config5_N100_M64_E64", 100, 64, 64, 0.2, 3.0, 10, 1000, config_id=5,
                precisions=("f64", "f32")),
}


def temperature_ladder(M: int, T_min: float, T_max: float) -> np.ndarray:
    """Geometric ladder, computed once in double; the same bits go to both sides."""
    if M == 1:
        return np.array([T_min], dtype=np.float64)
    i = np.arange(M, dtype=np.float64)
    return (T_min * (T_max / T_min) ** (i / (M - 1))).astype(np.float64)


def move_halfwidths(T: np.ndarray, scale: float = 0.1) -> np.ndarray:
    """BASELINE.json: uniform cube displacement of half-width 0.1*sqrt(T)."""
    return (scale * np.sqrt(np.asarray(T, dtype=np.float64))).astype(np.float64)


def paper_halfwidths(M: int) -> np.ndarray:
    """The paper's literal width: [-0.01, 0.01] at every temperature."""
    return np.full(M, 0.01, dtype=np.float64)


def seeds(config_id: int, E: int, rank: int = 0) -> np.ndarray:
    """One Philox key per ensemble: 0x1107349000000000 + (config << 32) + (rank << 16) + e."""
    base = 0x1107349000000000 + (int(config_id) << 32) + (int(rank) << 16)
    return np.array([base + e for e in range(E)], dtype=np.uint64)


def _unit_vectors(rng, n: int) -> np.ndarray:
    z = rng.uniform(-1.0, 1.0, size=n)
    phi = rng.uniform(0.0, 2.0 * np.pi, size=n)
    s = np.sqrt(1.0 - z * z)
    return np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=-1)


def random_walk_conformations(E: int, M: int, N: int, seed: int, r0: float = R0,
                              d_min: float = 0.6, tries: int = 64) -> np.ndarray:
    """[E][M][N][3] random walks: monomer 0 at the origin, every bond of length r0 in a
    direction uniform on the sphere.

    d_min > 0 (default): a growth step that would put the new monomer closer than d_min to
    an earlier non-bonded monomer is redrawn (up to `tries` times, then the best try is
    kept), so initial energies are O(N) and the running energy carries no cancellation
    error from relaxing huge overlap energies.
    d_min = 0: the plain walk, overlaps allowed (initial energies up to ~1e7 and beyond);
    used by the large-energy edge-case tests."""
    rng = np.random.Generator(np.random.PCG64(int(seed)))
    C = E * M
    x = np.zeros((C, N, 3), dtype=np.float64)
    for n in range(1, N):
        prev = x[:, n - 1, :]
        cand = prev + r0 * _unit_vectors(rng, C)
        if d_min > 0.0 and n >= 2:
            def min_dist(c, rows):
                d = x[rows, : n - 1, :] - c[:, None, :]
                return np.sqrt((d * d).sum(-1)).min(-1)
            best = cand.copy()
            best_d = min_dist(cand, np.arange(C))
            todo = np.nonzero(best_d < d_min)[0]
            for _ in range(tries):
                if todo.size == 0:
                    break
                c2 = prev[todo] + r0 * _unit_vectors(rng, todo.size)
                d2 = min_dist(c2, todo)
                better = d2 > best_d[todo]
                best[todo[better]] = c2[better]
                best_d[todo[better]] = d2[better]
                todo = todo[best_d[todo] < d_min]
            cand = best
        x[:, n, :] = cand
    return np.ascontiguousarray(x.reshape(E, M, N, 3))


@dataclass
class Inputs:
    workload: Workload
    temperatures: np.ndarray
    widths: np.ndarray
    seeds: np.ndarray
    conformations: np.ndarray
    meta: dict = field(default_factory=dict)


def make_inputs(config_id: int, rank: int = 0, E: int | None = None, M: int | None = None) -> Inputs:
    """All arrays for BASELINE config `config_id` (1-5).  `E`/`M` override the ensemble /
    replica count for sampled checks; the per-ensemble seeds and walks keep their values, so
    ensemble e of a sub-sample is bit-identical to ensemble e of the full workload."""
    wl = CONFIGS[config_id]
    Efull = wl.E
    T = temperature_ladder(wl.M, wl.T_min, wl.T_max)
    conf = random_walk_conformations(Efull, wl.M, wl.N, seed=1107349000 + 1000 * config_id + rank)
    sd = seeds(config_id, Efull, rank)
    if E is not None:
        conf, sd = conf[:E], sd[:E]
        wl = Workload(**{**wl.__dict__, "E": int(E)})
    return Inputs(wl, T, move_halfwidths(T), sd, np.ascontiguousarray(conf),
                  meta={"config_id": config_id, "rank": rank})


def shard_ensembles(E_total: int, world_size: int, rank: int) -> range:
    """Replicas-only multi-GPU: rank r simulates ensembles [lo, hi) of the job; no exchange
    of data between ranks is ever needed."""
    per = E_total // world_size
    extra = E_total % world_size
    lo = rank * per + min(rank, extra)
    hi = lo + per + (1 if rank < extra else 0)
    return range(lo, hi)
