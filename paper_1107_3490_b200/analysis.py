"""Host-side post-processing of what pt_read returns.

Nothing here is on the hot path: the device accumulates per-temperature moments and energy
histograms, and these few NumPy lines turn them into the paper's thermodynamic quantities:

  * <E>(T_i) and the specific heat C_V(T_i) = beta_i^2 (<E^2> - <E>^2), Eq. (7);
  * a continuous C_V(T) curve around each simulated temperature by single-histogram
    reweighting of the energy histogram at T_i (the "eyeball against Fig. 4" of SURVEY.md 8(f)).

k_B = 1 (R15).
"""
from __future__ import annotations

import numpy as np


def mean_energy(moments: np.ndarray) -> np.ndarray:
    """moments [..., 3] = (n_meas, sum E, sum E^2) -> <E>."""
    m = np.asarray(moments, dtype=np.float64)
    return m[..., 1] / m[..., 0]


def specific_heat(moments: np.ndarray, temperatures: np.ndarray) -> np.ndarray:
    """Eq. (7): C_V = (<E^2> - <E>^2) / T^2, per temperature (last-but-one axis of `moments`)."""
    m = np.asarray(moments, dtype=np.float64)
    e1 = m[..., 1] / m[..., 0]
    e2 = m[..., 2] / m[..., 0]
    return (e2 - e1 * e1) / np.asarray(temperatures, dtype=np.float64) ** 2


def bin_centres(nbins: int, emin: float, emax: float) -> np.ndarray:
    w = (emax - emin) / nbins
    return emin + w * (np.arange(nbins) + 0.5)


def reweight(hist: np.ndarray, centres: np.ndarray, T0: float, T: np.ndarray):
    """Single-histogram reweighting: from the interior bins of the histogram sampled at T0 to
    temperatures T (array).  Returns (<E>(T), C_V(T)).  P_T(E) ~ H(E) exp(-(1/T - 1/T0) E)."""
    h = np.asarray(hist, dtype=np.float64)
    e = np.asarray(centres, dtype=np.float64)
    T = np.atleast_1d(np.asarray(T, dtype=np.float64))
    keep = h > 0
    h, e = h[keep], e[keep]
    db = 1.0 / T[:, None] - 1.0 / T0
    logw = np.log(h)[None, :] - db * e[None, :]
    logw -= logw.max(axis=1, keepdims=True)
    w = np.exp(logw)
    z = w.sum(axis=1)
    e1 = (w * e).sum(axis=1) / z
    e2 = (w * e * e).sum(axis=1) / z
    return e1, (e2 - e1 * e1) / T ** 2


def mean_rgyr2(moments: np.ndarray, obs_moments: np.ndarray) -> np.ndarray:
    """<r_gyr^2> per temperature (Eq. 8) from obs_moments [..., 5]."""
    return np.asarray(obs_moments, dtype=np.float64)[..., 1] / np.asarray(moments, dtype=np.float64)[..., 0]


def d_rgyr2_dT(moments: np.ndarray, obs_moments: np.ndarray, temperatures: np.ndarray) -> np.ndarray:
    """The quantity of Fig. 5: d<r_gyr^2>/dT = (<E r_gyr^2> - <E><r_gyr^2>) / T^2,
    from the energy moments and the cross moment sum E r_gyr^2 the device accumulates."""
    m = np.asarray(moments, dtype=np.float64)
    o = np.asarray(obs_moments, dtype=np.float64)
    n = m[..., 0]
    return (o[..., 4] / n - (m[..., 1] / n) * (o[..., 1] / n)) / np.asarray(temperatures, dtype=np.float64) ** 2
