"""Post-processing of the library's own outputs (Eq. 9-12).

Host-side arithmetic on small arrays (a few thousand numbers per run): the integer histograms of
``mc_pair_hist`` and the running energies of ``mc_get_stats``.  Nothing here is on the hot path and
nothing here touches the oracle.

* ``pair_correlation``       g_ab(r) from ordered-pair counts (normalisation of SURVEY.md 8(c), reading G17)
* ``potential_of_mean_force`` U_ab(r)/k_BT = -ln g_ab(r)                      (Eq. 11)
* ``charge_density``         rho^q_b(r) = n_+ q_+ g_{+b}(r) + n_- q_- g_{-b}(r)   (Eq. 12)
* ``autocorrelation``        C_n of a series of total energies                 (Eq. 9)
* ``integrated_time``        T_c = 1/2 + sum_k C_k                             (Eq. 10)
* ``standard_error``         sqrt(2 T_c var / M): the standard error the 3-SE checks use
"""
from __future__ import annotations

import numpy as np


def shell_volumes(bin_width: float, nbins: int) -> np.ndarray:
    """Volumes of the spherical shells [k w, (k+1) w): (4 pi / 3)(r_hi^3 - r_lo^3)."""
    edges = bin_width * np.arange(nbins + 1, dtype=np.float64)
    return (4.0 * np.pi / 3.0) * (edges[1:] ** 3 - edges[:-1] ** 3)


def pair_correlation(hist, n_centres, n_species, cavity_R: float, bin_width: float):
    """g_ab(r_k) = hist[a][b][k] / (n_centres[a] * (N_b / V) * shell volume k), V = 4 pi R^3 / 3.

    hist: [2][2][nbins] ordered-pair counts (centre species a, partner species b) accumulated over samples;
    n_centres: [2] centres accumulated over the same samples; n_species: [2] particles of each species.
    Returns (r_mid[nbins], g[2][2][nbins]); bins of a species pair without centres are NaN."""
    hist = np.asarray(hist, dtype=np.float64)
    n_centres = np.asarray(n_centres, dtype=np.float64)
    n_species = np.asarray(n_species, dtype=np.float64)
    nbins = hist.shape[-1]
    V = 4.0 * np.pi * cavity_R ** 3 / 3.0
    shells = shell_volumes(bin_width, nbins)
    g = np.full((2, 2, nbins), np.nan)
    for a in range(2):
        for b in range(2):
            if n_centres[a] > 0 and n_species[b] > 0:
                g[a, b] = hist[a, b] / (n_centres[a] * (n_species[b] / V) * shells)
    r_mid = bin_width * (np.arange(nbins) + 0.5)
    return r_mid, g


def potential_of_mean_force(g):
    """U_ab(r) / k_BT = -ln g_ab(r) (Eq. 11); +inf where g = 0 (inside the hard core)."""
    g = np.asarray(g, dtype=np.float64)
    with np.errstate(divide="ignore", invalid="ignore"):
        return -np.log(g)


def charge_density(g, n_species, valences, cavity_R: float):
    """rho^q_b(r) = n_+ q_+ g_{+b}(r) + n_- q_- g_{-b}(r) (Eq. 12), n = N / V, in units of e / sigma^3.

    Returns [2][nbins]: the mean charge density around a fixed ion of species b (the ion itself excluded)."""
    g = np.asarray(g, dtype=np.float64)
    V = 4.0 * np.pi * cavity_R ** 3 / 3.0
    n = np.asarray(n_species, dtype=np.float64) / V
    z = np.asarray(valences, dtype=np.float64)
    return np.stack([n[0] * z[0] * g[0, b] + n[1] * z[1] * g[1, b] for b in range(2)])


def autocorrelation(energies, max_lag: int) -> np.ndarray:
    """C_n, n = 0..max_lag (Eq. 9): time average over one series, mean and variance of the whole series."""
    e = np.asarray(energies, dtype=np.float64)
    M = e.size
    if M < 2 or max_lag >= M:
        raise ValueError("need more samples than lags")
    d = e - e.mean()
    var = np.mean(d * d)
    if var == 0.0:
        return np.concatenate([[1.0], np.zeros(max_lag)])
    return np.array([np.mean(d[: M - n] * d[n:]) / var for n in range(max_lag + 1)])


def integrated_time(C, window: int | None = None) -> float:
    """T_c = 1/2 + sum_{k>=1} C_k (Eq. 10).  The infinite sum is cut at ``window`` lags, or -- if not given --
    at the first non-positive C_k (the usual self-consistent cut: beyond it the estimate is noise)."""
    C = np.asarray(C, dtype=np.float64)
    if window is None:
        neg = np.nonzero(C[1:] <= 0.0)[0]
        window = int(neg[0]) if neg.size else C.size - 1
    return 0.5 + float(C[1: window + 1].sum())


def standard_error(series, max_lag: int | None = None) -> float:
    """Standard error of the mean of a correlated series: sqrt(2 T_c var / M)."""
    x = np.asarray(series, dtype=np.float64)
    M = x.size
    lag = min(M // 4, 200) if max_lag is None else max_lag
    Tc = max(0.5, integrated_time(autocorrelation(x, lag)))
    return float(np.sqrt(2.0 * Tc * x.var() / M))
