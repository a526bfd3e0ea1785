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
* ``bare_kappa``             kappa of the Poisson-Boltzmann theory                              (Eq. 5)
* ``fit_kappa_R``            far-field straight-line fit of log(r |rho^q|) -> kappa_R           (Eq. 13-14)
* ``renormalized_valence``   q^R from beta U against rho^q / e, two ways each                   (Eq. 15-17)
* ``renormalized_permittivity`` eps_R / eps, two ways                                          (Eq. 18)
* ``dressed_ion_identity``   both sides of (kappa_R/kappa)^2 = (q_+^R - q_-^R)/(q_+ - q_-)     (Eq. 8)
* ``renormalized_parameters`` the whole chain on the accumulators of ``mc_pair_hist``
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


# ---------------------------------------------------------------------------------------------------
# The renormalised parameters from the tails of the pair correlations (Eq. 5-8, 13-18).
#
# Reduced units: lengths in sigma, energies in k_B T, charges in units of e.  Then beta e^2 / (4 pi eps) = l_B
# (the Bjerrum length), i.e. the solvent permittivity enters as eps = 1 / (4 pi l_B), and eps_R is reported
# as the ratio eps_R / eps.  Readings (also in DESIGN.md section 7):
#  * Eq. 13 is printed without the sign: rho^q = -eps laplace(phi) = -eps kappa_R^2 phi is NEGATIVE around a
#    positive ion (Eq. 16 carries the minus).  The straight-line fit of Eq. 14 therefore uses log(r |rho^q|).
#  * "fitting the long range data to straight-lines" (Fig. 14): q^R of Eq. 17 is the slope of beta U
#    against rho^q / e through the origin over the fit window, times -kappa_R^2 / (4 pi l_B).
# ---------------------------------------------------------------------------------------------------
def bare_kappa(n_species, valences, cavity_R: float, bjerrum: float) -> float:
    """Bare inverse Debye length (Eq. 5): kappa^2 = 4 pi l_B (n_+ q_+^2 + n_- q_-^2), n = N / V."""
    V = 4.0 * np.pi * cavity_R ** 3 / 3.0
    n = np.asarray(n_species, dtype=np.float64) / V
    z = np.asarray(valences, dtype=np.float64)
    return float(np.sqrt(4.0 * np.pi * bjerrum * np.sum(n * z * z)))


def _window(r, r_min, r_max, *arrays):
    r = np.asarray(r, dtype=np.float64)
    m = (r >= r_min) & (r <= r_max)
    for a in arrays:
        m &= np.isfinite(np.asarray(a, dtype=np.float64))
    return m


def fit_kappa_R(r, rho_q, r_min: float, r_max: float):
    """Far-field straight-line fit of log(r |rho^q(r)|) = A - kappa_R r (Eq. 14).

    rho_q: the charge density around one species (one row of ``charge_density``).  Bins where rho^q is zero or has
    the sign opposite to the window's majority are left out (noise around zero).  Returns a dict: kappa_R,
    intercept A, sign of rho^q in the window, number of bins used, and the standard error of the slope."""
    r = np.asarray(r, dtype=np.float64)
    rho = np.asarray(rho_q, dtype=np.float64)
    m = _window(r, r_min, r_max, rho) & (rho != 0.0)
    if m.sum() < 3:
        raise ValueError("fewer than 3 usable bins in the fit window")
    sign = 1.0 if np.sum(rho[m] > 0) >= np.sum(rho[m] < 0) else -1.0
    m &= (rho * sign) > 0
    if m.sum() < 3:
        raise ValueError("fewer than 3 bins of one sign in the fit window")
    x, y = r[m], np.log(r[m] * np.abs(rho[m]))
    xm, ym = x.mean(), y.mean()
    sxx = np.sum((x - xm) ** 2)
    slope = np.sum((x - xm) * (y - ym)) / sxx
    icpt = ym - slope * xm
    res = y - (icpt + slope * x)
    se = float(np.sqrt(np.sum(res ** 2) / max(1, x.size - 2) / sxx))
    return {"kappa_R": float(-slope), "intercept": float(icpt), "sign": sign, "bins": int(m.sum()), "stderr": se}


def renormalized_valence(r, U_ab, rho_a, kappa_R: float, bjerrum: float, r_min: float, r_max: float) -> float:
    """q_b^R = -eps kappa_R^2 U_ab(r) / rho_a^q(r) in the far field (Eq. 16-17), eps = 1/(4 pi l_B).

    U_ab: potential of mean force between a centre of species a and a partner of species b (Eq. 11);
    rho_a: charge density around species a (Eq. 12).  The ratio is taken as the least-squares slope of
    beta U against rho^q through the origin over [r_min, r_max] (Fig. 14).  Each q^R can be had two ways:
    (a, b) = (+, b) and (-, b)."""
    U = np.asarray(U_ab, dtype=np.float64)
    rho = np.asarray(rho_a, dtype=np.float64)
    m = _window(r, r_min, r_max, U, rho)
    if m.sum() < 1 or not np.any(rho[m] != 0.0):
        raise ValueError("no usable bins in the window")
    slope = np.sum(U[m] * rho[m]) / np.sum(rho[m] * rho[m])
    return float(-kappa_R ** 2 / (4.0 * np.pi * bjerrum) * slope)


def renormalized_permittivity(r, rho_a, qR_a: float, kappa_R: float, r_min: float, r_max: float) -> float:
    """eps_R / eps = -kappa_R^2 q_a^R exp(-kappa_R r) / (4 pi r rho_a^q(r)) in the far field (Eq. 18).

    Averaged over the window with weights rho^2 (least squares of rho against the Yukawa form).  Two ways: a = +, -."""
    r = np.asarray(r, dtype=np.float64)
    rho = np.asarray(rho_a, dtype=np.float64)
    m = _window(r, r_min, r_max, rho)
    y = -kappa_R ** 2 * qR_a * np.exp(-kappa_R * r[m]) / (4.0 * np.pi * r[m])      # = (eps_R / eps) * rho
    return float(np.sum(y * y) / np.sum(y * rho[m]))


def dressed_ion_identity(kappa_R: float, kappa: float, qR_plus: float, qR_minus: float, q_plus: float, q_minus: float):
    """Both sides of the exact relation (kappa_R / kappa)^2 = (q_+^R - q_-^R) / (q_+ - q_-) (Eq. 8)."""
    return (kappa_R / kappa) ** 2, (qR_plus - qR_minus) / (q_plus - q_minus)


def renormalized_parameters(hist, n_centres, n_species, valences, cavity_R, bin_width, bjerrum, r_min, r_max) -> dict:
    """The whole chain of PAPER.md:364-419 on the accumulators of ``mc_pair_hist``: g (G17) -> U (Eq. 11) and
    rho^q (Eq. 12) -> kappa_R from both species' tails (Eq. 14) -> q_+-^R two ways each (Eq. 17) -> eps_R / eps two
    ways (Eq. 18) -> the two sides of Eq. 8."""
    r, g = pair_correlation(hist, n_centres, n_species, cavity_R, bin_width)
    U = potential_of_mean_force(g)
    rho = charge_density(g, n_species, valences, cavity_R)
    fits = [fit_kappa_R(r, rho[b], r_min, r_max) for b in range(2)]
    kR = 0.5 * (fits[0]["kappa_R"] + fits[1]["kappa_R"])
    # U[a][b]: centre a, partner b; rho[a]: around species a
    qR = {"plus": (renormalized_valence(r, U[0, 0], rho[0], kR, bjerrum, r_min, r_max),
                   renormalized_valence(r, U[1, 0], rho[1], kR, bjerrum, r_min, r_max)),
          "minus": (renormalized_valence(r, U[0, 1], rho[0], kR, bjerrum, r_min, r_max),
                    renormalized_valence(r, U[1, 1], rho[1], kR, bjerrum, r_min, r_max))}
    qp, qm = 0.5 * sum(qR["plus"]), 0.5 * sum(qR["minus"])
    eps = (renormalized_permittivity(r, rho[0], qp, kR, r_min, r_max),
           renormalized_permittivity(r, rho[1], qm, kR, r_min, r_max))
    k0 = bare_kappa(n_species, valences, cavity_R, bjerrum)
    lhs, rhs = dressed_ion_identity(kR, k0, qp, qm, valences[0], valences[1])
    return {"r": r, "g": g, "U": U, "rho_q": rho, "kappa": k0, "kappa_R": kR, "kappa_R_fits": fits,
            "qR_plus": qR["plus"], "qR_minus": qR["minus"], "epsR_over_eps": eps, "eq8": (lhs, rhs)}
