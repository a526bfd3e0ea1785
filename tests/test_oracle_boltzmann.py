"""P8 / P9: the oracle's chain samples the Boltzmann distribution (no GPU).

Detailed balance holds for the sequential updating scheme, so the stationary law
is exp(-E) on the allowed configurations.  For two ions that law has a closed form; for three
ions it is obtained by brute-force simple sampling.  A wrong sign or prefactor of dE, an
asymmetric proposal, a leaky wall or overlap test, or a wrong acceptance rule all fail here.
Standard errors use the integrated autocorrelation time of PAPER.md:353-358 (Eq. 9-10).
"""
import math

import numpy as np
import pytest
from scipy import integrate

from oracle import Oracle


def integrated_autocorr_time(x, kmax=200):
    """T_c = 1/2 + sum_k C_k (Eq. 10), C_k as in Eq. 9, summed until C_k first drops below 0."""
    x = np.asarray(x, dtype=float) - np.mean(x)
    var = np.mean(x * x)
    T = 0.5
    for k in range(1, kmax):
        c = np.mean(x[:-k] * x[k:]) / var
        if c <= 0:
            break
        T += c
    return T


@pytest.mark.parametrize("z1,z2,seed", [(1.0, -1.0, 3), (1.0, 1.0, 4)])
def test_p8_two_ion_distance_law(z1, z2, seed):
    lB, d, R, delta = 1.68, 1.0, 2.5, 0.9
    a = R - 0.5 * d
    pos = np.array([[-0.8, 0.8], [0.0, 0.1], [0.0, -0.1]])
    o = Oracle(pos, np.array([z1, z2]), np.array([d, d]), R, lB, delta, seed)
    o.sweep(2000)                                         # equilibrate
    n, thin = 150000, 2
    r = np.empty(n)
    for k in range(n):
        o.sweep(thin)
        p = o.positions
        r[k] = math.dist(p[:, 0], p[:, 1])
    assert r.min() >= d and r.max() <= 2 * a
    assert np.all(np.einsum("ij,ij->j", o.positions, o.positions) <= a * a)

    # textbook pair-distance density of two uniform points in a ball of radius a, times Boltzmann
    def w(x):
        return math.exp(-lB * z1 * z2 / x) * x * x * (1 - 3 * x / (4 * a) + x ** 3 / (16 * a ** 3))

    edges = np.linspace(d, 2 * a, 25)
    mass = np.array([integrate.quad(w, lo, hi)[0] for lo, hi in zip(edges[:-1], edges[1:])])
    prob = mass / mass.sum()
    h, _ = np.histogram(r, bins=edges)
    Tc = integrated_autocorr_time(r)
    n_eff = n / (2 * Tc)
    chi2 = np.sum((h / n - prob) ** 2 / prob) * n_eff
    dof = len(prob) - 1
    assert 0.5 <= Tc < 20
    assert chi2 < dof + 5 * math.sqrt(2 * dof), (chi2, Tc)
    # per-bin 4 SE check, and the mean
    se = np.sqrt(prob * (1 - prob) / n_eff)
    assert np.all(np.abs(h / n - prob) < 4.5 * se)
    mean_ref = integrate.quad(lambda x: x * w(x), d, 2 * a)[0] / mass.sum()
    assert abs(r.mean() - mean_ref) < 4 * r.std() / math.sqrt(n_eff)
    # the test has teeth: the other sign of the interaction is far outside the tolerance
    wrong = np.array([integrate.quad(lambda x: w(x) * math.exp(2 * lB * z1 * z2 / x), lo, hi)[0]
                      for lo, hi in zip(edges[:-1], edges[1:])])
    wrong /= wrong.sum()
    assert np.sum((h / n - wrong) ** 2 / wrong) * n_eff > 20 * dof


def test_p9_three_ion_energy_law_by_simple_sampling():
    lB, R, delta = 1.68, 2.6, 0.8
    q = np.array([2.0, -1.0, -1.0])
    d = np.array([1.0, 0.8, 0.8])
    a = R - 0.5 * d

    def energies(p):                                      # p [M,3,3]: sample, ion, xyz
        out = np.zeros(len(p))
        ok = np.ones(len(p), dtype=bool)
        for i, j in ((0, 1), (0, 2), (1, 2)):
            rij = np.linalg.norm(p[:, i] - p[:, j], axis=1)
            out += lB * q[i] * q[j] / rij
            ok &= rij >= 0.5 * (d[i] + d[j])
        return out, ok

    # reference: independent uniform points in their balls, weighted by exp(-E) 1[no overlap]
    rng = np.random.default_rng(99)
    M = 3_000_000
    g = rng.normal(size=(M, 3, 3))
    g /= np.linalg.norm(g, axis=2, keepdims=True)
    p = g * (a[None, :, None] * rng.random((M, 3, 1)) ** (1 / 3))
    E, ok = energies(p)
    wgt = np.where(ok, np.exp(-E), 0.0)
    Z = wgt.sum()
    E_ref = (wgt * E).sum() / Z
    se_ref = math.sqrt(np.sum(wgt ** 2 * (E - E_ref) ** 2)) / Z
    edges = np.array([-np.inf, -6.0, -5.0, -4.0, -3.0, -2.0, -1.0, 0.0, np.inf])
    prob_ref = np.array([wgt[(E >= lo) & (E < hi)].sum() for lo, hi in zip(edges[:-1], edges[1:])]) / Z

    pos = np.array([[0.0, 1.2, -1.2], [0.0, 0.3, 0.2], [0.0, 0.0, 0.4]])
    o = Oracle(pos, q, d, R, lB, delta, 17)
    o.sweep(2000)
    n = 200000
    Ec = np.empty(n)
    for k in range(n):
        o.sweep(1)
        Ec[k] = o.stats()["E_running"]
    assert abs(Ec[-1] - o.energy()) < 1e-8                  # bookkeeping still exact (P5)
    Tc = integrated_autocorr_time(Ec)
    n_eff = n / (2 * Tc)
    se = math.sqrt(Ec.var() / n_eff + se_ref ** 2)
    assert abs(Ec.mean() - E_ref) < 4 * se, (Ec.mean(), E_ref, se, Tc)
    h, _ = np.histogram(Ec, bins=edges)
    se_b = np.sqrt(prob_ref * (1 - prob_ref) * (1 / n_eff + 30.0 / M))
    assert np.all(np.abs(h / n - prob_ref) < 4.5 * se_b + 1e-4), (h / n, prob_ref)
    # teeth: the energy scale is resolved far better than the bare-Coulomb scale of the problem
    assert se < 0.05 and E_ref < -1.5
