"""Pins of paper_1602_05716_b200/analysis.py against closed forms; CPU only."""
import numpy as np

from paper_1602_05716_b200 import analysis as A


def _uniform_ball(rng, n, R):
    x = rng.normal(size=(n, 3))
    x /= np.linalg.norm(x, axis=1)[:, None]
    return x * (R * rng.random(n) ** (1.0 / 3.0))[:, None]


def test_ideal_gas_has_g_equal_one_and_no_charge_density():
    """Uncorrelated points uniform in the cavity: g_ab(r) = 1 for every shell that lies inside the cavity
    (centres restricted to |x| <= R - r_max), U = 0, and the 1:1 charge density of Eq. 12 vanishes."""
    rng = np.random.default_rng(3)
    R, N, bw, nb = 10.0, 6000, 0.25, 12
    rmax = bw * nb
    hist = np.zeros((2, 2, nb))
    ncent = np.zeros(2)
    for _ in range(4):                                   # four independent "configurations"
        x = _uniform_ball(rng, N, R)
        sp = (np.arange(N) >= N // 2).astype(int)        # first half species 0 (+), second half species 1 (-)
        centres = np.nonzero(np.linalg.norm(x, axis=1) <= R - rmax)[0]
        for i in centres:
            r = np.linalg.norm(x - x[i], axis=1)
            r[i] = 1e9
            b = np.floor(r / bw).astype(int)
            ok = b < nb
            np.add.at(hist[sp[i]], (sp[ok], b[ok]), 1)
            ncent[sp[i]] += 1
    r_mid, g = A.pair_correlation(hist, ncent, [N // 2, N - N // 2], R, bw)
    assert r_mid[0] == 0.5 * bw and r_mid[-1] == (nb - 0.5) * bw
    tail = g[:, :, 3:]                                   # shells with enough counts
    assert np.all(np.abs(tail - 1.0) < 0.08), tail
    assert abs(g[:, :, 3:].mean() - 1.0) < 0.03
    U = A.potential_of_mean_force(g)
    assert np.all(np.abs(U[:, :, 3:]) < 0.09)
    rho = A.charge_density(g, [N // 2, N - N // 2], [+1.0, -1.0], R)
    n = (N / 2) / (4 * np.pi * R ** 3 / 3)
    assert np.all(np.abs(rho[:, 3:]) < 0.12 * n)


def test_pair_correlation_normalisation_on_a_hand_example():
    """One centre of species 0, three partners of species 1 in the second shell: g = 3 / (1 * n_1 * V_shell)."""
    hist = np.zeros((2, 2, 4)); hist[0, 1, 1] = 3
    R, bw = 5.0, 0.5
    _, g = A.pair_correlation(hist, [1, 0], [10, 20], R, bw)
    V = 4 * np.pi * R ** 3 / 3
    shell = 4 * np.pi / 3 * (1.0 ** 3 - 0.5 ** 3)
    assert np.isclose(g[0, 1, 1], 3 / (1 * (20 / V) * shell), rtol=1e-14)
    assert g[0, 1, 0] == 0 and np.all(np.isnan(g[1]))     # species 1 had no centres
    assert np.isinf(A.potential_of_mean_force(g)[0, 1, 0])
    assert np.allclose(A.shell_volumes(bw, 4).sum(), 4 * np.pi / 3 * 2.0 ** 3)


def test_autocorrelation_and_integrated_time_of_an_ar1_process():
    """x_{k+1} = phi x_k + noise has C_n = phi^n and T_c = 1/2 + phi / (1 - phi) (Eq. 9-10)."""
    rng = np.random.default_rng(11)
    phi, M = 0.6, 400000
    x = np.empty(M); x[0] = 0.0
    eps = rng.normal(size=M)
    for k in range(1, M):
        x[k] = phi * x[k - 1] + eps[k]
    C = A.autocorrelation(x + 5.0, 20)                   # the mean does not matter
    assert C[0] == 1.0
    assert np.all(np.abs(C[:8] - phi ** np.arange(8)) < 0.01)
    Tc = A.integrated_time(C, window=20)
    assert abs(Tc - (0.5 + phi / (1 - phi))) < 0.05
    assert abs(A.integrated_time(C) - Tc) < 0.1           # self-consistent cut agrees
    assert A.integrated_time(np.array([1.0, 0.0, 0.0])) == 0.5     # uncorrelated samples


def test_standard_error_of_a_correlated_series_matches_the_spread_of_independent_means():
    rng = np.random.default_rng(5)
    phi, M, reps = 0.7, 4000, 300
    means, ses = [], []
    for _ in range(reps):
        eps = rng.normal(size=M)
        x = np.empty(M); x[0] = eps[0]
        for k in range(1, M):
            x[k] = phi * x[k - 1] + eps[k]
        means.append(x.mean()); ses.append(A.standard_error(x))
    assert abs(np.mean(ses) / np.std(means) - 1.0) < 0.15
    assert A.standard_error(np.ones(50)) == 0.0
