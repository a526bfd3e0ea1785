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


# ---------------------------------------------------------------------------------------------------
# Eq. 5-8, 13-18 on synthetic Yukawa tails with known kappa_R, q^R, eps_R
# ---------------------------------------------------------------------------------------------------
def _yukawa_system(linear: bool):
    """A 3:-1 electrolyte whose pair correlations are EXACTLY the dressed-ion far field (Eq. 7):
    beta U_ab = q_a^R q_b^R (l_B eps/eps_R) exp(-kappa_R r) / r, with kappa_R^2 = 4 pi l_B sum_c n_c q_c q_c^R
    (the relation that makes Eq. 12 reproduce Eq. 13; for a neutral binary mixture it is Eq. 8).
    linear: g = 1 - beta U (then every identity of the chain holds exactly); else g = exp(-beta U)."""
    lB, R = 0.949, 200.0
    z = np.array([3.0, -1.0])
    N = np.array([25000.0, 75000.0])
    V = 4 * np.pi * R ** 3 / 3
    n = N / V
    zR = np.array([4.125, -0.884])                      # the paper's fitted values, as inputs here
    eps_ratio = 1.07
    kR = np.sqrt(4 * np.pi * lB * np.sum(n * z * zR))
    bw, nb = 0.25, 400
    r = bw * (np.arange(nb) + 0.5)
    U = np.array([[zR[a] * zR[b] * (lB / eps_ratio) * np.exp(-kR * r) / r for b in range(2)] for a in range(2)])
    g = 1.0 - U if linear else np.exp(-U)
    return dict(lB=lB, R=R, z=z, N=N, n=n, zR=zR, eps_ratio=eps_ratio, kR=kR, r=r, U=U, g=g, bw=bw, nb=nb)


def test_bare_kappa_is_the_pb_formula():
    # 1:1, n_+ = n_- = n: kappa^2 = 8 pi l_B n (textbook Debye-Hueckel); config 1 of BASELINE: 1/kappa = 0.688 sigma
    R = (3 * 512 / 0.1 / (4 * np.pi)) ** (1 / 3)
    k = A.bare_kappa([256, 256], [1.0, -1.0], R, 1.68)
    assert abs(k - np.sqrt(8 * np.pi * 1.68 * 0.05)) < 1e-12
    assert abs(1 / k - 0.688) < 1e-3
    # charge-asymmetric: every species weighs in with q^2
    assert abs(A.bare_kappa([100, 300], [3.0, -1.0], 10.0, 1.0) ** 2
               - 4 * np.pi * (100 * 9 + 300 * 1) / (4 * np.pi * 1000 / 3)) < 1e-12


def test_tail_fit_recovers_kappa_R_exactly_on_a_yukawa_tail():
    s = _yukawa_system(linear=True)
    rho = A.charge_density(s["g"], s["N"], s["z"], s["R"])
    # Eq. 13 with its sign: negative around the cation, positive around the anion
    assert np.all(rho[0][20:120] < 0) and np.all(rho[1][20:120] > 0)
    # window 5..30 sigma: beyond it the tail (< 1e-5 of the uniform background) drowns in the rounding of 1 - beta U
    for b in range(2):
        f = A.fit_kappa_R(s["r"], rho[b], 5.0, 30.0)
        assert abs(f["kappa_R"] - s["kR"]) < 1e-8 * s["kR"]
        assert f["sign"] == (-1.0 if b == 0 else 1.0)
        # intercept of Eq. 14: log(kappa_R^2 |q^R| / (4 pi eps_R/eps))
        want = np.log(s["kR"] ** 2 * abs(s["zR"][b]) / (4 * np.pi * s["eps_ratio"]))
        assert abs(f["intercept"] - want) < 1e-7
    # a wrong slope is seen: a tail that decays with another kappa gives that kappa
    f = A.fit_kappa_R(s["r"], rho[0] * np.exp(-0.01 * s["r"]), 5.0, 30.0)
    assert abs(f["kappa_R"] - (s["kR"] + 0.01)) < 1e-8


def test_renormalized_valences_two_ways_permittivity_and_eq8_exact_on_linear_tails():
    s = _yukawa_system(linear=True)
    rho = A.charge_density(s["g"], s["N"], s["z"], s["R"])
    U = s["U"]                                          # for g = 1 - U the PMF of Eq. 11 is not U; feed U itself
    w = (5.0, 30.0)
    qp = [A.renormalized_valence(s["r"], U[a, 0], rho[a], s["kR"], s["lB"], *w) for a in range(2)]   # Eq. 17a, both ways
    qm = [A.renormalized_valence(s["r"], U[a, 1], rho[a], s["kR"], s["lB"], *w) for a in range(2)]   # Eq. 17b
    assert np.allclose(qp, s["zR"][0], rtol=1e-8) and np.allclose(qm, s["zR"][1], rtol=1e-8)
    e = [A.renormalized_permittivity(s["r"], rho[a], s["zR"][a], s["kR"], *w) for a in range(2)]     # Eq. 18, both ways
    assert np.allclose(e, s["eps_ratio"], rtol=1e-8)
    k0 = A.bare_kappa(s["N"], s["z"], s["R"], s["lB"])
    lhs, rhs = A.dressed_ion_identity(s["kR"], k0, s["zR"][0], s["zR"][1], s["z"][0], s["z"][1])
    assert abs(lhs - rhs) < 1e-12                       # Eq. 8 holds identically for this construction
    assert lhs > 1.0                                    # 4.125, -0.884 vs 3, -1: kappa_R > kappa, as the paper finds (25.57 < 28.53 A)


def test_whole_chain_from_histogram_counts_on_exponential_tails():
    """Counts -> g -> U, rho -> kappa_R, q^R, eps_R: with g = exp(-beta U) the far-field values come back to the
    accuracy of the linearisation (beta U ~ 1e-3 in the window)."""
    s = _yukawa_system(linear=False)
    shells = A.shell_volumes(s["bw"], s["nb"])
    ncent = np.array([4000.0, 12000.0]) * 50            # centres accumulated over 50 samples
    hist = np.array([[s["g"][a, b] * ncent[a] * s["n"][b] * shells for b in range(2)] for a in range(2)])
    out = A.renormalized_parameters(hist, ncent, s["N"], s["z"], s["R"], s["bw"], s["lB"], 12.0, 30.0)
    assert abs(out["kappa_R"] - s["kR"]) < 2e-3 * s["kR"]
    assert np.allclose(out["qR_plus"], s["zR"][0], rtol=5e-3) and np.allclose(out["qR_minus"], s["zR"][1], rtol=5e-3)
    assert np.allclose(out["epsR_over_eps"], s["eps_ratio"], rtol=1e-2)
    lhs, rhs = out["eq8"]
    assert abs(lhs - rhs) < 1e-2 * rhs
    assert abs(out["kappa"] - A.bare_kappa(s["N"], s["z"], s["R"], s["lB"])) == 0.0
