"""GPU tests of the SURVEY.md 8(f) rows: the paper-shaped workload (f3) and the analysis chain on the library's
own output (f1).  Need a B200 (``-m gpu``); inputs are seeded and synthetic, expected values come from oracle/."""
import os

import numpy as np
import pytest

from paper_1602_05716_b200 import analysis as A
from paper_1602_05716_b200 import workloads as W
from parity_util import compare_last_sweep, hard_constraints_ok, make_pair, record_margin

pytestmark = pytest.mark.gpu
NCPU = max(1, min(32, os.cpu_count() or 1))


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    torch.cuda.set_device(0)
    from paper_1602_05716_b200.binding import load_library
    load_library()


def test_paper_shaped_workload_n1048576_first_trials_and_invariants():
    """N = 2^20, 3:-1, R = 506 d, trial cube of edge L/3.  The oracle
    does the first 2100 trials of sweep 0 one by one (two chunks of the GPU schedule and a bit); the rest of the
    two sweeps by the invariants P5 / P6.  The geometry (R / d = 506, max_disp / d = 169) selects the canonical
    pair-distance form."""
    w = W.PAPER_SHAPED
    assert w.N == 1 << 20 and abs(w.cavity_R - 506.04) < 0.01 and abs(w.rho_star - 1.9318e-3) < 1e-6
    g, o = make_pair(w, threads=NCPU, validate=False)
    assert g.mc_get_option("form") == 2
    pos, q, d = w.arrays()
    g.mc_set_positions(pos)
    e0 = g.mc_energy()
    k = 2100
    g.mc_sweep(1)
    o.partial_sweep(0, k)
    emax, _ = compare_last_sweep(g, o, tag=w.name, first=0, count=k)
    assert np.array_equal(g.positions[:, :k], o.positions[:, :k])
    st = g.mc_get_stats()                                     # raises on MC_ESTALL (2 s watchdog, 1.8 ms per chunk)
    e1 = g.mc_energy()
    assert abs(st["E_running"] - e1) <= 1e-9 * max(1.0, abs(e1) + abs(e0))
    lg = g.mc_get_trial_log()
    acc = (lg["flags"] & 1) != 0
    assert abs(lg["dE"][acc].sum() - (st["E_running"] - e0)) <= 1e-9 * np.abs(lg["dE"][acc]).sum()
    g.mc_sweep(1)
    st = g.mc_get_stats()
    e2 = g.mc_energy()
    assert g.sweep_index == 2
    assert abs(st["E_running"] - e2) <= 1e-9 * max(1.0, abs(e2) + abs(e0))
    assert hard_constraints_ok(g.positions, d, w.cavity_R)
    ratio = st["accepted"] / (2 * w.N)
    record_margin(w.name, N=w.N, sweeps=2, max_dE_err=emax, form=2, R_over_dmin=w.cavity_R, acceptance=ratio,
                  E0=e0, E2=e2)
    assert 0.02 < ratio < 0.99
    assert e2 < e0                                            # relaxing from the uncorrelated start (~10 cycles)


def test_analysis_chain_on_the_library_output_against_independent_oracle_chains():
    """200 sweeps of config 2 on the GPU and on independent oracle chains (other seeds) ->
    mc_pair_hist after every sweep -> analysis.pair_correlation -> g_ab(r) agrees bin by bin within 3 standard
    errors.  The standard error comes from the scatter of FIVE oracle chains: 200 sweeps
    from a uniform start are not yet stationary (the density profile in the hard-wall cavity relaxes slowly), so
    a single chain's own fluctuations underestimate it -- two oracle chains differ from each other by far more than
    their blocked errors.  With 196 bins and a t-distribution with 4 degrees of freedom a few |z| > 3 are expected
    by chance; the bar is on their share, on the worst one and on the mean square."""
    w = W.CONFIGS[1]
    bw, nb = 0.1, 60
    rc = w.cavity_R - bw * nb - 0.5
    nsp = [s.count for s in w.species]
    skip = 40                                                  # the first, fastest part of the equilibration
    g, _ = make_pair(w, seed=11)
    gs, eg = [], []
    for s in range(w.sweeps):
        g.mc_sweep(1)
        hg, ng = g.mc_pair_hist(bw, nb, rc)
        r, g1 = A.pair_correlation(hg.cpu().numpy(), ng.cpu().numpy(), nsp, w.cavity_R, bw)
        gs.append(g1)
        eg.append(g.mc_get_stats()["E_running"])
    m1 = np.array(gs)[skip:].mean(axis=0)
    means = []
    for seed in (22, 23, 24, 25, 26):
        _, o = make_pair(w, seed=seed, threads=NCPU)
        acc = []
        for s in range(w.sweeps):
            o.sweep(1)
            ho, no = o.pair_hist(bw, nb, rc)
            acc.append(A.pair_correlation(ho, no, nsp, w.cavity_R, bw)[1])
        means.append(np.array(acc)[skip:].mean(axis=0))
    means = np.array(means)
    K = len(means)
    m2, sd = means.mean(axis=0), means.std(axis=0, ddof=1)
    use = r > 1.05                                             # beyond contact
    z = np.abs(m1 - m2)[:, :, use] / (sd[:, :, use] * np.sqrt(1.0 + 1.0 / K))
    record_margin("analysis_g_of_r_config2", zmax=float(z.max()), frac_above_3=float((z > 3).mean()),
                  mean_z2=float((z ** 2).mean()))
    assert (z > 3).mean() <= 0.10 and z.max() < 8.0 and (z ** 2).mean() < 3.0
    # the physics is there: contact peak of unlike ions, depletion of like ions, g -> 1 far out, U = -ln g
    k = np.argmax(use)
    assert m1[0, 1, k] > 1.5 and m1[0, 0, k] < 0.9
    assert abs(m1[:, :, -10:].mean() - 1.0) < 0.12
    U = A.potential_of_mean_force(m1)
    assert U[0, 1, k] < 0 < U[0, 0, k]
    rho = A.charge_density(m1, nsp, [s.valence for s in w.species], w.cavity_R)
    assert rho[0, k] < 0 < rho[1, k]                           # counter-charge around each ion (Eq. 12-13)
    # energy autocorrelation of the library's own E_running (Eq. 9-10)
    C = A.autocorrelation(np.array(eg)[skip:], 40)
    Tc = A.integrated_time(C)
    assert C[0] == 1.0 and 0.5 <= Tc < 80.0


@pytest.mark.parametrize("base,N", [(3, 5000), (2, 3000)])
def test_fp32_position_variant_matches_the_oracle_in_the_same_mode(base, N):
    """SURVEY.md 8(f) rank 4 (PAPER.md:83 float4 positions, PAPER.md:99 FP64 energy arithmetic): with
    position_bits = 32 on both sides the chain is again bit-identical to the oracle's, every position it holds is
    an FP32 value, and it differs from the FP64 chain."""
    from parity_util import assert_stats_equal, lockstep
    from paper_1602_05716_b200.binding import MCSystem
    w = W.scaled(W.CONFIGS[base], N)
    g, o = make_pair(w, threads=NCPU)
    g.mc_set_option("position_bits", 32)
    o.set_position_bits(32)
    assert g.mc_get_option("position_bits") == 32
    assert np.array_equal(g.positions, o.positions)
    r = lockstep(g, o, 8, tag="fp32 positions")
    record_margin(f"fp32_positions_{w.name}", N=w.N, sweeps=8, max_dE_err=r["max_dE_err"])
    assert_stats_equal(g, o, r["near_tie_flips"])
    p = g.positions
    assert np.array_equal(p, p.astype(np.float32).astype(np.float64))
    pos, q, d = w.arrays()
    ref = MCSystem(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, w.seed)
    ref.mc_sweep(8)
    assert not np.array_equal(ref.positions, p)
    assert hard_constraints_ok(p, d, w.cavity_R)


@pytest.mark.parametrize("base,N", [(2, 1500), (3, 2500)])
def test_parallel_reduction_comparison_kernel_runs_the_same_chain(base, N):
    """the paper's comparison code -- one kernel launch per trial,
    block reductions, atomic sub-totals, the last block decides -- gives the oracle's chain bit for bit, may be
    mixed with mc_sweep, and costs N launches per sweep."""
    from parity_util import assert_stats_equal
    w = W.scaled(W.CONFIGS[base], N)
    g, o = make_pair(w, threads=NCPU)

    class ViaReduction:
        """lockstep() drives mc_sweep; here every odd call goes through the comparison kernel instead."""
        def __init__(self, g):
            self.g, self.k = g, 0

        def mc_sweep(self, n):
            (self.g.mc_sweep_reduction if self.k % 2 == 0 else self.g.mc_sweep)(n)
            self.k += 1

        def __getattr__(self, name):
            return getattr(self.g, name)

        @property
        def positions(self):
            return self.g.positions

        @property
        def sweep_index(self):
            return self.g.sweep_index

        @sweep_index.setter
        def sweep_index(self, s):
            self.g.sweep_index = s

    from parity_util import lockstep
    l0 = g.mc_get_launch_count()
    r = lockstep(ViaReduction(g), o, 6, tag="parallel reduction")
    record_margin(f"parallel_reduction_{w.name}", N=w.N, sweeps=6, max_dE_err=r["max_dE_err"])
    assert_stats_equal(g, o, r["near_tie_flips"])
    assert g.sweep_index == 6
    assert g.mc_get_launch_count() - l0 >= 3 * w.N          # three of the six sweeps took N launches each
    assert abs(g.mc_get_stats()["E_running"] - g.mc_energy()) <= 1e-9 * abs(g.mc_energy())


def test_selfcheck_and_tune_scripts_run():
    """The two user-facing scripts of the package: the oracle-free invariants of a small run, and the option sweep
    behind the scheduling defaults (here on a tiny grid of settings)."""
    from paper_1602_05716_b200 import selfcheck, tune
    r = selfcheck.run(n=1200, sweeps=2)
    assert r["N"] == 1200 and r["accepted"] > 0
    t = tune.run(n=3000, workload=3, sweeps=2, top=3, full=False)
    assert t["N"] == 3000 and len(t["best"]) == 3
    assert t["best"][0]["us_per_sweep"] <= t["best"][-1]["us_per_sweep"]
    assert t["best"][0]["us_per_sweep"] < 3.0 * t["defaults_us_per_sweep"]
