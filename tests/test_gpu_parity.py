"""Parity of the CUDA path (through the C ABI of include/mcb200.h) against the CPU oracle.

All tests here need a B200 (``-m gpu``).  Inputs are seeded and synthetic (workloads.py); no expected
value comes from the CUDA path.  Bars (BASELINE.json north_star): identical accept/reject bits and
positions, per-trial dE within 1e-10 relative, integer histograms bit-exact.
"""
import os

import numpy as np
import pytest

from paper_1602_05716_b200 import workloads as W
from parity_util import (assert_stats_equal, compare_last_sweep, hard_constraints_ok, lockstep, make_pair,
                         record_margin)

pytestmark = pytest.mark.gpu

NCPU = max(1, min(32, os.cpu_count() or 1))


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    torch.cuda.set_device(0)
    from paper_1602_05716_b200.binding import load_library
    load_library()           # must be the in-tree libmcb200.so; raises if it is missing


# ---------------------------------------------------------------------------------------------------
# the five BASELINE configs
# ---------------------------------------------------------------------------------------------------
def _full_config_run(w, threads, hist_every_sweep=False):
    """All of the configuration's sweeps in lockstep with the oracle (north_star: identical accept/reject
    bits and positions over the run, per-trial dE within 1e-10); returns the lockstep summary."""
    g, o = make_pair(w, threads=threads, validate=w.N <= 20000)
    if w.N > 20000:
        g.mc_set_positions(w.arrays()[0])          # E_running := from-scratch energy (validate=False left it 0)
    e0 = g.mc_energy()
    hg = ng = ho = no = None

    def sample(done):
        nonlocal hg, ng, ho, no
        hg, ng = g.mc_pair_hist(w.hist_bin_width, w.hist_nbins, w.hist_centre_rmax, hg, ng)
        ho, no = o.pair_hist(w.hist_bin_width, w.hist_nbins, w.hist_centre_rmax, ho, no)
        # compared after every sweep, not only at the end: a wrong sample cannot hide in the sum
        assert np.array_equal(hg.cpu().numpy().astype(np.uint64), ho), f"{w.name}: g(r) counts differ after sweep {done - 1}"
        assert np.array_equal(ng.cpu().numpy().astype(np.uint64), no)

    r = lockstep(g, o, w.sweeps, tag=w.name, after_sweep=sample if hist_every_sweep else None)
    record_margin(w.name, N=w.N, sweeps=w.sweeps, max_dE_err=r["max_dE_err"], near_tie_flips=r["near_tie_flips"],
                  form=g.mc_get_option("form"), R_over_dmin=w.cavity_R / min(s.diameter for s in w.species),
                  oracle_threads=threads, oracle_seconds=r["oracle_seconds"],
                  oracle_pair_evals_per_s=w.sweeps * w.pair_evals_per_sweep / r["oracle_seconds"])
    assert r["max_dE_err"] <= 1e-10
    assert g.sweep_index == w.sweeps == o.sweep_index
    st = g.mc_get_stats()
    e1 = g.mc_energy()
    if w.N <= 20000:
        assert_stats_equal(g, o, r["near_tie_flips"])
    else:     # the oracle was not validated (its E_running started at 0): compare the increments
        so = o.stats()
        if r["near_tie_flips"] == 0:
            for k in ("accepted", "veto_overlap", "veto_wall", "near_ties"):
                assert st[k] == so[k], (k, st[k], so[k])
        assert abs((st["E_running"] - e0) - so["E_running"]) <= 1e-9 * max(1.0, abs(e1))
    # P5 on the GPU side: E(init) + sum of accepted dE == from-scratch E(final)
    assert abs(st["E_running"] - e1) <= 1e-9 * max(1.0, abs(e1) + abs(e0))
    assert 0.05 < st["accepted"] / (w.sweeps * w.N) < 0.99
    assert hard_constraints_ok(g.positions, w.arrays()[2], w.cavity_R)
    if hist_every_sweep:
        assert int(no.sum()) > 0.2 * w.N * w.sweeps      # the bulk centres the bench's call uses, not a thin shell
    return r


def test_config1_n512_all_100_sweeps_lockstep():
    _full_config_run(W.CONFIGS[0], threads=1)


def test_config2_n4096_all_200_sweeps_lockstep():
    _full_config_run(W.CONFIGS[1], threads=NCPU)


def test_config3_n16383_all_100_sweeps_lockstep_two_diameters_ragged_tail():
    # N = 16383 = 15 chunks of 1024 + 1023: ghost padding in the tail
    _full_config_run(W.CONFIGS[2], threads=NCPU)


def test_config4_n65536_headline_all_50_sweeps_lockstep_with_g_of_r_every_sweep():
    """The headline configuration in the launch configuration bench.py times (library defaults), all 50
    sweeps, with the bench's mc_pair_hist call (500 bins of 0.02 sigma, centre_rmax = w.hist_centre_rmax,
    about 21,000 centres) accumulated after every sweep on both sides and compared bit for bit."""
    _full_config_run(W.CONFIGS[3], threads=NCPU, hist_every_sweep=True)


def test_config5_n262144_one_full_oracle_sweep_then_invariants():
    """N = 262144: one full sweep against the oracle (every trial), then the configuration's 10 sweeps by
    invariants (the oracle is timed on one sweep only, BASELINE.json)."""
    w = W.CONFIGS[4]
    g, o = make_pair(w, threads=NCPU, validate=False)
    pos, q, d = w.arrays()
    g.mc_set_positions(pos)
    e0 = g.mc_energy()
    r = lockstep(g, o, 1, tag=w.name)
    record_margin(w.name, N=w.N, sweeps=1, max_dE_err=r["max_dE_err"], near_tie_flips=r["near_tie_flips"],
                  form=g.mc_get_option("form"), R_over_dmin=w.cavity_R / min(s.diameter for s in w.species),
                  oracle_threads=NCPU, oracle_seconds=r["oracle_seconds"],
                  oracle_pair_evals_per_s=w.pair_evals_per_sweep / r["oracle_seconds"])
    g.mc_sweep(w.sweeps - 1)
    st = g.mc_get_stats()
    e1 = g.mc_energy()
    assert g.sweep_index == w.sweeps
    assert abs(st["E_running"] - e1) <= 1e-9 * max(1.0, abs(e1) + abs(e0))
    assert hard_constraints_ok(g.positions, d, w.cavity_R)
    assert abs(np.sum(q)) == 0.0 and 0.05 < st["accepted"] / (w.sweeps * w.N) < 0.99


# ---------------------------------------------------------------------------------------------------
# tile / chunk boundaries and degenerate sizes
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N", [2, 3, 31, 32, 33, 63, 64, 65, 257, 1023, 1024, 1025, 2047, 2049, 3000])
def test_sizes_across_tile_and_chunk_boundaries(N):
    # exactly N ions (odd N is not neutral: the method does not need neutrality); two diameters if 3 | N
    w = W.Workload(f"n{N}", (W.Species(N - N // 2, +1.0, 1.0), W.Species(N // 2, -1.0, 0.8 if N % 3 == 0 else 1.0)),
                   0.2, 0.4, 12, seed=N)
    g, o = make_pair(w)
    assert g.N == o.N == N
    r = lockstep(g, o, 4 if N > 1500 else 12, tag=f"N={g.N}")
    assert_stats_equal(g, o, r["near_tie_flips"])


def test_single_ion():
    pos = np.array([[0.3], [0.1], [-0.2]])
    q, d = np.array([1.0]), np.array([1.0])
    from oracle import Oracle
    from paper_1602_05716_b200.binding import MCSystem
    g = MCSystem(pos, q, d, 1.2, 1.68, 0.5, 5)
    o = Oracle(pos, q, d, 1.2, 1.68, 0.5, 5)
    r = lockstep(g, o, 50, tag="N=1")
    assert_stats_equal(g, o, r["near_tie_flips"])
    assert g.mc_get_stats()["veto_wall"] > 0


@pytest.mark.parametrize("interleave", [False, True])
def test_species_order_is_the_callers(interleave):
    w = W.scaled(W.CONFIGS[2], 1200, interleave=interleave)      # reading G16
    g, o = make_pair(w)
    lockstep(g, o, 6, tag=f"interleave={interleave}")


@pytest.mark.parametrize("z,dcat,dan", [(3.0, 1.2, 1.0), (2.0, 1.0, 0.8)])
def test_multivalent_size_asymmetric(z, dcat, dan):
    n_cat = 300
    w = W.Workload("mv", (W.Species(n_cat, z, dcat), W.Species(int(z) * n_cat, -1.0, dan)), 0.3, 0.2, 5)
    g, o = make_pair(w)
    r = lockstep(g, o, 5, tag="multivalent")
    assert_stats_equal(g, o, r["near_tie_flips"])


# ---------------------------------------------------------------------------------------------------
# degenerate physics (P7)
# ---------------------------------------------------------------------------------------------------
def test_zero_displacement_accepts_everything_and_moves_nothing():
    w = W.scaled(W.CONFIGS[0], 300, max_disp=0.0)
    g, o = make_pair(w)
    p0 = g.positions
    lockstep(g, o, 3, tag="max_disp=0")
    assert np.array_equal(g.positions, p0)
    assert g.mc_get_stats()["accepted"] == 3 * w.N


def test_zero_bjerrum_is_pure_hard_spheres():
    w = W.scaled(W.CONFIGS[0], 700, bjerrum=0.0, rho_star=0.4)
    g, o = make_pair(w)
    lockstep(g, o, 5, tag="lB=0")
    fl = g.mc_get_trial_log()["flags"]
    assert np.array_equal((fl & 1) != 0, (fl & 6) == 0)      # accept <=> no veto
    assert (fl & 2).any()


def test_trial_landing_exactly_on_another_ion_is_vetoed_without_nan():
    # ion 1 sits where ion 0's first trial lands (the oracle's trial log gives that position)
    from oracle import Oracle
    from paper_1602_05716_b200.binding import MCSystem
    R, lB, delta, seed = 8.0, 1.68, 0.5, 11
    q, d = np.array([1.0, -1.0, 1.0]), np.array([0.1, 0.1, 0.1])
    pos = np.array([[0.0, 3.0, -3.0], [0.0, 0.0, 0.0], [0.0, 0.0, 0.0]])
    probe = Oracle(pos, q, d, R, lB, delta, seed)
    probe.partial_sweep(0, 1)
    pos[:, 1] = probe.trial_log()["trial"][:, 0]
    g = MCSystem(pos, q, d, R, lB, delta, seed)
    o = Oracle(pos, q, d, R, lB, delta, seed)
    g.mc_sweep(1)
    o.sweep(1)
    compare_last_sweep(g, o, tag="on-top")
    assert g.mc_get_trial_log()["flags"][0] & 2
    assert np.isfinite(g.mc_get_stats()["E_running"])
    lockstep(g, o, 20, tag="on-top continue")


def _on_top_case(N, i, j, offset, prows, seed0, dcat=0.25, dan=0.25):
    """A system in which ion j sits ``offset`` away from where ion i's trial of sweep 0 lands, with j's own
    move of that sweep rejected when j < i (so the trial really lands on it).  Returns (pos, q, d, seed, R, delta)."""
    from oracle import Oracle
    R, lB, delta = 14.0, 1.68, 0.5
    w = W.Workload("ontop", (W.Species(N - N // 2, +1.0, dcat), W.Species(N // 2, -1.0, dan)),
                   N / (4.0 * np.pi * R ** 3 / 3.0), delta, 1, seed=seed0)
    pos, q, d = w.arrays()
    for seed in range(seed0, seed0 + 40):
        probe = Oracle(pos, q, d, w.cavity_R, lB, delta, seed, validate=False)
        probe.partial_sweep(0, i + 1)                    # trial positions depend only on x_i and the seed
        t = probe.trial_log()["trial"][:, i].copy()
        p2 = pos.copy()
        p2[:, j] = t + np.asarray(offset)
        try:
            chk = Oracle(p2, q, d, w.cavity_R, lB, delta, seed)      # validates: no overlap in the start configuration
        except Exception:
            continue
        chk.partial_sweep(0, max(i, j) + 1)
        fl = chk.trial_log()["flags"]
        if j < i and (fl[j] & 1):
            continue                                     # j moved away before i's turn: try another seed
        assert fl[i] & 2, "the oracle must veto the trial that lands on another ion"
        return p2, q, d, seed, w.cavity_R, delta
    raise AssertionError("no seed gave the wanted on-top case")


@pytest.mark.parametrize("prows,N,i,j", [
    (1, 1100, 300, 700),     # partner in a later chunk: FAR-U (sweep-start position)
    (1, 1100, 1000, 40),     # partner three chunks back: FAR-L
    (1, 1100, 600, 70),      # two chunks back: MID
    (1, 1100, 600, 300),     # previous chunk: FIX
    (4, 4300, 1500, 3000),   # 1024-row chunks: FAR-U
    (4, 4300, 4200, 100),    # FAR-L
    (4, 4300, 2100, 1900),   # FIX
    (4, 4300, 3100, 1900),   # MID
])
@pytest.mark.parametrize("offset", [(0.0, 0.0, 0.0), (1e-7, 0.0, 0.0)])
@pytest.mark.parametrize("mixed", [False, True])
def test_trial_landing_on_an_ion_of_another_chunk_is_vetoed(prows, N, i, j, offset, mixed):
    """SURVEY P7 / PAPER.md:101 across chunks: the Gram-form r^2 of such a pair is 0 +- a few ulp(R^2) and may
    come out negative; the veto must still be an overlap and nothing non-finite may reach E_running."""
    from oracle import Oracle
    from paper_1602_05716_b200.binding import MCSystem
    pos, q, d, seed, R, delta = _on_top_case(N, i, j, offset, prows, seed0=3, dan=0.3 if mixed else 0.25)
    g = MCSystem(pos, q, d, R, 1.68, delta, seed)
    g.mc_set_option("prows", prows)
    assert g.mc_get_option("form") == 0
    g.mc_set_option("form", -1)
    o = Oracle(pos, q, d, R, 1.68, delta, seed)
    for form in (g.mc_get_option("form_auto"), 2):
        g.mc_set_state(pos, 0, o.energy())
        g.mc_set_option("form", form)
        o2 = Oracle(pos, q, d, R, 1.68, delta, seed)
        g.mc_sweep(1)
        o2.sweep(1)
        compare_last_sweep(g, o2, tag=f"on-top form {form}")
        assert g.mc_get_trial_log()["flags"][i] & 2
        assert np.array_equal(g.positions, o2.positions)
        assert np.isfinite(g.mc_get_stats()["E_running"])
    lockstep(g, o2, 3, tag="on-top continue")


def test_dense_packing_many_overlap_vetoes():
    w = W.scaled(W.CONFIGS[3], 2500, max_disp=0.6)        # rho* = 0.4, big moves: many vetoes inside chunks
    g, o = make_pair(w)
    r = lockstep(g, o, 6, tag="dense")
    assert_stats_equal(g, o, r["near_tie_flips"])
    st = g.mc_get_stats()
    assert st["veto_overlap"] > 0.3 * 6 * w.N


# ---------------------------------------------------------------------------------------------------
# dilute, large cavities: the pair-distance form follows the geometry
# ---------------------------------------------------------------------------------------------------
def _dilute(N, R, delta, sweeps, species=None, seed=7):
    sp = species or (W.Species(N // 4, +3.0, 1.0), W.Species(3 * (N // 4), -1.0, 1.0))
    n = sum(x.count for x in sp)
    return W.Workload(f"dilute_R{R:g}", sp, n / (4.0 * np.pi * R ** 3 / 3.0), delta, sweeps, seed=seed)


@pytest.mark.parametrize("R,delta,form", [
    (60.0, 0.5, 0),        # R / d_min = 60
    (128.0, 0.5, 0),       # the Gram form's limit
    (500.0, 0.5, 1),       # paper-like dilution, small moves: differences + displacement
    (500.0, 170.0, 2),     # paper-like dilution and trial cube ~ L/3: canonical form
    (2.0e4, 30.0, 1),      # the old admitted limit R / d_min = 2e4
    (9.0e5, 3.0e5, 2),     # close to the new limit R / d_min = 1e6
])
def test_large_cavity_parity_and_form_selection(R, delta, form):
    """dE within 1e-10 of max(|dE|, M_i) (G13) wherever mc_init admits the geometry; the automatic form is
    the documented one and a less exact one is refused."""
    from paper_1602_05716_b200.binding import MCError
    w = _dilute(4096, R, delta, 4)
    g, o = make_pair(w, threads=NCPU)
    assert g.mc_get_option("form_auto") == form == g.mc_get_option("form")
    if form > 0:
        with pytest.raises(MCError):
            g.mc_set_option("form", form - 1)
    r = lockstep(g, o, w.sweeps, tag=w.name)
    record_margin(w.name + f"_delta{delta:g}", N=w.N, sweeps=w.sweeps, max_dE_err=r["max_dE_err"], form=form,
                  R_over_dmin=R, near_tie_flips=r["near_tie_flips"])
    assert_stats_equal(g, o, r["near_tie_flips"])
    eg, eo = g.mc_energy(), o.energy()
    assert abs(eg - eo) <= 1e-10 * max(1.0, abs(eo)) * np.sqrt(w.N)
    g.mc_set_option("form", 2)                      # a more exact form is always allowed and gives the same chain
    lockstep(g, o, 2, tag=w.name + " canon")


def test_near_contact_pairs_stress_the_gram_form_at_its_limit():
    """R / d_min = 128 exactly, two diameters, small moves: the largest admitted (R / r)^2 for the
    |x_i|^2 + |x_j|^2 - 2 x_i.x_j form's absolute error, with the mixed-diameter veto key."""
    N = 50000
    sp = (W.Species(N // 2, +1.0, 0.25), W.Species(N // 2, -1.0, 0.125))
    V = 4.0 * np.pi * 16.0 ** 3 / 3.0
    w = W.Workload("gram_limit", sp, N / V, 0.05, 3, seed=5)
    g, o = make_pair(w, threads=NCPU, validate=False)
    assert g.mc_get_option("form_auto") == 0
    r = lockstep(g, o, w.sweeps, tag=w.name)
    assert g.mc_get_stats()["veto_overlap"] > 0.01 * w.sweeps * N
    record_margin(w.name, N=N, sweeps=w.sweeps, max_dE_err=r["max_dE_err"], form=0, R_over_dmin=128.0,
                  near_tie_flips=r["near_tie_flips"])
    assert_stats_equal(g, o, r["near_tie_flips"])


@pytest.mark.parametrize("R,N", [(128.0, 8192), (500.0, 8192), (500.0, 65536)])
def test_gram_form_error_beyond_its_admitted_range_is_measured(R, N):
    """Diagnostic (debug = 1 lets a LESS exact form be forced): the dE error of the Gram form where mc_init no
    longer selects it, so that the selection threshold rests on measured figures."""
    w = _dilute(N, R, 0.5, 2)
    g, o = make_pair(w, threads=NCPU, validate=N <= 10000)
    g.mc_set_option("debug", 1)
    g.mc_set_option("form", 0)
    worst = 0.0
    for s_ in range(w.sweeps):
        g.mc_sweep(1); o.sweep(1)
        lg, lo = g.mc_get_trial_log(), o.trial_log()
        same = (lg["flags"] & 7) == (lo["flags"] & 7)
        ok = ((lo["flags"] & 2) == 0) & same
        err = np.abs(lg["dE"][ok] - lo["dE"][ok]) / np.maximum(np.maximum(np.abs(lo["dE"][ok]), lo["scale"][ok]), 1e-300)
        worst = max(worst, float(err.max()))
        g.mc_set_state(o.positions, o.sweep_index, o.stats()["E_running"])       # stay on the oracle's chain whatever happened
    record_margin(f"gram_forced_R{R:g}_N{N}", N=w.N, max_dE_err=worst, form=0, R_over_dmin=R)
    assert worst < 1e-6                       # a measurement, not a bar: the figure goes to DESIGN.md


def test_geometry_limits_of_mc_init():
    from paper_1602_05716_b200.binding import MC_EINVAL, MCError, MCSystem
    q, ok = np.array([1.0, -1.0]), np.array([[0.0, 2.0], [0.0, 0.0], [0.0, 0.0]])
    with pytest.raises(MCError) as e:
        MCSystem(ok, q, np.array([1.0, 1.0]), 2.0e7, 1.68, 0.1, 1)          # cavity_R > 1e7
    assert e.value.code == MC_EINVAL
    with pytest.raises(MCError) as e:
        MCSystem(ok, q, np.array([1.0, 4.0e-6]), 5.0, 1.68, 0.1, 1)        # cavity_R / d_min > 1e6
    assert e.value.code == MC_EINVAL
    g = MCSystem(ok, q, np.array([1.0, 1.0e-4]), 5.0, 1.68, 0.1, 1)        # 5e4: fine now, canonical form
    assert g.mc_get_option("form_auto") == 2


def test_strong_coupling_low_acceptance():
    w = W.scaled(W.CONFIGS[0], 1500, bjerrum=12.0)
    g, o = make_pair(w)
    r = lockstep(g, o, 6, tag="lB=12")
    assert_stats_equal(g, o, r["near_tie_flips"])


# ---------------------------------------------------------------------------------------------------
# host logic of the library: options, re-entrancy, resume, validation
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("opts", [
    # rows per thread / chunk size, item width, near workers, wave rounding, pair-distance form, diameter path
    {"prows": 1}, {"prows": 2}, {"prows": 3}, {"prows": 4}, {"far_cols": 64}, {"far_cols": 1024}, {"pnear": 0}, {"pnear": 32},
    {"wave": 0}, {"prows": 2, "far_cols": 8, "pnear": 1}, {"debug": 1}, {"form": 1}, {"form": 2},
    {"form": 1, "prows": 1}, {"form": 2, "prows": 4}, {"uniform_path": 0, "form": 2},
    {"fix_cols": 4}, {"fix_cols": 8, "prows": 4}, {"fix_cols": 16}, {"diag_split": 1}, {"diag_split": 2}, {"diag_split": 8, "prows": 1}, {"max_ctas": 32}, {"max_ctas": 9, "diag_split": 4}])
@pytest.mark.parametrize("base", [2, 3])      # two diameters / equal diameters (the specialised path)
def test_every_launch_configuration_gives_the_same_chain(opts, base):
    w = W.scaled(W.CONFIGS[base], 2500)
    g, o = make_pair(w)
    for k, v in opts.items():
        g.mc_set_option(k, v)
    r = lockstep(g, o, 4, tag=str(opts))
    assert_stats_equal(g, o, r["near_tie_flips"])


@pytest.mark.parametrize("N,prows", [(700, 1), (5000, 2), (5000, 4), (20000, 4)])
def test_persistent_kernel_is_bit_reproducible(N, prows):
    """Which CTA runs which item, and in what order, differs from run to run; the fixed-point accumulation
    makes every sum -- and so the whole trial log -- independent of it."""
    from paper_1602_05716_b200.binding import MCSystem
    w = W.scaled(W.CONFIGS[3], N)
    pos, q, d = w.arrays()
    logs = []
    for rep in range(3):
        g = MCSystem(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 5)
        g.mc_set_option("prows", prows)
        g.mc_set_option("wave", 0)                    # item counts independent of the number of FAR workers
        g.mc_set_option("pnear", (0, 4, 16)[rep])     # perturbs the schedule, not the items
        g.mc_sweep(6)
        lg = g.mc_get_trial_log()
        logs.append((g.positions.copy(), lg["dE"].copy(), lg["flags"].copy(), g.mc_get_stats()))
    for other in logs[1:]:
        assert np.array_equal(logs[0][0], other[0])
        assert np.array_equal(logs[0][1], other[1], equal_nan=True)
        assert np.array_equal(logs[0][2], other[2])
        assert logs[0][3] == other[3]


@pytest.mark.parametrize("N,pnear", [(700, 0), (700, 4), (5000, 4), (5000, 16), (20000, 0), (20000, 4)])
def test_soak_completion_counters_after_every_sweep(N, pnear):
    """The flag/counter protocol of the sweep kernel: after every sweep
    each chunk's three completion counters must equal the number of items the host-side plan gives for it --
    a lost or doubled increment ("the lost increments") would show here long before
    it stalls a chain.  2000+ sweeps in all over the sizes and near-worker settings."""
    from paper_1602_05716_b200.binding import MCSystem
    w = W.scaled(W.CONFIGS[3], N)
    pos, q, d = w.arrays()
    g = MCSystem(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 77)
    g.mc_set_option("pnear", pnear)
    rows = g.mc_get_option("prows")
    C_, Np = 256 * rows, (N + 31) // 32 * 32
    nchunks = (Np + C_ - 1) // C_
    HDR = 256
    sweeps = {700: 600, 5000: 300, 20000: 120}[N]
    want = None
    for s_ in range(sweeps):
        g.mc_sweep(1)
        g.synchronize()
        W_ = HDR + 4 * (Np // 256 + 1)                       # live words, then the snapshot of the completed sweep
        peek = np.array(g.mc_debug_peek(2 * W_))
        assert not peek[:W_].any(), "the live scheduling words must be zero between sweeps"
        sy = peek[W_:]
        far, diag, fix = (sy[HDR + k * nchunks: HDR + (k + 1) * nchunks] for k in range(3))
        if want is None:
            # the plan: diag items = ceil(nt^2 / 8); urgent = C/32 (c >= 2) + C/16 (c >= 1); far from the first sweep,
            # cross-checked against the total mc_plan_check reports
            nt = [min(C_, Np - c * C_) // 32 for c in range(nchunks)]
            split = 4 if Np <= 768 else 2 if Np <= 6144 else 1   # warps per DIAG unit, by N
            want_diag = np.array([(t * t * split + 7) // 8 for t in nt])
            fixc = 16 if Np >= 53248 else 8 if Np >= 36864 else 4   # columns per FIX item, by N
            want_fix = np.array([(C_ // 32 if c >= 2 else 0) + (C_ // fixc if c >= 1 else 0) for c in range(nchunks)])
            assert np.array_equal(diag, want_diag) and np.array_equal(fix, want_fix)
            want = (far.copy(), want_diag, want_fix)
            assert far.sum() + want_diag.sum() + want_fix.sum() > 0
        assert np.array_equal(far, want[0]), f"sweep {s_}: FAR completion counters {far} != {want[0]}"
        assert np.array_equal(diag, want[1]), f"sweep {s_}: DIAG completion counters"
        assert np.array_equal(fix, want[2]), f"sweep {s_}: urgent completion counters"
        assert sy[160] == 0                                  # abort flag
    st = g.mc_get_stats()                                    # raises on MC_ESTALL
    assert g.sweep_index == sweeps
    e = g.mc_energy()
    assert abs(st["E_running"] - e) < 1e-8 * max(1.0, abs(e))
    assert hard_constraints_ok(g.positions, d, w.cavity_R)


def test_far_item_count_matches_the_host_plan():
    """The FAR completion counts the soak test takes from the first sweep are the plan's: total items per sweep
    = mc_plan_check's count for the same (N, rows, far_cols, far workers)."""
    from paper_1602_05716_b200.binding import MCSystem, mc_plan_check
    import torch
    for N in (700, 5000, 20000):
        w = W.scaled(W.CONFIGS[3], N)
        pos, q, d = w.arrays()
        g = MCSystem(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 1)
        g.mc_set_option("diag_split", 1)                 # the host plan counts one warp per in-chunk unit
        g.mc_set_option("fix_cols", 16)                  # ... and 16 columns per FIX item
        g.mc_sweep(1)
        g.synchronize()
        rows = g.mc_get_option("prows")
        C_, Np = 256 * rows, (N + 31) // 32 * 32
        nchunks = (Np + C_ - 1) // C_
        W_ = 256 + 4 * (Np // 256 + 1)
        sy = np.array(g.mc_debug_peek(2 * W_))[W_:]
        nsm = torch.cuda.get_device_properties(0).multi_processor_count
        plan = mc_plan_check(N, rows, g.mc_get_option("far_cols"), max(1, 2 * nsm - 2 - g.mc_get_option("pnear")))
        assert plan["violations"] == 0
        assert int(sy[256:256 + 3 * nchunks].sum()) == plan["items"]


def test_stalled_sweep_is_reported_by_every_synchronising_call_and_recoverable():
    """A sweep whose deciding warp never runs ("probe" = 2) must end through the watchdog, not hang; afterwards
    every synchronising call says MC_ESTALL, later sweeps are no-ops, and loading a configuration recovers."""
    from paper_1602_05716_b200.binding import MC_EINVAL, MC_ESTALL, MCError, MCSystem
    w = W.scaled(W.CONFIGS[0], 1500)
    pos, q, d = w.arrays()
    g = MCSystem(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 4)
    with pytest.raises(MCError) as e:
        g.mc_set_option("probe", 2)                     # refused without debug
    assert e.value.code == MC_EINVAL
    g.mc_sweep(2)
    good = g.positions.copy()
    st_good = g.mc_get_stats()
    g.mc_set_option("debug", 1)
    g.mc_set_option("stall_ms", 50)
    g.mc_set_option("probe", 2)
    g.mc_sweep(1)
    for call in (g.mc_get_stats, g.mc_energy, lambda: g.sweep_index, g.mc_sweep_timed):
        with pytest.raises(MCError) as e:
            call()
        assert e.value.code == MC_ESTALL
    g.mc_set_option("probe", 0)
    g.mc_set_option("debug", 0)
    g.mc_set_option("stall_ms", 2000)
    g.mc_sweep(3)                                       # no-ops: the state is invalid
    with pytest.raises(MCError):
        g.mc_get_stats()
    # recovery: load the last good state and go on; the chain continues as an undisturbed one does
    g.mc_set_state(good, 2, st_good["E_running"])
    assert g.sweep_index == 2
    g.mc_sweep(3)
    ref = MCSystem(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 4)
    ref.mc_sweep(5)
    assert np.array_equal(g.positions, ref.positions)
    assert abs(g.mc_get_stats()["E_running"] - ref.mc_get_stats()["E_running"]) < 1e-9


def test_many_sweeps_never_stall():
    """200 sweeps of a mid-size system: the watchdog (MC_ESTALL) must stay silent and the invariants hold."""
    w = W.scaled(W.CONFIGS[1], 6000)
    g, o = make_pair(w)
    g.mc_sweep(200)
    st = g.mc_get_stats()                      # raises on MC_ESTALL
    assert hard_constraints_ok(g.positions, w.arrays()[2], w.cavity_R)
    e = g.mc_energy()
    assert abs(st["E_running"] - e) < 1e-8 * max(1.0, abs(e))


def test_reentrancy_and_resume():
    from paper_1602_05716_b200.binding import MCSystem
    w = W.scaled(W.CONFIGS[0], 1100)
    pos, q, d = w.arrays()
    a = MCSystem(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 9)
    b = MCSystem(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 9)
    a.mc_sweep(7)
    b.mc_sweep(3); b.mc_sweep(4)
    assert np.array_equal(a.positions, b.positions)
    assert a.mc_get_stats() == b.mc_get_stats()
    # checkpoint / resume: positions + sweep index are the whole state
    c = MCSystem(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 9)
    c.mc_set_positions(a.positions)
    c.sweep_index = a.sweep_index
    a.mc_sweep(2); c.mc_sweep(2)
    assert np.array_equal(a.positions, c.positions)
    la, lc = a.mc_get_trial_log(), c.mc_get_trial_log()
    assert np.array_equal(la["flags"], lc["flags"]) and np.array_equal(la["dE"], lc["dE"])
    # another seed is another chain
    e = MCSystem(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 10)
    e.mc_sweep(1)
    b2 = MCSystem(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 9)
    b2.mc_sweep(1)
    assert not np.array_equal(e.positions, b2.positions)


def test_sweep_host_roundtrip_matches_device_path():
    import torch
    from paper_1602_05716_b200.binding import MCSystem
    w = W.scaled(W.CONFIGS[0], 900)
    pos, q, d = w.arrays()
    a = MCSystem(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 3)
    b = MCSystem(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 3)
    a.mc_sweep(3)
    pin = torch.from_numpy(pos).pin_memory()
    pout = torch.empty((3, w.N), dtype=torch.float64).pin_memory()
    _, st = b.mc_sweep_host(3, pin, pout)
    assert np.array_equal(pout.numpy(), a.positions)
    assert st == a.mc_get_stats()
    # feeding back the downloaded positions with their running energy continues the chain without a recompute
    a.mc_sweep(2)
    _, st2 = b.mc_sweep_host(2, pout, pout, E_running_in=st["E_running"])
    assert np.array_equal(pout.numpy(), a.positions)
    assert st2 == a.mc_get_stats()


def test_init_validation_errors():
    from paper_1602_05716_b200.binding import MC_EINVAL, MC_EOUTSIDE, MC_EOVERLAP, MCError, MCSystem
    q, d = np.array([1.0, -1.0]), np.array([1.0, 1.0])
    ok = np.array([[0.0, 2.0], [0.0, 0.0], [0.0, 0.0]])
    MCSystem(ok, q, d, 5.0, 1.68, 0.1, 1)
    with pytest.raises(MCError) as e:
        MCSystem(np.array([[0.0, 0.9], [0.0, 0.0], [0.0, 0.0]]), q, d, 5.0, 1.68, 0.1, 1)
    assert e.value.code == MC_EOVERLAP
    with pytest.raises(MCError) as e:
        MCSystem(np.array([[0.0, 4.6], [0.0, 0.0], [0.0, 0.0]]), q, d, 5.0, 1.68, 0.1, 1)
    assert e.value.code == MC_EOUTSIDE
    for bad in (dict(R=-1.0), dict(lB=-0.1), dict(delta=-1.0), dict(R=float("nan"))):
        with pytest.raises(MCError) as e:
            MCSystem(ok, q, d, bad.get("R", 5.0), bad.get("lB", 1.68), bad.get("delta", 0.1), 1)
        assert e.value.code == MC_EINVAL
    with pytest.raises(MCError) as e:
        MCSystem(ok, q, np.array([1.0, 0.0]), 5.0, 1.68, 0.1, 1)
    assert e.value.code == MC_EINVAL
    with pytest.raises(MCError) as e:
        MCSystem(np.array([[0.0, np.inf], [0.0, 0.0], [0.0, 0.0]]), q, d, 5.0, 1.68, 0.1, 1)
    assert e.value.code == MC_EINVAL
    # contact is allowed (G6, G7): touching the wall and each other
    MCSystem(np.array([[-0.5, 0.5], [0.0, 0.0], [0.0, 0.0]]), q, d, 1.0, 1.68, 0.1, 1)


def test_workspace_too_small_and_bad_arguments_through_the_raw_abi():
    import ctypes as C
    import torch
    from paper_1602_05716_b200 import binding as B
    lib = B.load_library()
    assert lib.mc_workspace_bytes(0) == 0 and lib.mc_workspace_bytes(-5) == 0
    n = 64
    need = lib.mc_workspace_bytes(n)
    assert need > 0
    ws = torch.empty(need + 256, dtype=torch.uint8, device="cuda")
    base = (ws.data_ptr() + 255) // 256 * 256
    w = W.scaled(W.CONFIGS[0], n)
    pos, q, d = (torch.from_numpy(a).cuda() for a in w.arrays())
    h = C.c_void_p()
    args = (n, pos.data_ptr(), q.data_ptr(), d.data_ptr(), w.cavity_R, 1.68, 0.1, 1)
    assert lib.mc_init(C.byref(h), *args, base, need - 1, None, 1) == B.MC_ENOSPACE
    assert b"workspace" in lib.mc_last_error()
    assert lib.mc_init(C.byref(h), *args, base + 8, need, None, 1) == B.MC_EINVAL
    assert lib.mc_init(C.byref(h), 0, *args[1:], base, need, None, 1) == B.MC_EINVAL
    assert lib.mc_init(C.byref(h), *args, base, need, None, 1) == B.MC_OK
    assert lib.mc_sweep(h, -1) == B.MC_EINVAL
    assert lib.mc_sweep(h, 0) == B.MC_OK
    assert lib.mc_energy(h, None) == B.MC_EINVAL
    assert lib.mc_set_option(h, b"nonsense", 1) == B.MC_EINVAL
    assert lib.mc_set_option(h, b"chunk", 48) == B.MC_EINVAL
    assert lib.mc_pair_hist(h, 0.0, 10, 1.0, base, base) == B.MC_EINVAL
    assert lib.mc_free(h) == B.MC_OK
    assert lib.mc_free(None) == B.MC_OK


# ---------------------------------------------------------------------------------------------------
# a5 / a6
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N", [2, 33, 700, 5000])
def test_energy_matches_the_oracle(N):
    w = W.scaled(W.CONFIGS[2], N)
    g, o = make_pair(w)
    eg, eo = g.mc_energy(), o.energy()
    # relative to the sum of magnitudes the pair sum cancels from (same idea as reading G13)
    assert abs(eg - eo) <= 1e-11 * max(abs(eo), 1.0) * max(1.0, np.sqrt(N))
    assert abs(g.mc_get_stats()["E_running"] - eo) <= 1e-11 * max(abs(eo), 1.0) * max(1.0, np.sqrt(N))


def test_two_ion_closed_form_on_the_gpu():
    from paper_1602_05716_b200.binding import MCSystem
    pos = np.array([[0.0, 1.5], [0.0, 2.0], [0.0, 0.0]])
    g = MCSystem(pos, np.array([2.0, -3.0]), np.array([1.0, 1.0]), 6.0, 1.68, 0.1, 1)
    assert abs(g.mc_energy() - (-6.0 * 1.68 / 2.5)) < 1e-14


@pytest.mark.parametrize("N,bw,nb", [(3000, 0.02, 500), (3000, 0.1, 37), (500, 0.5, 3), (16383, 0.02, 500)])
def test_pair_hist_bit_exact(N, bw, nb):
    base = W.CONFIGS[2]
    w = base if N == base.N else W.scaled(base, N)
    g, o = make_pair(w, validate=N < 10000)
    g.mc_sweep(2)
    o.set_threads(NCPU)
    o.sweep(2)
    assert np.array_equal(g.positions, o.positions)
    rc = max(0.5, w.cavity_R - bw * nb - 0.5)
    hg, ng = g.mc_pair_hist(bw, nb, rc)
    ho, no = o.pair_hist(bw, nb, rc)
    assert np.array_equal(hg.cpu().numpy().astype(np.uint64), ho)
    assert np.array_equal(ng.cpu().numpy().astype(np.uint64), no)
    assert ho.sum() > 0
    hg, ng = g.mc_pair_hist(bw, nb, rc, hg, ng)               # accumulates
    assert np.array_equal(hg.cpu().numpy().astype(np.uint64), 2 * ho)
    assert np.array_equal(ng.cpu().numpy().astype(np.uint64), 2 * no)


def test_pair_hist_headline_shape_sampled_centres():
    """Config 4's histogram call (500 bins of 0.02 sigma, bulk centres) at full N: the oracle does a
    thin shell of centres (centre_rmax small) one by one; counts must match bit for bit."""
    w = W.CONFIGS[3]
    g, o = make_pair(w, validate=False)
    hg, ng = g.mc_pair_hist(w.hist_bin_width, w.hist_nbins, 6.0)
    ho, no = o.pair_hist(w.hist_bin_width, w.hist_nbins, 6.0)
    assert no.sum() > 100
    assert np.array_equal(hg.cpu().numpy().astype(np.uint64), ho)
    assert np.array_equal(ng.cpu().numpy().astype(np.uint64), no)


# ---------------------------------------------------------------------------------------------------
# statistics: independent seeds, long runs (makes the 3-SE clause of north_star non-vacuous)
# ---------------------------------------------------------------------------------------------------
def _blocked_mean_se(x, nblocks=20):
    x = np.asarray(x, dtype=np.float64)
    m = len(x) // nblocks
    b = x[: m * nblocks].reshape(nblocks, m).mean(axis=1)
    return b.mean(), b.std(ddof=1) / np.sqrt(nblocks)


def test_long_run_mean_energy_and_g_of_r_agree_with_independent_oracle_chain():
    """north_star: long-run mean energy per ion and g_{+-}(r), g_{++}(r) within 3 standard errors.  GPU and
    oracle run DIFFERENT seeds, so nothing but the sampled distribution is shared.  Standard errors by
    blocking (20 blocks, each many autocorrelation times long) -- per quantity and per bin."""
    w = W.scaled(W.CONFIGS[0], 64, rho_star=0.05, max_disp=1.5)
    g, _ = make_pair(w, seed=101)
    _, o = make_pair(w, seed=202)
    warm, n, every = 500, 8000, 4
    bw, nb, rc = 0.5, 6, 2.0
    g.mc_sweep(warm); o.sweep(warm)
    eg, eo, cg, co = [], [], [], []
    import torch
    for _ in range(n // every):
        g.mc_sweep(every); o.sweep(every)
        eg.append(g.mc_get_stats()["E_running"]); eo.append(o.stats()["E_running"])
        hg, ng = g.mc_pair_hist(bw, nb, rc)                   # one sample each: fresh accumulators
        ho, no = o.pair_hist(bw, nb, rc)
        hg = hg.cpu().numpy().astype(np.float64); ng = np.maximum(ng.cpu().numpy().astype(np.float64), 1.0)
        cg.append(np.stack([hg[0, 1] / ng[0], hg[0, 0] / ng[0]]))      # partners per + centre and bin: +-, ++
        co.append(np.stack([ho[0, 1] / max(no[0], 1), ho[0, 0] / max(no[0], 1)]).astype(np.float64))
    mg, sg = _blocked_mean_se(np.array(eg) / w.N)
    mo, so = _blocked_mean_se(np.array(eo) / w.N)
    assert abs(mg - mo) <= 3.0 * np.hypot(sg, so), (mg, sg, mo, so)
    assert mg < -0.05                                          # the electrolyte is bound, not ideal
    cg, co = np.array(cg), np.array(co)                        # [samples][2][nb]
    zmax = 0.0
    for a in range(2):
        for b in range(2, nb):                                 # bins beyond contact (r >= 1 sigma)
            m1, s1 = _blocked_mean_se(cg[:, a, b])
            m2, s2 = _blocked_mean_se(co[:, a, b])
            assert m1 > 0 and m2 > 0
            z = abs(m1 - m2) / np.hypot(s1, s2)
            zmax = max(zmax, z)
            assert z <= 3.0, (a, b, m1, s1, m2, s2)
    # the check has teeth: the same statistic separates +- from ++ (different distributions) by far more than 3 SE
    m1, s1 = _blocked_mean_se(cg[:, 0, 2]); m2, s2 = _blocked_mean_se(cg[:, 1, 2])
    assert (m1 - m2) / np.hypot(s1, s2) > 6.0                  # unlike ions sit closer than like ions
    record_margin("long_run_statistics", energy_z=abs(mg - mo) / np.hypot(sg, so), g_of_r_zmax=zmax)


def test_more_sweeps_than_one_launch_holds():
    """mc_sweep(n) runs at most 1024 sweeps per launch: n = 1030 is two launches and must equal 1000 + 30."""
    from paper_1602_05716_b200.binding import MCSystem
    w = W.scaled(W.CONFIGS[0], 300)
    pos, q, d = w.arrays()
    a = MCSystem(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 9)
    b = MCSystem(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 9)
    a.mc_sweep(1030)
    b.mc_sweep(1000); b.mc_sweep(30)
    assert a.sweep_index == b.sweep_index == 1030
    assert np.array_equal(a.positions, b.positions)
    assert a.mc_get_stats() == b.mc_get_stats()
    e = a.mc_energy()
    assert abs(a.mc_get_stats()["E_running"] - e) < 1e-8 * max(1.0, abs(e))
    assert hard_constraints_ok(a.positions, d, w.cavity_R)
