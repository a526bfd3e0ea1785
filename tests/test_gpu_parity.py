"""Parity of the CUDA path (through the C ABI of include/mcb200.h) against the CPU oracle.

All tests here need a B200 (``-m gpu``).  Inputs are seeded and synthetic (workloads.py); no expected
value comes from the CUDA path.  Bars (BASELINE.json north_star): identical accept/reject bits and
positions, per-trial dE within 1e-10 relative, integer histograms bit-exact.
"""
import os

import numpy as np
import pytest

from paper_1602_05716_b200 import workloads as W
from parity_util import (assert_stats_equal, compare_last_sweep, hard_constraints_ok, lockstep, make_pair)

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
def test_config1_n512_100_sweeps_lockstep():
    w = W.CONFIGS[0]
    g, o = make_pair(w)
    r = lockstep(g, o, w.sweeps, tag=w.name)
    assert_stats_equal(g, o, r["near_tie_flips"])
    assert abs(g.mc_energy() - o.energy()) <= 1e-10 * abs(o.energy())
    st = g.mc_get_stats()
    assert 0.05 < st["accepted"] / (w.sweeps * w.N) < 0.99
    assert g.sweep_index == w.sweeps == o.sweep_index


def test_config2_n4096_lockstep_then_full_run():
    w = W.CONFIGS[1]
    g, o = make_pair(w, threads=NCPU)
    r = lockstep(g, o, 10, tag=w.name)
    # the remaining sweeps in one mc_sweep call; the chain is the same chain, so the final state matches
    rest = 30
    g.mc_sweep(rest)
    o.sweep(rest)
    e, f = compare_last_sweep(g, o, tag=f"{w.name} sweep {10 + rest - 1}")
    if f == 0 and r["near_tie_flips"] == 0:
        assert np.array_equal(g.positions, o.positions)
        assert_stats_equal(g, o)


def test_config3_n16383_two_diameters_ragged_tail():
    w = W.CONFIGS[2]                      # N = 16383 = 15 chunks of 1024 + 1023: ghost padding in the tail
    g, o = make_pair(w, threads=NCPU)
    r = lockstep(g, o, 3, tag=w.name)
    assert_stats_equal(g, o, r["near_tie_flips"])
    pos, q, d = w.arrays()
    assert hard_constraints_ok(g.positions, d, w.cavity_R)


def test_config4_n65536_headline_full_sweep_in_bench_configuration():
    """Full size, the launch configuration bench.py times (defaults: graph + overlap, chunk 1024):
    every trial of one sweep against the oracle, then invariants over more sweeps."""
    w = W.CONFIGS[3]
    g, o = make_pair(w, threads=NCPU, validate=False)
    e0 = g.mc_energy()
    g.mc_set_positions(w.arrays()[0])      # sets E_running = from-scratch energy
    g.mc_sweep(1)
    o.sweep(1)
    e, f = compare_last_sweep(g, o, tag=w.name)
    if f == 0:
        assert np.array_equal(g.positions, o.positions)
    # P5 at full size: E(init) + sum of accepted dE == from-scratch E(final)
    g.mc_sweep(4)
    st = g.mc_get_stats()
    e1 = g.mc_energy()
    assert abs(st["E_running"] - e1) <= 1e-9 * max(1.0, abs(e1) + abs(e0))
    assert st["accepted"] > 0 and g.sweep_index == 5
    pos, q, d = w.arrays()
    assert hard_constraints_ok(g.positions, d, w.cavity_R)


def test_config5_n262144_first_trials_and_invariants():
    """N = 262144: the oracle does the first 1100 trials of sweep 0 one by one (they need only the
    sweep-start state and each other: two chunks of the GPU schedule); the rest by invariants."""
    w = W.CONFIGS[4]
    g, o = make_pair(w, threads=NCPU, validate=False)
    pos, q, d = w.arrays()
    g.mc_set_positions(pos)
    e0 = g.mc_energy()
    k = 1100
    g.mc_sweep(1)
    o.partial_sweep(0, k)
    compare_last_sweep(g, o, tag=w.name, first=0, count=k)
    assert np.array_equal(g.positions[:, :k], o.positions[:, :k])
    st = g.mc_get_stats()
    e1 = g.mc_energy()
    assert abs(st["E_running"] - e1) <= 1e-9 * max(1.0, abs(e1) + abs(e0))
    assert hard_constraints_ok(g.positions, d, w.cavity_R)
    lg = g.mc_get_trial_log()
    acc = (lg["flags"] & 1) != 0
    assert abs(lg["dE"][acc].sum() - (st["E_running"] - e0)) <= 1e-9 * np.abs(lg["dE"][acc]).sum()


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


def test_dense_packing_many_overlap_vetoes():
    w = W.scaled(W.CONFIGS[3], 2500, max_disp=0.6)        # rho* = 0.4, big moves: many vetoes inside chunks
    g, o = make_pair(w)
    r = lockstep(g, o, 6, tag="dense")
    assert_stats_equal(g, o, r["near_tie_flips"])
    st = g.mc_get_stats()
    assert st["veto_overlap"] > 0.3 * 6 * w.N


def test_strong_coupling_low_acceptance():
    w = W.scaled(W.CONFIGS[0], 1500, bjerrum=12.0)
    g, o = make_pair(w)
    r = lockstep(g, o, 6, tag="lB=12")
    assert_stats_equal(g, o, r["near_tie_flips"])


# ---------------------------------------------------------------------------------------------------
# host logic of the library: options, re-entrancy, resume, validation
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("opts", [
    # persistent engine (the default): rows per thread / chunk size, item width, near workers, wave rounding
    {"prows": 1}, {"prows": 2}, {"prows": 4}, {"far_cols": 64}, {"far_cols": 1024}, {"pnear": 0}, {"pnear": 32},
    {"wave": 0}, {"prows": 2, "far_cols": 8, "pnear": 1}, {"debug": 1},
    # kernels-per-chunk engine
    {"engine": 0}, {"engine": 0, "chunk": 32}, {"engine": 0, "chunk": 96}, {"engine": 0, "chunk": 512},
    {"engine": 0, "graph": 0}, {"engine": 0, "overlap": 0}, {"engine": 0, "graph": 0, "chunk": 256}])
def test_every_launch_configuration_gives_the_same_chain(opts):
    w = W.scaled(W.CONFIGS[2], 2500)
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
        g.mc_set_option("pnear", (0, 4, 16)[rep])     # perturbs the schedule, not the items
        g.mc_sweep(6)
        lg = g.mc_get_trial_log()
        logs.append((g.positions.copy(), lg["dE"].copy(), lg["flags"].copy(), g.mc_get_stats()))
    for other in logs[1:]:
        assert np.array_equal(logs[0][0], other[0])
        assert np.array_equal(logs[0][1], other[1], equal_nan=True)
        assert np.array_equal(logs[0][2], other[2])
        assert logs[0][3] == other[3]


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
    # the range the FP64 veto band covers: cavity_R / d_min <= 2e4
    with pytest.raises(MCError) as e:
        MCSystem(ok, q, np.array([1.0, 1.0e-4]), 5.0, 1.68, 0.1, 1)
    assert e.value.code == MC_EINVAL


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
    w = W.scaled(W.CONFIGS[0], 64, rho_star=0.05, max_disp=1.5)
    g, _ = make_pair(w, seed=101)
    _, o = make_pair(w, seed=202)
    warm, n, every = 500, 6000, 3
    bw, nb, rc = 0.25, 12, 2.0
    g.mc_sweep(warm); o.sweep(warm)
    eg, eo = [], []
    hg = ng = None
    ho = no = None
    for _ in range(n // every):
        g.mc_sweep(every); o.sweep(every)
        eg.append(g.mc_get_stats()["E_running"]); eo.append(o.stats()["E_running"])
        hg, ng = g.mc_pair_hist(bw, nb, rc, hg, ng)
        ho, no = o.pair_hist(bw, nb, rc, ho, no)
    mg, sg = _blocked_mean_se(np.array(eg) / w.N)
    mo, so = _blocked_mean_se(np.array(eo) / w.N)
    assert abs(mg - mo) <= 3.0 * np.hypot(sg, so) + 1e-12, (mg, sg, mo, so)
    assert mg < -0.05                                          # the electrolyte is bound, not ideal
    # g_{+-} and g_{++} shapes: per-centre counts per bin, Poisson-ish errors inflated for correlation
    hg = hg.cpu().numpy().astype(np.float64); ng = ng.cpu().numpy().astype(np.float64)
    ho = ho.astype(np.float64); no = no.astype(np.float64)
    for a, b in ((0, 1), (0, 0)):
        cg, co = hg[a, b] / ng[a], ho[a, b] / no[a]
        se = 3.0 * np.sqrt(hg[a, b] + 1.0) / ng[a] + 3.0 * np.sqrt(ho[a, b] + 1.0) / no[a]
        assert np.all(np.abs(cg - co) <= 3.0 * se), (a, b, cg, co, se)
    assert hg[0, 1, 4:8].sum() / ng[0] > hg[0, 0, 4:8].sum() / ng[0]      # unlike ions closer than like ions
