"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

P1 Philox known answers        P2 uniform mapping          P3 two-ion closed form
P4 brute force on tiny N       P5 energy bookkeeping       P6 hard constraints
P7 degenerate cases            P10 re-entrancy             + library-routine cross-checks
(P8/P9, the Boltzmann-law pins, are in test_oracle_boltzmann.py.)
Numbering follows SURVEY.md section 8(c).
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest
from scipy.spatial.distance import pdist

from oracle import Oracle, philox4x32_10, uniform_open01
from oracle.binding import OracleError
from paper_1602_05716_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")
M32 = 0xFFFFFFFF


# ---- an independent transcription of the round description, used only to widen P1 ----------------
def py_philox(ctr, key):
    c = list(ctr)
    k0, k1 = key
    for r in range(10):
        if r:
            k0 = (k0 + 0x9E3779B9) & M32
            k1 = (k1 + 0xBB67AE85) & M32
        p0 = 0xD2511F53 * c[0]
        p1 = 0xCD9E8D57 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k0, p1 & M32, (p0 >> 32) ^ c[3] ^ k1, p0 & M32]
    return tuple(c)


def py_uniform(lo, hi):
    k = ((hi << 32) | lo) >> 12
    return Fraction(2 * k + 1, 2 ** 53)


def py_trial(seed, sweep, i, x, max_disp):
    """Exact-rational restatement of the trial move: round((u - 1/2) * D + x) once per axis."""
    key = (seed & M32, seed >> 32)
    A = py_philox((i, sweep & M32, sweep >> 32, 0), key)
    B = py_philox((i, sweep & M32, sweep >> 32, 1), key)
    us = [py_uniform(A[0], A[1]), py_uniform(A[2], A[3]), py_uniform(B[0], B[1])]
    D = Fraction(2.0 * max_disp)
    t = [float((u - Fraction(1, 2)) * D + Fraction(float(xc))) for u, xc in zip(us, x)]
    return t, float(py_uniform(B[2], B[3]))


def energy_exact(pos, q, lB):
    """l_B sum_{i<j} q_i q_j / r_ij with math.fsum (plain definition, independent of the oracle)."""
    N = pos.shape[1]
    terms = []
    for i in range(N):
        for j in range(i + 1, N):
            r = math.sqrt(math.fsum((pos[k, i] - pos[k, j]) ** 2 for k in range(3)))
            terms.append(q[i] * q[j] / r)
    return lB * math.fsum(terms)


# ---- P1 -----------------------------------------------------------------------------------------
def test_p1_philox_known_answers():
    n = 0
    for line in open(os.path.join(GOLD, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(t, 16) for t in line.split()]
        assert philox4x32_10(w[0:4], w[4:6]) == tuple(w[6:10])
        assert py_philox(w[0:4], w[4:6]) == tuple(w[6:10])
        n += 1
    assert n == 3


def test_p1_philox_matches_independent_transcription_on_random_counters():
    rng = np.random.default_rng(5)
    for _ in range(200):
        ctr = [int(v) for v in rng.integers(0, 2 ** 32, 4)]
        key = [int(v) for v in rng.integers(0, 2 ** 32, 2)]
        assert philox4x32_10(ctr, key) == py_philox(ctr, key)


# ---- P2 -----------------------------------------------------------------------------------------
def test_p2_uniform_edges_and_exactness():
    assert uniform_open01(0, 0) == 2.0 ** -53
    assert uniform_open01(M32, M32) == 1.0 - 2.0 ** -53
    assert uniform_open01(0, 0x80000000) == 0.5 + 2.0 ** -53
    assert uniform_open01(0xFFF, 0) == 2.0 ** -53            # low 12 bits are dropped
    assert uniform_open01(0x1000, 0) == 3 * 2.0 ** -53
    rng = np.random.default_rng(11)
    for _ in range(500):
        lo, hi = (int(v) for v in rng.integers(0, 2 ** 32, 2))
        u = uniform_open01(lo, hi)
        assert 0.0 < u < 1.0
        assert Fraction(u) == py_uniform(lo, hi)                      # exactly representable
        assert Fraction(u - 0.5) == py_uniform(lo, hi) - Fraction(1, 2)  # and so is u - 1/2
        # symmetric about 1/2: complementing the word maps u -> 1 - u
        assert uniform_open01(lo ^ M32, hi ^ M32) == 1.0 - u


def test_p2_uniform_statistics():
    n = 200000
    u = np.empty(n)
    k = 0
    i = 0
    while k < n:
        o = philox4x32_10((i, 0, 0, 0), (123, 456))
        u[k] = uniform_open01(o[0], o[1]); u[k + 1] = uniform_open01(o[2], o[3])
        k += 2; i += 1
    assert abs(u.mean() - 0.5) < 4 * math.sqrt(1 / 12 / n)
    assert abs(u.var() - 1 / 12) < 4 * math.sqrt(1 / 180 / n)
    h, _ = np.histogram(u, bins=64, range=(0, 1))
    chi2 = ((h - n / 64) ** 2 / (n / 64)).sum()
    assert chi2 < 63 + 5 * math.sqrt(2 * 63)


# ---- trial positions: exact-rational restatement ----------------------------------------------
def test_trial_positions_are_correctly_rounded_fma():
    w = W.scaled(W.CONFIGS[2], 60)
    pos, q, d = w.arrays()
    seed = 0x1234567_89ABCDEF
    o = Oracle(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, seed)
    o.sweep_index = (1 << 33) + 5          # exercise the high counter word
    s = o.sweep_index
    o.sweep(1)
    log = o.trial_log()
    for i in range(w.N):
        t, _ = py_trial(seed, s, i, pos[:, i], w.max_disp)
        assert tuple(log["trial"][:, i]) == tuple(t)
        assert np.all(np.abs(log["trial"][:, i] - pos[:, i]) <= w.max_disp)


# ---- P3 -----------------------------------------------------------------------------------------
@pytest.mark.parametrize("z1,z2", [(1.0, -1.0), (2.0, 3.0), (-1.0, -2.0)])
def test_p3_two_ion_closed_form(z1, z2):
    lB = 1.68
    pos = np.array([[0.3, -0.9], [0.1, 0.4], [-0.2, 0.7]])
    q = np.array([z1, z2]); d = np.array([1.0, 0.8])
    r = math.dist(pos[:, 0], pos[:, 1])
    o = Oracle(pos, q, d, 4.0, lB, 0.3, 7)
    assert o.energy() == pytest.approx(z1 * z2 * lB / r, rel=1e-15)
    assert o.stats()["E_running"] == pytest.approx(z1 * z2 * lB / r, rel=1e-15)
    # dE of the first trial is l_B z1 z2 (1/r' - 1/r)
    o.partial_sweep(0, 1)
    log = o.trial_log()
    rn = math.dist(log["trial"][:, 0], pos[:, 1])
    assert log["dE"][0] == pytest.approx(lB * z1 * z2 * (1 / rn - 1 / r), rel=1e-13)


# ---- P4 -----------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", [1, 2, 3])
def test_p4_brute_force_total_energy_differences(seed):
    """Per trial: E_total(after) - E_total(before), from scratch, equals the logged dE.

    Catches a wrong sign, a dropped partner, the wrong (old/new) position of j<i or j>i, a
    missing prefactor.  Also checks the veto bits and the decision against their definitions.
    """
    lB, R, delta = 1.68, 3.2, 0.6
    q = np.array([2.0, -1.0, -1.0, 1.0, -1.0, 3.0, -2.0, -1.0])
    d = np.array([1.0, 0.8, 0.8, 1.0, 0.9, 1.2, 1.0, 0.8])
    N = len(q)
    pos = W.random_sequential_insertion(d, R, seed)
    o = Oracle(pos, q, d, R, lB, delta, seed)
    cur = pos.copy()
    E_run = energy_exact(cur, q, lB)
    n_acc = 0
    for s in range(12):
        o.sweep(1)
        log = o.trial_log()
        for i in range(N):
            t, u_acc = py_trial(seed, s, i, cur[:, i], delta)
            assert tuple(log["trial"][:, i]) == tuple(t)
            trial = cur.copy(); trial[:, i] = t
            ov = any(math.dist(trial[:, i], trial[:, j]) ** 2 < (0.5 * (d[i] + d[j])) ** 2
                     for j in range(N) if j != i)
            wall = math.fsum(c * c for c in t) > (R - 0.5 * d[i]) ** 2
            f = int(log["flags"][i])
            assert bool(f & 2) == ov and bool(f & 4) == wall
            if not ov:
                dE = energy_exact(trial, q, lB) - energy_exact(cur, q, lB)
                assert abs(log["dE"][i] - dE) <= 1e-12 * max(1.0, log["scale"][i])
                if not wall and abs(dE + math.log(u_acc)) > 1e-9:
                    assert bool(f & 1) == (dE + math.log(u_acc) < 0)
            else:
                assert not f & 1
            if wall:
                assert not f & 1
            if f & 1:
                cur = trial
                E_run += log["dE"][i]
                n_acc += 1
        assert np.array_equal(o.positions, cur)
    assert 0 < n_acc < 12 * N
    assert o.stats()["accepted"] == n_acc
    assert o.stats()["E_running"] == pytest.approx(energy_exact(cur, q, lB), abs=1e-11)


# ---- P5, P6 ---------------------------------------------------------------------------------------
def test_p5_p6_bookkeeping_and_hard_constraints_config1():
    w = W.CONFIGS[0]
    pos, q, d = w.arrays()
    o = Oracle(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, w.seed)
    E0 = o.energy()
    tot_abs = 0.0
    for _ in range(20):
        o.sweep(5)
        p = o.positions
        # P6: no overlaps, everyone inside, nothing else touched
        assert pdist(p.T).min() >= 1.0                      # all diameters are 1 in config 1
        assert np.all(np.einsum("ij,ij->j", p, p) <= (w.cavity_R - 0.5) ** 2)
        log = o.trial_log()
        tot_abs += np.abs(log["dE"][(log["flags"] & 1) == 1]).sum()
    st = o.stats()
    assert o.sweep_index == 100
    # P5: E(init) + sum of accepted dE == from-scratch E(final)
    assert abs(st["E_running"] - o.energy()) <= 1e-9 * max(1.0, 5 * tot_abs)
    assert 0.2 < st["accepted"] / (100 * w.N) < 0.9
    assert st["near_ties"] == 0
    assert q.sum() == 0
    # energy() itself against the plain definition evaluated with numpy
    p = o.positions
    iu = np.triu_indices(w.N, 1)
    Enp = w.bjerrum * np.sum((q[:, None] * q[None, :])[iu] / pdist(p.T))
    assert o.energy() == pytest.approx(Enp, rel=1e-12)
    assert E0 != o.energy()


def test_p6_mixed_diameters_no_overlap():
    w = W.scaled(W.CONFIGS[2], 300)
    pos, q, d = w.arrays()
    o = Oracle(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 3)
    o.sweep(30)
    p = o.positions
    dist = pdist(p.T)
    iu = np.triu_indices(w.N, 1)
    sij = 0.5 * (d[:, None] + d[None, :])[iu]
    assert np.all(dist >= sij * (1 - 1e-15))
    assert np.all(np.sqrt(np.einsum("ij,ij->j", p, p)) <= w.cavity_R - 0.5 * d + 1e-12)


# ---- P7 -----------------------------------------------------------------------------------------
def test_p7_zero_displacement_accepts_everything_and_moves_nothing():
    w = W.scaled(W.CONFIGS[0], 64)
    pos, q, d = w.arrays()
    o = Oracle(pos, q, d, w.cavity_R, w.bjerrum, 0.0, 9)
    o.sweep(3)
    assert o.stats()["accepted"] == 3 * w.N
    assert np.array_equal(o.positions, pos)
    assert np.all(o.trial_log()["dE"] == 0.0)


def test_p7_zero_bjerrum_is_pure_hard_spheres():
    w = W.scaled(W.CONFIGS[3], 128)
    pos, q, d = w.arrays()
    o = Oracle(pos, q, d, w.cavity_R, 0.0, 0.4, 9)
    for _ in range(5):
        o.sweep(1)
        f = o.trial_log()["flags"]
        assert np.array_equal((f & 1) == 1, (f & 6) == 0)      # accept <=> no veto
    assert o.stats()["veto_overlap"] > 0


def test_p7_single_ion_accepts_iff_inside_wall():
    o = Oracle(np.array([[0.9], [0.0], [0.0]]), np.array([1.0]), np.array([1.0]), 1.5, 1.68, 0.5, 4)
    n_in = 0
    for s in range(200):
        before = o.positions
        o.sweep(1)
        log = o.trial_log()
        inside = np.sum(log["trial"][:, 0] ** 2) <= 1.0 ** 2
        assert bool(log["flags"][0] & 1) == inside and bool(log["flags"][0] & 4) == (not inside)
        assert np.array_equal(o.positions[:, 0], log["trial"][:, 0] if inside else before[:, 0])
        n_in += inside
    assert 0 < n_in < 200


def test_p7_trial_exactly_on_another_ion_is_vetoed_without_nan():
    pos = np.array([[0.0, 5.0], [0.0, 0.0], [0.0, 0.0]])
    q = np.array([1.0, -1.0]); d = np.array([1.0, 1.0])
    t, _ = py_trial(21, 0, 0, pos[:, 0], 0.5)
    pos[:, 1] = t                                            # ion 1 sits where ion 0 will try to go
    o = Oracle(pos, q, d, 8.0, 1.68, 0.5, 21, validate=False)
    o.partial_sweep(0, 1)
    f = o.trial_log()["flags"][0]
    assert f & 2 and not f & 1
    assert math.isfinite(o.stats()["E_running"])
    assert np.array_equal(o.positions, pos)


def test_init_validation_errors():
    q = np.array([1.0, -1.0]); d = np.array([1.0, 1.0])
    with pytest.raises(OracleError) as e:
        Oracle(np.array([[0.0, 0.5], [0, 0], [0, 0.0]]), q, d, 5.0, 1.68, 0.1, 1)
    assert e.value.code == -2
    with pytest.raises(OracleError) as e:
        Oracle(np.array([[0.0, 4.8], [0, 0], [0, 0.0]]), q, d, 5.0, 1.68, 0.1, 1)
    assert e.value.code == -3
    with pytest.raises(OracleError) as e:
        Oracle(np.array([[0.0, 2.0], [0, 0], [0, np.nan]]), q, d, 5.0, 1.68, 0.1, 1)
    assert e.value.code == -1
    # touching is allowed both for the pair and for the wall (readings G6, G7)
    Oracle(np.array([[0.0, 1.0], [0, 0], [0, 0.0]]), q, d, 1.5, 1.68, 0.1, 1)


# ---- P10 ----------------------------------------------------------------------------------------
def test_p10_reentrancy_and_resume():
    w = W.scaled(W.CONFIGS[1], 200)
    pos, q, d = w.arrays()
    a = Oracle(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 5)
    b = Oracle(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 5)
    a.sweep(3); a.sweep(4)
    b.sweep(7)
    assert np.array_equal(a.positions, b.positions)
    assert a.stats() == b.stats()
    # checkpoint / resume through positions + sweep index
    c = Oracle(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 5)
    c.sweep(3)
    r = Oracle(c.positions, q, d, w.cavity_R, w.bjerrum, w.max_disp, 5)
    r.sweep_index = 3
    r.sweep(4)
    assert np.array_equal(r.positions, b.positions)
    # a different seed gives a different chain
    e = Oracle(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 6)
    e.sweep(7)
    assert not np.array_equal(e.positions, b.positions)


def test_threaded_variant_matches_serial():
    w = W.scaled(W.CONFIGS[2], 700)
    pos, q, d = w.arrays()
    a = Oracle(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 2)
    b = Oracle(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 2, threads=4)
    for _ in range(3):
        a.sweep(1); b.sweep(1)
        la, lb = a.trial_log(), b.trial_log()
        assert np.array_equal(la["flags"], lb["flags"])
        ok = (la["flags"] & 2) == 0
        assert np.all(np.abs(la["dE"][ok] - lb["dE"][ok]) <= 1e-13 * np.maximum(1.0, la["scale"][ok]))
    assert np.array_equal(a.positions, b.positions)


# ---- pair histogram against a library routine ------------------------------------------------
def test_pair_hist_against_numpy():
    w = W.scaled(W.CONFIGS[2], 500)
    pos, q, d = w.arrays()
    o = Oracle(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 2)
    o.sweep(2)
    p = o.positions
    bw, nb, crm = 0.05, 40, 0.6 * w.cavity_R
    hist, nc = o.pair_hist(bw, nb, crm)
    sp = np.where(q > 0, 0, 1)
    centre = np.einsum("ij,ij->j", p, p) <= crm * crm
    ref = np.zeros((2, 2, nb), dtype=np.uint64)
    diff = p[:, :, None] - p[:, None, :]
    r = np.sqrt(np.einsum("kij,kij->ij", diff, diff))
    b = np.floor(r * (1.0 / bw))
    for i in np.nonzero(centre)[0]:
        for j in range(w.N):
            if j != i and b[i, j] < nb:
                ref[sp[i], sp[j], int(b[i, j])] += 1
    assert np.array_equal(hist, ref)
    assert list(nc) == [int(np.sum(centre & (sp == 0))), int(np.sum(centre & (sp == 1)))]
    assert hist.sum() > 0 and hist[:, :, : int(0.8 / bw)].sum() == 0   # nothing inside the hard core
    # accumulates
    hist2, nc2 = o.pair_hist(bw, nb, crm, hist.copy(), nc.copy())
    assert np.array_equal(hist2, 2 * ref) and np.array_equal(nc2, 2 * nc)


def test_pair_hist_hand_placed_example():
    """A configuration whose histogram can be written down by hand (reading G17):
    known distances on and off bin edges, both species, one centre just inside and one just outside
    centre_rmax.  Pins the [centre species][partner species] order, the bin edges (left-closed:
    bin k = [k w, (k+1) w)), the <= at centre_rmax, the dropped bins >= nbins and the ordered-pair count."""
    # ions on the x axis: index, x, charge
    #   0: 0.0   +     1: 1.5   -     2: 3.0   +     3: 6.0   -      4: (0, 2.0, 0) -
    pos = np.array([[0.0, 1.5, 3.0, 6.0, 0.0],
                    [0.0, 0.0, 0.0, 0.0, 2.0],
                    [0.0, 0.0, 0.0, 0.0, 0.0]])
    q = np.array([1.0, -1.0, 1.0, -1.0, -1.0])
    d = np.full(5, 1.0)
    o = Oracle(pos, q, d, 50.0, 1.68, 0.1, 1)
    bw, nb = 0.5, 8                     # bins [0,.5) [.5,1) ... [3.5,4.0); r >= 4.0 is dropped
    # centre_rmax = 3.0: ions 0 (r=0), 1 (1.5), 2 (3.0, ON the limit: counts, <=), 4 (2.0) are centres; 3 (6.0) is not
    hist, nc = o.pair_hist(bw, nb, 3.0)
    assert list(nc) == [2, 2]           # centres: + {0, 2}, - {1, 4}
    exp = np.zeros((2, 2, nb), dtype=np.uint64)
    P, M = 0, 1
    def add(a, b, r):
        k = int(np.floor(r / bw))
        if k < nb:
            exp[a, b, k] += 1
    # centre 0 (+): partners 1 (-, 1.5 -> bin 3 exactly on the edge 1.5 = 3 w), 2 (+, 3.0 -> bin 6), 3 (-, 6.0 dropped), 4 (-, 2.0 -> bin 4)
    add(P, M, 1.5); add(P, P, 3.0); add(P, M, 6.0); add(P, M, 2.0)
    # centre 1 (-): 0 (+, 1.5), 2 (+, 1.5), 3 (-, 4.5 dropped), 4 (-, 2.5 -> bin 5)
    add(M, P, 1.5); add(M, P, 1.5); add(M, M, 4.5); add(M, M, 2.5)
    # centre 2 (+): 0 (+, 3.0), 1 (-, 1.5), 3 (-, 3.0 -> bin 6), 4 (-, sqrt(13) = 3.606 -> bin 7)
    add(P, P, 3.0); add(P, M, 1.5); add(P, M, 3.0); add(P, M, np.sqrt(13.0))
    # centre 4 (-): 0 (+, 2.0), 1 (-, 2.5), 2 (+, 3.606), 3 (-, sqrt(40) dropped)
    add(M, P, 2.0); add(M, M, 2.5); add(M, P, np.sqrt(13.0)); add(M, M, np.sqrt(40.0))
    assert np.array_equal(hist, exp), (hist, exp)
    # written out: the table above in numbers
    assert hist[P, M, 3] == 2 and hist[P, P, 6] == 2 and hist[P, M, 4] == 1 and hist[P, M, 6] == 1 and hist[P, M, 7] == 1
    assert hist[M, P, 3] == 2 and hist[M, M, 5] == 2 and hist[M, P, 4] == 1 and hist[M, P, 7] == 1
    assert hist.sum() == 13
    # just inside the limit: ion 2 leaves the centres, nothing else changes
    hist2, nc2 = o.pair_hist(bw, nb, 3.0 - 1e-12)
    assert list(nc2) == [1, 2] and hist2.sum() == 13 - 4
    # not symmetric in (centre, partner): ion 3 is a partner but never a centre
    assert hist[P, M].sum() != hist[M, P].sum()


def test_pair_hist_threaded_matches_serial():
    w = W.scaled(W.CONFIGS[2], 900)
    pos, q, d = w.arrays()
    a = Oracle(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 2)
    b = Oracle(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 2, threads=4)
    ha, na = a.pair_hist(0.05, 60, 0.7 * w.cavity_R)
    hb, nb_ = b.pair_hist(0.05, 60, 0.7 * w.cavity_R)
    assert np.array_equal(ha, hb) and np.array_equal(na, nb_) and ha.sum() > 0


# ---- FP32-position variant -----------------------------------
def test_fp32_position_mode_holds_only_fp32_values_and_rounds_the_trial_once_more():
    from fractions import Fraction
    w = W.scaled(W.CONFIGS[2], 300)
    pos, q, d = w.arrays()
    o = Oracle(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 9)
    o.set_position_bits(32)
    p0 = o.positions
    assert np.array_equal(p0, pos.astype(np.float32).astype(np.float64))            # rounded to nearest at the switch
    assert abs(o.stats()["E_running"] - o.energy()) < 1e-12 * abs(o.energy())         # running energy of the rounded state
    o.sweep(1)
    lg = o.trial_log()
    # every proposed position = float32( correctly rounded fma(u - 1/2, 2 delta, x) ), checked with exact rationals
    D = Fraction(2.0 * w.max_disp)
    for i in (0, 1, 17, 150, 299):
        A = philox4x32_10((i, 0, 0, 0), (9, 0)); B = philox4x32_10((i, 0, 0, 1), (9, 0))
        u = [uniform_open01(A[0], A[1]), uniform_open01(A[2], A[3]), uniform_open01(B[0], B[1])]
        for k in range(3):
            # x_i at its turn: unchanged since the switch unless an earlier particle... no: only i moves x_i
            exact = (Fraction(u[k]) - Fraction(1, 2)) * D + Fraction(p0[k, i])
            want = float(np.float32(float(exact)))                                   # double rounding, as defined
            assert lg["trial"][k, i] == want
    p1 = o.positions
    assert np.array_equal(p1, p1.astype(np.float32).astype(np.float64))              # still FP32 values after a sweep
    assert (lg["flags"] & 1).sum() > 30
    # the invariants hold in this mode as well (P5, P6)
    o.sweep(20)
    assert abs(o.stats()["E_running"] - o.energy()) < 1e-9 * abs(o.energy())
    x = o.positions.T
    r = np.linalg.norm(x[:, None] - x[None], axis=2) + np.eye(w.N) * 10
    assert (r >= 0.5 * (d[:, None] + d[None, :]) * (1 - 1e-15)).all()
    # and it is a different chain from the FP64 one
    o64 = Oracle(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, 9)
    o64.sweep(21)
    assert not np.array_equal(o64.positions, o.positions)
