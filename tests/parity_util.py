"""Helpers of the GPU-vs-oracle parity tests (BASELINE.json north_star).

Agreement = identical accept / overlap-veto / wall-veto bits and identical positions in every
sweep, except trials the ORACLE flagged as near-ties (|dE + ln u| < 1e-8, reading G15), after which
the GPU chain is re-synchronised to the oracle's state; per-trial dE within
1e-10 * max(|dE_oracle|, M_i) for trials without an overlap veto (readings G13, G14).
"""
from __future__ import annotations

import numpy as np

DE_RTOL = 1e-10      # north_star: per-trial dE within 1e-10 relative (scale of reading G13)
POS_ATOL = 1e-12     # north_star: positions within 1e-12 sigma (they are in fact bit-identical)


def record_margin(name, **values):
    """Appends one line to gpurun_out/parity_margins.jsonl (the figures DESIGN.md section 3 quotes) and prints it."""
    import json
    import os
    line = json.dumps({"case": name, **values})
    print("parity margin:", line)
    try:
        d = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")
        os.makedirs(d, exist_ok=True)
        with open(os.path.join(d, "parity_margins.jsonl"), "a") as f:
            f.write(line + "\n")
    except OSError:
        pass


def make_pair(w, threads=1, validate=True, seed=None):
    """(gpu chain, oracle chain) for workload ``w`` from the same generated inputs."""
    from oracle import Oracle
    from paper_1602_05716_b200.binding import MCSystem
    pos, q, d = w.arrays()
    seed = w.seed if seed is None else seed
    g = MCSystem(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, seed, validate=validate)
    o = Oracle(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, seed, validate=validate, threads=threads)
    return g, o


def compare_last_sweep(g, o, tag="", first=0, count=None):
    """Compare the trial logs of the sweep both chains just ran.  Returns (max dE error, #near-ties that
    went the other way).  Raises AssertionError on any disagreement not excused by an oracle near-tie."""
    lg, lo = g.mc_get_trial_log(), o.trial_log()
    sl = slice(first, None if count is None else first + count)
    fg, fo = lg["flags"][sl], lo["flags"][sl]
    tie = (fo & 8) != 0
    diff = (fg & 7) != (fo & 7)
    bad = diff & ~tie
    assert not bad.any(), (f"{tag}: accept/veto bits differ from the oracle at trials "
                           f"{(np.nonzero(bad)[0][:8] + first).tolist()} (gpu {fg[bad][:8].tolist()}, "
                           f"oracle {fo[bad][:8].tolist()})")
    ok = ((fo & 2) == 0) & ~diff                      # dE of an overlapping trial is unspecified (G14)
    dg, do, sc = lg["dE"][sl][ok], lo["dE"][sl][ok], lo["scale"][sl][ok]
    err = np.abs(dg - do) / np.maximum(np.maximum(np.abs(do), sc), 1e-300)
    emax = float(err.max()) if err.size else 0.0
    assert emax <= DE_RTOL, f"{tag}: per-trial dE off by {emax:.3e} (limit {DE_RTOL})"
    return emax, int((diff & tie).sum())


def lockstep(g, o, sweeps, tag="", every=1, after_sweep=None):
    """Run both chains ``sweeps`` sweeps, comparing after every ``every`` sweeps.  ``after_sweep(done)`` is
    called once both chains are known to be in the same state.  Returns a summary."""
    import time
    worst, flips, done, t_oracle = 0.0, 0, 0, 0.0
    while done < sweeps:
        n = min(every, sweeps - done)
        g.mc_sweep(n)
        t0 = time.perf_counter()
        o.sweep(n)
        t_oracle += time.perf_counter() - t0      # the CPU-baseline protocol of SURVEY.md 8(d): the oracle's full runs, timed
        done += n
        e, f = compare_last_sweep(g, o, tag=f"{tag} sweep {done - 1}")
        worst = max(worst, e)
        pg, po = g.positions, o.positions
        if f:   # a flagged near-tie went the other way: legal (G15); re-synchronise and go on
            flips += f
            g.mc_set_positions(po)
            g.sweep_index = o.sweep_index
        else:
            assert np.array_equal(pg, po), (f"{tag} sweep {done - 1}: positions differ "
                                            f"(max {np.abs(pg - po).max():.3e})")
        if after_sweep is not None:
            after_sweep(done)
    return {"max_dE_err": worst, "near_tie_flips": flips, "oracle_seconds": t_oracle}


def assert_stats_equal(g, o, flips=0):
    sg, so = g.mc_get_stats(), o.stats()
    if flips == 0:
        for k in ("accepted", "veto_overlap", "veto_wall", "near_ties"):
            assert sg[k] == so[k], (k, sg[k], so[k])
    assert abs(sg["E_running"] - so["E_running"]) <= 1e-9 * max(1.0, abs(so["E_running"])), (sg, so)


def hard_constraints_ok(pos, d, R):
    """min_{i<j}(r_ij - s_ij) >= 0 and max_i(|x_i| - a_i) <= 0, by a k-d tree (test-side check only)."""
    from scipy.spatial import cKDTree
    x = np.ascontiguousarray(pos.T)
    tree = cKDTree(x)
    dmax = float(d.max())
    pairs = tree.query_pairs(r=dmax, output_type="ndarray")
    if len(pairs):
        r = np.linalg.norm(x[pairs[:, 0]] - x[pairs[:, 1]], axis=1)
        s = 0.5 * (d[pairs[:, 0]] + d[pairs[:, 1]])
        if (r < s * (1 - 1e-14)).any():
            return False
    return bool((np.linalg.norm(x, axis=1) <= (R - 0.5 * d) * (1 + 1e-14)).all())
