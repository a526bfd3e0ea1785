"""Self-check of an installed libmcb200 on the current GPU, without the oracle:

    python -m paper_1602_05716_b200.selfcheck [--n 2500] [--sweeps 3] [--prows 1|2|4] [--form -1|0|1|2]
                                              [--workload 0..4] [--stall-ms 2000]

Runs a few sweeps of a small synthetic electrolyte through the C ABI and checks what must hold for any
correct chain: E(init) + sum of accepted dE equals the from-scratch energy, no
overlap and nobody outside the wall, mc_sweep(a); mc_sweep(b) == mc_sweep(a + b) bit for bit, no stall, and
the pair histogram's total equals a direct count.  Small enough to run under compute-sanitizer (raise
--stall-ms there: the tools slow the kernels down by one to two orders of magnitude).
"""
from __future__ import annotations

import argparse
import sys

import numpy as np


def run(n=2500, sweeps=3, prows=None, form=-1, workload=2, stall_ms=2000, seed=3) -> dict:
    import torch
    from . import workloads as W
    from .binding import MCSystem
    torch.cuda.set_device(0)
    w = W.scaled(W.CONFIGS[workload], n)
    pos, q, d = w.arrays()

    def make():
        g = MCSystem(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, seed)
        if prows:
            g.mc_set_option("prows", prows)
        g.mc_set_option("form", form)
        g.mc_set_option("stall_ms", stall_ms)
        return g

    a, b = make(), make()
    e0 = a.mc_energy()
    a.mc_sweep(sweeps)
    for _ in range(sweeps):
        b.mc_sweep(1)
    st = a.mc_get_stats()                        # raises on MC_ESTALL
    pa, pb = a.positions, b.positions
    assert np.array_equal(pa, pb), "mc_sweep(a); mc_sweep(b) differs from mc_sweep(a + b)"
    assert st == b.mc_get_stats()
    e1 = a.mc_energy()
    assert abs(st["E_running"] - e1) <= 1e-9 * max(1.0, abs(e0) + abs(e1)), (st["E_running"], e1)
    assert st["accepted"] > 0 and a.sweep_index == sweeps
    # hard constraints by brute force (small n)
    x = pa.T
    r = np.linalg.norm(x[:, None, :] - x[None, :, :], axis=2)
    s = 0.5 * (d[:, None] + d[None, :])
    iu = np.triu_indices(w.N, 1)
    assert (r[iu] >= s[iu] * (1 - 1e-14)).all(), "overlapping ions after the sweeps"
    assert (np.linalg.norm(x, axis=1) <= (w.cavity_R - 0.5 * d) * (1 + 1e-14)).all(), "an ion left the cavity"
    # pair histogram: total count of the ordered pairs with a centre inside centre_rmax and r < nbins * bin_width
    bw, nb, rc = 0.1, 40, 0.5 * w.cavity_R
    h, nc = a.mc_pair_hist(bw, nb, rc)
    centre = np.linalg.norm(x, axis=1) <= rc
    direct = int(((r < bw * nb) & centre[:, None]).sum() - centre.sum())
    assert abs(int(h.sum().item()) - direct) <= 2, (int(h.sum().item()), direct)     # +-: pairs within an ulp of the last edge
    assert int(nc.sum().item()) == int(centre.sum())
    return {"N": w.N, "sweeps": sweeps, "prows": a.mc_get_option("prows"), "form": a.mc_get_option("form"),
            "accepted": st["accepted"], "E": e1, "launches": a.mc_get_launch_count()}


def main(argv=None) -> int:
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--n", type=int, default=2500)
    ap.add_argument("--sweeps", type=int, default=3)
    ap.add_argument("--prows", type=int, default=0)
    ap.add_argument("--form", type=int, default=-1)
    ap.add_argument("--workload", type=int, default=2)
    ap.add_argument("--stall-ms", type=int, default=2000)
    args = ap.parse_args(argv)
    out = run(args.n, args.sweeps, args.prows or None, args.form, args.workload, args.stall_ms)
    print("selfcheck ok:", out)
    return 0


if __name__ == "__main__":
    sys.exit(main())
