"""Option sweep of the sweep kernel's scheduling parameters for one system size:

    python -m paper_1602_05716_b200.tune [--n 65536] [--workload 3] [--sweeps 4] [--top 5] [--full]

Builds a synthetic electrolyte of ``--n`` ions with the composition, density and move size of BASELINE
configuration ``--workload`` (0..4), then times ``mc_sweep_timed`` (one launch of k_sweep running ``--sweeps``
sweeps) for every combination of the options that shape the work items -- ``prows`` (rows per thread, i.e. the chunk
size), ``far_cols`` and ``fix_cols`` (columns per FAR / FIX item), and with ``--full`` also ``pnear``,
``diag_split`` and ``wave``.  Every setting gives the same chain (tests/test_gpu_parity.py); only the time differs.
Prints the library's defaults for this size and the best settings found.  The defaults by N in csrc/mcb200.cu
(mc_init, launch_sweep) come from runs of this script on a B200 (profiles/r02_small_configs.md).
"""
from __future__ import annotations

import argparse
import itertools
import json
import sys


def run(n: int, workload: int, sweeps: int, top: int, full: bool) -> dict:
    import torch
    from . import workloads as W
    from .binding import MCSystem
    torch.cuda.set_device(0)
    base = W.CONFIGS[workload]
    w = base if n == base.N else W.scaled(base, n)
    pos, q, d = w.arrays()

    def fresh():
        g = MCSystem(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, w.seed, validate=False)
        g.mc_set_positions(pos)
        g.mc_sweep(2)
        return g

    def timed(g):
        return min(g.mc_sweep_timed(sweeps) for _ in range(2)) / sweeps * 1e3

    g = fresh()
    keys = ("prows", "far_cols", "fix_cols", "pnear", "diag_split", "wave")
    defaults = {k: g.mc_get_option(k) for k in keys}
    out = {"workload": w.name, "N": w.N, "sweeps_per_launch": sweeps, "defaults": defaults, "defaults_us_per_sweep": round(timed(g), 1)}
    grid = {"prows": (2, 3, 4) if w.N >= 2048 else (1, 2, 4), "far_cols": (64, 128, 192, 256, 384), "fix_cols": (4, 8, 16)}
    if full:
        grid.update({"pnear": (0, 4, 8, 16), "diag_split": (1, 2, 4, 8), "wave": (0, 1)})
    results = []
    names = list(grid)
    for combo in itertools.product(*(grid[k] for k in names)):
        for k, v in zip(names, combo):
            g.mc_set_option(k, v)
        results.append((round(timed(g), 1), dict(zip(names, combo))))
    results.sort(key=lambda r: r[0])
    out["best"] = [{"us_per_sweep": us, **opts} for us, opts in results[:top]]
    g.close()
    return out


def main(argv=None) -> int:
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--n", type=int, default=65536)
    ap.add_argument("--workload", type=int, default=3, help="BASELINE configuration whose composition is scaled to --n (0..4)")
    ap.add_argument("--sweeps", type=int, default=4, help="sweeps per timed launch")
    ap.add_argument("--top", type=int, default=5)
    ap.add_argument("--full", action="store_true", help="also sweep pnear, diag_split and wave (16x more settings)")
    args = ap.parse_args(argv)
    print(json.dumps(run(args.n, args.workload, args.sweeps, args.top, args.full)))
    return 0


if __name__ == "__main__":
    sys.exit(main())
