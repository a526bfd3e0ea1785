#!/usr/bin/env python
"""bench.py -- throughput of the exact sequential Metropolis sweep (arXiv 1602.05716) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl ours|reference]

Metric (BASELINE.json): Coulomb pair evaluations per second (and sweeps/s) at N = 65536 -- config 4 of
BASELINE.json, ``rpm_1to1_n65536``.  One STEP is one pass of every row of SURVEY.md 8(a) over the
configuration: one full sequential sweep (a1-a4: N trials = N(N-1) pair evaluations), one g(r) histogram
sample (a6: 500 bins of 0.02 sigma, bulk centres) and one from-scratch energy (a5).  Only the N(N-1) pair
evaluations of the sweep count towards the metric; histogram, energy, speculative and correction work do not.

Multi-GPU: replicas only -- every rank runs an independent chain (seed + rank) of the
same size, no data-path collective; value = all ranks' pair evaluations / max-over-ranks time ("weak").

``--impl reference`` times the CPU oracle (oracle/, test infrastructure) on the host cores on a bounded
sample of the same workload; it is a deliberately plain program, a baseline and not the target.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "coulomb_pair_evaluations_per_second"
UNIT = "pair_evals/s"
FP64_INSTR_PER_PAIR = 27          # SURVEY.md 8(d) canonical count
FP64_LANES_PER_SM = 64            # DFMA lanes per SM per clock (confirmed by mc_measure_fp64_peak)
L2_FLUSH_BYTES = 256 << 20        # > 126 MB L2
# FP64-pipe instructions the sweep kernel EXECUTES per pair, by pair-distance form (persist.cuh) and
# (equal diameters, mixed diameters); the roofline fraction credits the canonical 27 whatever the form
EXECUTED_FP64_PER_PAIR = {0: (20, 22), 1: (22, 24), 2: (25, 27)}


# ---------------------------------------------------------------------------------------------------
# helpers that hold no GPU work (covered by the CPU tests)
# ---------------------------------------------------------------------------------------------------
def dist_env():
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def aggregate_over_ranks(local_ms: float, local_units: float, world: int, dist=None, device=None):
    """(max-over-ranks milliseconds, sum-over-ranks units).  Replicas only: these two all-reduces of the
    TIMING are the only communication; the data path has none."""
    if world == 1 or dist is None:
        return local_ms, local_units
    import torch
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([local_units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def fp64_nominal_peak(num_sms: int, sm_mhz: float) -> float:
    """Thread-level FP64-pipe instructions per second: lanes/SM x SMs x clock."""
    return FP64_LANES_PER_SM * num_sms * sm_mhz * 1e6


TRAFFIC_FILE = os.path.join("profiles", "r02_k_sweep_traffic.csv")


def read_measured_traffic():
    """DRAM bytes per launch of the dominant kernel (dram__bytes_read.sum + dram__bytes_write.sum of one
    ``ncu --set full`` capture of this command, kept under profiles/), or None if there is no capture."""
    path = os.path.join(ROOT, TRAFFIC_FILE)
    try:
        with open(path) as f:
            for line in f:
                parts = line.strip().split(",")
                if parts[0] == "dram_bytes_per_launch":
                    return float(parts[2])
    except (OSError, ValueError, IndexError):
        pass
    return None


class ClockSampler:
    """Samples SM clock and throttle reasons of one GPU through NVML while the timed region runs."""
    BAD = {"hw_slowdown": 0x8, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40}
    NOTE = {"sw_power_cap": 0x4, "hw_power_brake": 0x80, "sync_boost": 0x10}

    def __init__(self, index: int, period=0.1):
        self.index, self.period = index, period
        self.samples, self.reasons = [], 0
        self.max_mhz = None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nv = None

    def _loop(self):
        nv = self._nv
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                self.reasons |= int(nv.nvmlDeviceGetCurrentClocksEventReasons(self._h))
            except Exception:
                try:
                    self.reasons |= int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                except Exception:
                    pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self._nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self) -> dict:
        names = [k for k, bit in {**self.BAD, **self.NOTE}.items() if self.reasons & bit]
        return {"sm_mhz": statistics.median(self.samples) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": names, "samples": len(self.samples)}


# ---------------------------------------------------------------------------------------------------
# the reference arm: the CPU oracle, as it stands, on the host cores
# ---------------------------------------------------------------------------------------------------
def oracle_sample_rate(w, threads: int, seconds: float, state=None):
    """Pair evaluations per second of the oracle on a bounded sample: consecutive trials (in sweep order,
    continuing into the next sweeps) for about ``seconds``.  Returns (rate, trials done, seconds, state)."""
    from oracle import Oracle
    if state is None:
        pos, q, d = w.arrays()
        state = {"o": Oracle(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, w.seed, validate=False, threads=threads),
                 "next": 0}
        state["o"].partial_sweep(0, min(8, w.N))          # thread start-up, untimed
        state["next"] = min(8, w.N) % w.N
    o = state["o"]
    done, spent, batch = 0, 0.0, 32
    while spent < seconds:
        first = state["next"]
        cnt = min(batch, w.N - first)
        t0 = time.perf_counter()
        o.partial_sweep(first, cnt)
        dt = time.perf_counter() - t0
        spent += dt
        done += cnt
        state["next"] = first + cnt
        if state["next"] >= w.N:                          # next sweep of the same chain
            o.sweep_index = o.sweep_index + 1
            state["next"] = 0
        if dt < 0.25 * seconds:
            batch = min(w.N, max(batch, int(batch * min(8.0, 0.25 * seconds / max(dt, 1e-6)))))
    return done * (w.N - 1) / spent, done, spent, state


def run_reference(args, w):
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    cores = os.cpu_count() or 1
    per_step = max(0.5, min(15.0, 150.0 / max(1, args.steps + args.warmup)))
    state = None
    for _ in range(args.warmup):
        _, _, _, state = oracle_sample_rate(w, cores, per_step, state)
    tot_pairs, tot_s, trials = 0.0, 0.0, 0
    for _ in range(args.steps):
        r, n, s, state = oracle_sample_rate(w, cores, per_step, state)
        tot_pairs += r * s
        tot_s += s
        trials += n
    value = tot_pairs / tot_s
    sample = (f"{trials} consecutive trials in sweep order in {args.steps} steps (~{per_step:.1f} s each), "
              f"each trial against all N-1 partners, OpenMP over j")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_s / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(w, world=1, parallelism="cpu"),
            "sweeps_per_s": value / w.pair_evals_per_sweep,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                             "note": "the plain scalar parity oracle as it stands, not a tuned CPU code"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def workload_config(w, world, parallelism):
    return {"workload": w.name, "N": w.N, "species": [[s.count, s.valence, s.diameter] for s in w.species],
            "rho_star": w.rho_star, "cavity_R": w.cavity_R, "bjerrum": w.bjerrum, "max_disp": w.max_disp,
            "seed": w.seed, "hist": {"bin_width": w.hist_bin_width, "nbins": w.hist_nbins,
                                     "centre_rmax": w.hist_centre_rmax},
            "step": "1 sweep (N trials) + 1 mc_pair_hist + 1 mc_energy",
            "pair_evals_per_step": w.pair_evals_per_sweep,
            "l2": "flushed between steps (256 MiB memset, inside the timed region)",
            "parallelism": parallelism, "replicas": world}


# ---------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------
def run_ours(args, w):
    import torch
    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU path (use --impl reference for the oracle)")
    dist = None
    if world > 1:
        import torch.distributed as dist
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    else:
        torch.cuda.set_device(0)
    dev = torch.device("cuda", torch.cuda.current_device())
    from paper_1602_05716_b200.binding import MCSystem, mc_measure_fp64_peak

    pos, q, d = w.arrays()
    sysm = MCSystem(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, w.seed + rank, validate=False)
    sysm.mc_set_positions(pos)                      # E_running := from-scratch energy
    N, pairs_per_step = w.N, w.pair_evals_per_sweep
    hist = torch.zeros((2, 2, w.hist_nbins), dtype=torch.int64, device=dev)
    ncent = torch.zeros(2, dtype=torch.int64, device=dev)
    e_dev = torch.zeros(1, dtype=torch.float64, device=dev)
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()

    def step():
        sysm.mc_sweep(1)
        sysm.mc_pair_hist(w.hist_bin_width, w.hist_nbins, w.hist_centre_rmax, hist, ncent)
        sysm.mc_energy_dev(e_dev)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    # ---- device-resident throughput: W warm-up steps, then exactly K timed steps ----
    for _ in range(max(args.warmup, 0)):
        step()
        flush.zero_()
    barrier()
    l0 = sysm.mc_get_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(torch.cuda.current_device()) as clk:
        ev0.record(stream)
        for _ in range(args.steps):
            step()
            flush.zero_()
        ev1.record(stream)
        barrier()
    ms_local = ev0.elapsed_time(ev1)
    launches = sysm.mc_get_launch_count() - l0
    ms, units = aggregate_over_ranks(ms_local, float(pairs_per_step) * args.steps, world, dist, dev)
    value = units / (ms * 1e-3)
    clocks = clk.summary()

    # ---- sweep only (a1-a4), same protocol, for the sweeps/s figure of the metric ----
    barrier()
    ev0.record(stream)
    for _ in range(args.steps):
        sysm.mc_sweep(1)
        flush.zero_()
    ev1.record(stream)
    barrier()
    ms_sweep, units_sweep = aggregate_over_ranks(ev0.elapsed_time(ev1), float(pairs_per_step) * args.steps, world,
                                                 dist, dev)

    # ---- end to end through host buffers: H2D of the configuration, the step, D2H of the results ----
    pin_in = torch.from_numpy(pos).pin_memory()
    pin_out = torch.empty((3, N), dtype=torch.float64).pin_memory()
    pin_hist = torch.empty((2, 2, w.hist_nbins), dtype=torch.int64).pin_memory()
    pin_ncent = torch.empty(2, dtype=torch.int64).pin_memory()

    e_run = [sysm.mc_get_stats()["E_running"]]
    pin_in.copy_(torch.from_numpy(sysm.positions))              # the chain's current state, with its running energy

    pins = [pin_in, pin_out]

    def step_e2e():
        hist.zero_(); ncent.zero_()
        # H2D positions (+ the running energy that belongs to them: no from-scratch pass), sweep, D2H positions + stats
        _, st = sysm.mc_sweep_host(1, pins[0], pins[1], E_running_in=e_run[0])
        e_run[0] = st["E_running"]
        sysm.mc_pair_hist(w.hist_bin_width, w.hist_nbins, w.hist_centre_rmax, hist, ncent)
        pin_hist.copy_(hist, non_blocking=True)
        pin_ncent.copy_(ncent, non_blocking=True)
        e = sysm.mc_energy()                                    # host scalar (synchronises)
        pins.reverse()                                          # the next step continues the chain: its input is this step's output buffer
        return st, e

    h2d = 3 * N * 8 + 8
    d2h = 3 * N * 8 + 40 + 4 * w.hist_nbins * 8 + 16 + 8
    for _ in range(min(args.warmup, 3)):
        step_e2e()
    barrier()
    t0 = time.perf_counter()
    ev0.record(stream)
    for _ in range(args.steps):
        step_e2e()
        flush.zero_()
    ev1.record(stream)
    barrier()
    wall_ms = (time.perf_counter() - t0) * 1e3
    ms_e2e, units_e2e = aggregate_over_ranks(max(ev0.elapsed_time(ev1), wall_ms), float(pairs_per_step) * args.steps,
                                             world, dist, dev)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel (k_sweep): CUDA events on the launching stream around its launch,
    #      average over the launches of a timed region of its own (L2 flushed in between, as in the steps) ----
    runs = []
    for _ in range(max(3, min(args.steps, 10))):
        flush.zero_()
        runs.append(sysm.mc_sweep_timed(1))
    bulk_ms, bulk_launches, bulk_pairs = sum(runs) / len(runs), 1, pairs_per_step
    # mc_sweep(n) is ONE launch: the per-sweep cost without the launch (what paces the small configurations)
    n_multi = max(2, min(100, w.sweeps))
    multi_ms = min(sysm.mc_sweep_timed(n_multi) for _ in range(3)) / n_multi
    # the paper's comparison code (one kernel launch per trial, parallel reduction), one sweep
    red_ms = None
    if not args.skip_comparison:
        ev0.record(stream)
        sysm.mc_sweep_reduction(1)
        ev1.record(stream)
        torch.cuda.synchronize()
        red_ms = ev0.elapsed_time(ev1)
    form = sysm.mc_get_option("form")
    executed = EXECUTED_FP64_PER_PAIR[form][0 if sysm.mc_get_option("uniform_path") else 1]
    prop = torch.cuda.get_device_properties(dev)
    sm_max = clocks["sm_max_mhz"] or 1965.0
    peak_instr = fp64_nominal_peak(prop.multi_processor_count, sm_max)
    measured_dfma = mc_measure_fp64_peak(100.0)
    achieved_instr = bulk_pairs * FP64_INSTR_PER_PAIR / (bulk_ms * 1e-3) if bulk_ms > 0 else 0.0
    roofline = {
        "bound": "alu", "kernel": "k_sweep (persistent: the whole sweep in one cooperative launch)",
        "achieved": 2.0 * achieved_instr / 1e12, "peak": 2.0 * peak_instr / 1e12, "unit": "TFLOP/s",
        "frac": achieved_instr / peak_instr, "traffic": read_measured_traffic(),
        "note": ("FP64 plain-ALU pipe; frac = ALGORITHMIC work / peak: 27 FP64-pipe instructions per pair evaluation "
                 "(SURVEY.md 8(d)), one FMA (2 flop) each, against peak = 64 lanes/SM x SMs x max SM clock (derived, "
                 "DESIGN.md section 4; MEASURED_PEAKS.json has no FP64 entry; the builder-measured DFMA rate of this "
                 "run is beside it). The kernel EXECUTES fewer instructions per pair (executed_fp64_per_pair), so "
                 "frac can exceed the pipe's own utilisation: pipe_utilisation_executed is that one"),
        "executed_fp64_per_pair": executed, "pair_distance_form": ("gram", "diffw", "canon")[form],
        "pipe_utilisation_executed": (bulk_pairs * executed / (bulk_ms * 1e-3) / measured_dfma) if bulk_ms > 0 else 0.0,
        "traffic_source": TRAFFIC_FILE,
        "launches_per_sweep": bulk_launches, "avg_launch_ms": bulk_ms / max(1, bulk_launches),
        "pairs_per_launch": bulk_pairs / max(1, bulk_launches),
        "builder_measured_dfma_per_s": measured_dfma, "frac_of_builder_measured_dfma_peak": achieved_instr / measured_dfma,
        "kernel_share_of_sweep": 1.0,     # trial generation, pair sums, resolution and commit are all inside k_sweep
    }
    step_frac = value / world * FP64_INSTR_PER_PAIR / peak_instr

    # ---- CPU baseline: the oracle as it stands, bounded sample, this box's cores ----
    cpu_baseline = None
    if not args.skip_cpu_baseline:
        cores = os.cpu_count() or 1
        cpu_all, n_all, s_all, _ = oracle_sample_rate(w, cores, 12.0)
        cpu_one, n_one, s_one, _ = oracle_sample_rate(w, 1, 8.0)
        cpu_baseline = {"value": cpu_all, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": (f"{n_all} consecutive trials in sweep order from sweep 0 at N={N} ({s_all:.1f} s, "
                                   f"OpenMP over j, {cores} threads)"),
                        "single_thread": {"value": cpu_one, "cores": 1,
                                          "sample": f"first {n_one} trials of sweep 0 ({s_one:.1f} s)"},
                        "note": "the plain scalar parity oracle as it stands, not a tuned CPU code",
                        "paper_context": "paper: 440x over one Xeon core on Tesla K20 (PAPER.md:315)"}

    st = sysm.mc_get_stats()
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": workload_config(w, world, f"replicas{world}"),
        "sweeps_per_s": value / pairs_per_step,
        "sweep_only": {"value": units_sweep / (ms_sweep * 1e-3), "unit": UNIT,
                       "sweeps_per_s": units_sweep / (ms_sweep * 1e-3) / pairs_per_step,
                       "ms_per_sweep": ms_sweep / args.steps,
                       "fp64_roofline_frac": units_sweep / (ms_sweep * 1e-3) / world * FP64_INSTR_PER_PAIR / peak_instr},
        "fp64_roofline_frac_whole_step": step_frac,
        "multi_sweep_launch": {"sweeps_per_launch": n_multi, "ms_per_sweep": multi_ms,
                               "value": pairs_per_step / (multi_ms * 1e-3), "unit": UNIT,
                               "fp64_roofline_frac": pairs_per_step / (multi_ms * 1e-3) * FP64_INSTR_PER_PAIR / peak_instr},
        "comparison_parallel_reduction": None if red_ms is None else {
            "ms_per_sweep": red_ms, "launches_per_sweep": N, "value": pairs_per_step / (red_ms * 1e-3), "unit": UNIT,
            "note": "the paper's comparison code (PAPER.md:278-282), same chain; context, not the product path"},
        "clocks": {k: clocks[k] for k in ("sm_mhz", "sm_max_mhz", "reasons")},
        "e2e": {"value": units_e2e / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "ms_per_step": ms_e2e / args.steps},
        "gpu_launches": int(launches),
        "roofline": roofline, "cpu_baseline": cpu_baseline,
        "acceptance_ratio": st["accepted"] / max(1, sysm.sweep_index * N),
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


def spawn_replicas(n: int, argv: list, runner=None) -> int:
    """``python bench.py --gpus N`` outside torchrun: start the N replicas itself, one process per GPU, the
    way the driver does (torch.distributed.run on 127.0.0.1); rank 0 of them prints the JSON line."""
    import socket
    import subprocess
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *argv]
    return (runner or subprocess.call)(cmd)


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default=None, help="workloads.CONFIGS name (default: the N=65536 headline)")
    ap.add_argument("--impl", choices=("ours", "reference"), default="ours")
    ap.add_argument("--skip-cpu-baseline", action="store_true",
                    help="leave out the oracle timing (profiling runs under ncu only)")
    ap.add_argument("--skip-comparison", action="store_true",
                    help="leave out the sweep through the paper's one-launch-per-trial comparison kernel (N launches)")
    args = ap.parse_args(argv)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "ours":
        return spawn_replicas(args.gpus, list(sys.argv[1:] if argv is None else argv))
    from paper_1602_05716_b200 import workloads as W
    w = W.by_name(args.workload) if args.workload else W.HEADLINE
    if args.impl == "reference":
        return run_reference(args, w)
    return run_ours(args, w)


if __name__ == "__main__":
    sys.exit(main())
