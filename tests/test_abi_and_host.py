"""CPU-only checks (-m "not gpu"): the C-ABI library builds for sm_100a, loads, and exports every symbol
include/mcb200.h declares; the host-side logic of bench.py (timing aggregation over ranks with gloo,
world_size 2; the reference arm) works without a GPU.  No compute call is made into libmcb200 here."""
import json
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "mcb200.h")


def declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mc_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    from paper_1602_05716_b200.build import build_extension
    from paper_1602_05716_b200 import binding
    build_extension()
    return binding.load_library()


def test_header_declares_the_boundary_of_survey_8b():
    names = declared_symbols()
    for must in ("mc_workspace_bytes", "mc_init", "mc_sweep", "mc_energy", "mc_pair_hist", "mc_get_positions",
                 "mc_set_positions", "mc_get_sweep_index", "mc_set_sweep_index", "mc_get_stats", "mc_get_trial_log",
                 "mc_free", "mc_last_error"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    from paper_1602_05716_b200 import binding
    names = declared_symbols()
    assert sorted(binding.EXPORTS) == names, "binding.EXPORTS and include/mcb200.h disagree"
    for n in names:
        assert hasattr(lib, n), f"libmcb200.so does not export {n}"
    out = subprocess.run(["nm", "-D", "--defined-only", str(binding._LIBPATH)], capture_output=True, text=True,
                         check=True).stdout
    exported = set(re.findall(r"\bT (mc_[a-z0-9_]+)", out))
    assert set(names) <= exported


def test_library_is_sm100a_native_with_bulk_async_copies(lib):
    from paper_1602_05716_b200 import binding
    out = subprocess.run(["cuobjdump", "-lelf", str(binding._LIBPATH)], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    sass = subprocess.run(["cuobjdump", "-sass", str(binding._LIBPATH)], capture_output=True, text=True).stdout
    sweep = [blk for blk in sass.split("Function :")[1:] if "k_sweep" in blk.splitlines()[0]]
    assert len(sweep) == 24, "k_sweep: 4 row counts x 2 diameter paths x 3 pair-distance forms"
    for blk in sweep:
        assert "UBLKCP" in blk          # cp.async.bulk (TMA unit) staging of the column ring
        assert "SYNCS" in blk           # mbarrier transactions
        assert "MUFU.RSQ64H" in blk     # FP64 rsqrt seed
        assert "DFMA" in blk
        assert "VIMNMX3" in blk         # integer overlap veto off the FP64 pipe


def test_host_argument_checks_need_no_gpu(lib):
    from paper_1602_05716_b200 import binding as B
    assert lib.mc_workspace_bytes(0) == 0
    assert lib.mc_workspace_bytes(65536) > 65536 * 64
    assert lib.mc_workspace_bytes(65536) % 256 == 0
    assert lib.mc_sweep(None, 1) == B.MC_EINVAL
    assert lib.mc_energy(None, None) == B.MC_EINVAL
    assert lib.mc_get_stats(None, None) == B.MC_EINVAL
    assert b"null" in lib.mc_last_error() or b"bad" in lib.mc_last_error()
    assert lib.mc_free(None) == B.MC_OK


def test_product_fails_loudly_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import numpy as np
    from paper_1602_05716_b200.binding import MCSystem
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        MCSystem(np.zeros((3, 1)), np.ones(1), np.ones(1), 2.0, 1.0, 0.1, 1)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1602_05716_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "oracle/" not in text or f.endswith((".cuh", ".cu")), f
    otext = open(os.path.join(ROOT, "oracle", "oracle.cpp")).read() + open(os.path.join(ROOT, "oracle", "binding.py")).read()
    assert "paper_1602_05716_b200" not in otext.replace("paper_1602_05716_b200/csrc (the CUDA path)", "")
    assert "mcb200.h" not in otext


def _gloo_worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    sys.path.insert(0, ROOT)
    import bench
    ms, units = bench.aggregate_over_ranks(10.0 + 5.0 * rank, 1000.0 * (rank + 1), world, dist, None)
    q.put((rank, ms, units))
    dist.barrier()
    dist.destroy_process_group()


def test_replica_timing_aggregation_world_size_2_gloo():
    import socket
    import torch.multiprocessing as mp
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_gloo_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # whole-job units = sum over replicas, time = max over ranks, on every rank
    assert got == [(0, 15.0, 3000.0), (1, 15.0, 3000.0)]


def test_bench_helpers():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate_over_ranks(3.0, 7.0, 1) == (3.0, 7.0)
    assert abs(bench.fp64_nominal_peak(148, 1965.0) - 1.861e13) < 1e10
    with bench.ClockSampler(0, period=0.01) as c:
        pass
    s = c.summary()
    assert set(s) >= {"sm_mhz", "sm_max_mhz", "reasons"}


def test_gpus_flag_spawns_the_replicas_itself_outside_torchrun(monkeypatch):
    """python bench.py --gpus N without WORLD_SIZE starts N ranks through torch.distributed.run on 127.0.0.1."""
    sys.path.insert(0, ROOT)
    import bench
    seen = {}
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    monkeypatch.setattr(bench, "spawn_replicas", lambda n, argv: seen.update(n=n, argv=argv) or 0)
    assert bench.main(["--gpus", "4", "--steps", "2", "--warmup", "3"]) == 0
    assert seen == {"n": 4, "argv": ["--gpus", "4", "--steps", "2", "--warmup", "3"]}
    cmd = []
    monkeypatch.undo()
    bench.spawn_replicas(2, ["--gpus", "2"], runner=lambda c: cmd.extend(c) or 0)
    assert "torch.distributed.run" in cmd and "--nproc-per-node=2" in cmd and "127.0.0.1" in cmd
    assert cmd[-2:] == ["--gpus", "2"] and cmd[-3].endswith("bench.py")


def test_reference_arm_prints_one_json_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload",
                          "rpm_1to1_n4096", "--steps", "1", "--warmup", "0"], capture_output=True, text=True,
                         timeout=300, check=True).stdout.strip().splitlines()
    line = json.loads(out[-1])
    assert line["impl"] == "reference" and line["value"] > 1e5 and line["unit"] == "pair_evals/s"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0


@pytest.mark.parametrize("N", [1, 2, 31, 33, 255, 257, 512, 1023, 1025, 4096, 16383, 65536, 100001])
@pytest.mark.parametrize("rows", [1, 2, 3, 4])
def test_persistent_kernel_items_cover_every_column_exactly_once(N, rows):
    """Host logic of csrc/persist.cuh: FAR-L + FAR-U + MID + FIX + DIAG partition the N columns of every chunk
    (Eq. 2: each partner enters a trial's sum exactly once)."""
    from paper_1602_05716_b200.binding import mc_plan_check
    for far_cols, workers in ((8, 0), (64, 0), (256, 290), (256, 7), (1024, 290), (65536, 3)):
        r = mc_plan_check(N, rows, far_cols, workers)
        assert r["violations"] == 0, (N, rows, far_cols, workers, r)
        assert r["items"] > 0
