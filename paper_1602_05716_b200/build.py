"""Builds libmcb200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

Translation units (compiled in parallel, linked into one shared object):
  csrc/mcb200.cu                      the C ABI and every kernel but the sweep
  csrc/sweep_inst.cu -DMCB_FORM=0|1|2 the sweep kernel, one pair-distance form per unit
"""
from __future__ import annotations

import os
import subprocess
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIB = PKG / "libmcb200.so"
OBJDIR = PKG / "build"
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-fmad=false",  # every fused multiply-add in the kernels is written explicitly (reading G11)
    "-Xcompiler", "-fPIC",
]
UNITS = (
    ("mcb200", "mcb200.cu", ()),
    ("sweep_gram", "sweep_inst.cu", ("-DMCB_FORM=0",)),
    ("sweep_diffw", "sweep_inst.cu", ("-DMCB_FORM=1",)),
    ("sweep_canon", "sweep_inst.cu", ("-DMCB_FORM=2",)),
)


def _sources():
    return [*sorted(CSRC.glob("*.cu")), *sorted(CSRC.glob("*.cuh")), *sorted(CSRC.glob("*.h")),
            PKG.parent / "include" / "mcb200.h", Path(__file__)]


def build_extension(force: bool = False, verbose: bool = False) -> Path:
    newest = max(p.stat().st_mtime for p in _sources())
    if not (force or not LIB.exists() or LIB.stat().st_mtime < newest):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    OBJDIR.mkdir(exist_ok=True)
    extra = ["-Xptxas", "-v"] if verbose else []
    extra += os.environ.get("MCB_NVCC_FLAGS", "").split()     # e.g. -DMCB_COLS_PER_ITER=2 for an experiment

    def compile_unit(unit):
        name, src, defs = unit
        obj = OBJDIR / f"{name}.{os.getpid()}.o"
        subprocess.run([nvcc, *NVCC_FLAGS, *extra, *defs, "-c", "-o", str(obj), str(CSRC / src)], check=True)
        return obj

    with ThreadPoolExecutor(max_workers=len(UNITS)) as pool:
        objs = list(pool.map(compile_unit, UNITS))
    tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
    subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", str(tmp), *map(str, objs)],
                   check=True)
    os.replace(tmp, LIB)
    for o in objs:
        o.unlink(missing_ok=True)
    return LIB


if __name__ == "__main__":
    print(build_extension(force=True, verbose=True))
