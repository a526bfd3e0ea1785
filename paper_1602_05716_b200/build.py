"""Builds libmcb200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
from pathlib import Path

PKG = Path(__file__).resolve().parent
SRC = PKG / "csrc" / "mcb200.cu"
LIB = PKG / "libmcb200.so"
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-fmad=false",  # every fused multiply-add in the kernels is written explicitly (reading G11)
    "-shared", "-Xcompiler", "-fPIC",
]


def _sources():
    return [SRC, *sorted((PKG / "csrc").glob("*.cuh")), PKG.parent / "include" / "mcb200.h"]


def build_extension(force: bool = False, verbose: bool = False) -> Path:
    newest = max(p.stat().st_mtime for p in _sources())
    if force or not LIB.exists() or LIB.stat().st_mtime < newest:
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
        cmd = [nvcc, *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", str(tmp), str(SRC)]
        subprocess.run(cmd, check=True)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build_extension(force=True, verbose=True))
