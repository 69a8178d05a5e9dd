"""Builds paper_2501_03383_b200/librad.so (the C-ABI library of include/rad.h) with nvcc
for sm_100a, and librad_ubench.so (the pipe microbenchmarks bench.py derives its measured ALU
peaks from; not part of the ABI).  In-tree, so that the .so files travel to the GPU box with the
repo snapshot.

    python -m paper_2501_03383_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
ROOT = PKG.parent
CSRC = PKG / "csrc"
LIB = PKG / "librad.so"
UBENCH_LIB = PKG / "librad_ubench.so"
SOURCES = ["rad_api.cu", "rad_kernels.cu", "rad_stream.cu", "rad_finalize.cu", "rad_gridded.cu", "rad_static.cu"]
UBENCH_SOURCES = ["rad_ubench.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "--use_fast_math", "-Xcompiler", "-fPIC,-fvisibility=hidden,-O2", "-shared",
              "-cudart", "static"]


def nvcc() -> str:
    cand = os.environ.get("NVCC") or "/usr/local/cuda/bin/nvcc"
    return cand if Path(cand).exists() else "nvcc"


def stale(lib: Path = LIB, sources=None) -> bool:
    if not lib.exists():
        return True
    t = lib.stat().st_mtime
    deps = ([CSRC / s for s in sources] if sources else list(CSRC.glob("*"))) + [ROOT / "include" / "rad.h",
                                                                                 Path(__file__)]
    return any(d.stat().st_mtime > t for d in deps)


def _compile(lib: Path, sources, verbose: bool) -> Path:
    tmp = lib.with_suffix(f".tmp{os.getpid()}.so")
    cmd = [nvcc(), *NVCC_FLAGS, "-I", str(ROOT / "include"), "-I", str(CSRC)]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [str(CSRC / s) for s in sources] + ["-o", str(tmp)]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError(f"nvcc failed building {lib.name}")
    os.replace(tmp, lib)
    return lib


def build(force: bool = False, verbose: bool = False) -> Path:
    if force or stale(UBENCH_LIB, UBENCH_SOURCES):
        _compile(UBENCH_LIB, UBENCH_SOURCES, verbose)
    if force or stale():
        _compile(LIB, SOURCES, verbose)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
