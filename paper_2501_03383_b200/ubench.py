"""ctypes binding of librad_ubench.so (csrc/rad_ubench.cu): the pipe microbenchmarks from which
bench.py derives the MEASURED ALU peaks of its rooflines.  Not part
of the product ABI (include/rad.h); argument marshalling only."""
from __future__ import annotations

import ctypes
from pathlib import Path

LIB_PATH = Path(__file__).resolve().parent / "librad_ubench.so"
_lib = None


def load() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise FileNotFoundError(f"{LIB_PATH} not found: build it with `python -m paper_2501_03383_b200.build`")
        lib = ctypes.CDLL(str(LIB_PATH))
        lib.rad_ubench_kinds.restype = ctypes.c_int
        lib.rad_ubench_name.restype = ctypes.c_char_p
        lib.rad_ubench_name.argtypes = [ctypes.c_int]
        lib.rad_ubench_run.restype = ctypes.c_int
        lib.rad_ubench_run.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                       ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
        _lib = lib
    return _lib


def kinds() -> list[str]:
    lib = load()
    return [lib.rad_ubench_name(k).decode() for k in range(lib.rad_ubench_kinds())]


def run(kind: int, device: int = 0, blocks_per_sm: int = 4, reps: int = 3) -> tuple[float, float]:
    """-> (thread-level results per clk per SM from clock64, 1e9 results/s from CUDA events)."""
    per_clk, gops = ctypes.c_double(), ctypes.c_double()
    rc = load().rad_ubench_run(device, kind, blocks_per_sm, reps, ctypes.byref(per_clk), ctypes.byref(gops))
    if rc != 0:
        raise RuntimeError(f"rad_ubench_run({kind}) failed with {rc}")
    return per_clk.value, gops.value


def run_all(device: int = 0, blocks_per_sm: int = 4, reps: int = 3) -> dict:
    """{name: {"per_clk_sm": ..., "gops": ...}} for every kind."""
    out = {}
    for k, name in enumerate(kinds()):
        per_clk, gops = run(k, device, blocks_per_sm, reps)
        out[name] = {"per_clk_sm": per_clk, "gops": gops}
    return out
