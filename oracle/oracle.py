"""ctypes wrapper around oracle/rad_oracle.c -- the fp64 CPU oracle.

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  The product package never imports this module.
It holds no arithmetic of its own: every number comes from rad_oracle.c, which follows
BASELINE.json north_star / PAPER.md lines 74, 79-81, 142.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "rad_oracle.c"
_LIB = _HERE / "librad_oracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile rad_oracle.c with gcc (-O2, OpenMP, no fast-math)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-fno-fast-math",
               "-ffp-contract=off", str(_SRC), "-o", str(tmp), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(str(_LIB))
        lib.oracle_default_scale.restype = ctypes.c_double
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_accumulate_step.restype = ctypes.c_int
        lib.oracle_accumulate_step.argtypes = (
            [ctypes.c_int, ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p,
             ctypes.c_double, ctypes.c_double, ctypes.c_longlong, ctypes.c_longlong, ctypes.c_int]
            + [ctypes.c_void_p] * 10
            + [ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p])
        lib.oracle_accumulate_step_w.restype = ctypes.c_int
        lib.oracle_accumulate_step_w.argtypes = (lib.oracle_accumulate_step.argtypes
                                                 + [ctypes.c_int, ctypes.c_void_p, ctypes.c_double])
        lib.oracle_accumulate_step_ff.restype = ctypes.c_int
        lib.oracle_accumulate_step_ff.argtypes = (lib.oracle_accumulate_step_w.argtypes
                                                  + [ctypes.c_int, ctypes.c_void_p])
        lib.oracle_accumulate_step_regions.restype = ctypes.c_int
        lib.oracle_accumulate_step_regions.argtypes = (
            [ctypes.c_int, ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p,
             ctypes.c_double, ctypes.c_double, ctypes.c_longlong, ctypes.c_longlong,
             ctypes.c_void_p, ctypes.c_int]
            + [ctypes.c_void_p] * 10
            + [ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p])
        lib.oracle_accumulate_step_regions_w.restype = ctypes.c_int
        lib.oracle_accumulate_step_regions_w.argtypes = (lib.oracle_accumulate_step_regions.argtypes
                                                         + [ctypes.c_int, ctypes.c_void_p, ctypes.c_double])
        lib.oracle_accumulate_step_regions_ff.restype = ctypes.c_int
        lib.oracle_accumulate_step_regions_ff.argtypes = (lib.oracle_accumulate_step_regions_w.argtypes
                                                          + [ctypes.c_int, ctypes.c_void_p])
        lib.oracle_spectrum_total.restype = ctypes.c_int
        lib.oracle_spectrum_total.argtypes = [ctypes.c_longlong, ctypes.c_longlong, ctypes.c_void_p,
                                              ctypes.c_double, ctypes.c_void_p]
        lib.oracle_spectrum.restype = ctypes.c_int
        lib.oracle_spectrum.argtypes = [ctypes.c_longlong, ctypes.c_void_p, ctypes.c_double,
                                        ctypes.c_void_p]
        _lib = lib
    return _lib


def default_scale() -> float:
    return float(_load().oracle_default_scale())


def num_threads() -> int:
    return int(_load().oracle_num_threads())


WINDOW_TYPES = {"none": 0, "triangle": 1, "hamming": 2}


def _window_args(window):
    """window = None or (type name, origin[3], extent[3]) -> (type code, fp64 array of 6 or None)."""
    if window is None:
        return 0, None
    name, origin, extent = window
    return WINDOW_TYPES[name], np.ascontiguousarray(list(origin) + list(extent), dtype=np.float64)


FORM_FACTOR_TYPES = {"none": 0, "gaussian": 1, "cic": 2, "incoherent": 3}


def _form_factor_args(form_factor):
    """form_factor = None or (type name, size[3] in metres) -> (type code, fp64 array of 3)."""
    if form_factor is None:
        return 0, np.zeros(3)
    name, size = form_factor
    return FORM_FACTOR_TYPES[name], np.ascontiguousarray(list(size), dtype=np.float64)


class Oracle:
    """Same call sequence as the C ABI (create / accumulate_step / spectrum / amplitude).

    dirs [D,3] and omega [W] are fp64 host arrays.  ``bins`` (optional flat indices
    dir*W + j) restricts the computation to a subset of bins; other bins stay zero.
    """

    def __init__(self, dirs, omega, dt, t0=0.0, scale=0.0, bins=None, window=None, nyquist=0.0,
                 form_factor=None):
        self.nyquist = float(nyquist)
        self.ff_type, self.ff_size = _form_factor_args(form_factor)
        self.dirs = np.ascontiguousarray(dirs, dtype=np.float64).reshape(-1, 3)
        self.omega = np.ascontiguousarray(omega, dtype=np.float64).reshape(-1)
        self.dt, self.t0, self.scale = float(dt), float(t0), float(scale)
        self.D, self.W = self.dirs.shape[0], self.omega.shape[0]
        self.bins = None if bins is None else np.ascontiguousarray(bins, dtype=np.int64)
        self.A = np.zeros((self.D, self.W, 3, 2), dtype=np.float64)
        self.win_type, self.win = _window_args(window)

    def reset(self):
        self.A[...] = 0.0

    def accumulate_step(self, step_index, rx, ry, rz, bx, by, bz, bdx, bdy, bdz, w):
        arrs = [rx, ry, rz, bx, by, bz, bdx, bdy, bdz, w]
        dt0 = np.asarray(arrs[0]).dtype
        if dt0 not in (np.dtype(np.float32), np.dtype(np.float64)):
            raise TypeError("state must be float32 or float64")
        arrs = [np.ascontiguousarray(a, dtype=dt0) for a in arrs]
        n = arrs[0].shape[0]
        if any(a.shape != (n,) for a in arrs):
            raise ValueError("state arrays must be 1-D and of equal length")
        nb = 0 if self.bins is None else self.bins.shape[0]
        bp = None if self.bins is None else self.bins.ctypes.data
        rc = _load().oracle_accumulate_step_ff(
            self.D, self.dirs.ctypes.data, self.W, self.omega.ctypes.data, self.dt, self.t0,
            int(step_index), n, int(dt0 == np.dtype(np.float32)),
            *[a.ctypes.data for a in arrs], nb, bp, self.A.ctypes.data,
            self.win_type, None if self.win is None else self.win.ctypes.data, self.nyquist,
            self.ff_type, self.ff_size.ctypes.data)
        if rc != 0:
            raise ValueError("oracle_accumulate_step: bad argument")

    def amplitude(self):
        """Complex amplitude [D, W, 3] (complex128)."""
        return self.A[..., 0] + 1j * self.A[..., 1]

    def spectrum(self):
        S = np.empty((self.D, self.W), dtype=np.float64)
        rc = _load().oracle_spectrum(self.D * self.W, self.A.ctypes.data, self.scale, S.ctypes.data)
        if rc != 0:
            raise ValueError("oracle_spectrum: bad argument")
        return S


class RegionOracle:
    """Per-region (sub-volume) detectors: A[r] is the oracle sum over the particles of region r
    only.  Particles are sorted by region; ``offsets`` [R+1] (non-decreasing) are passed with
    every step.  Same (optional) bin subset in every region."""

    def __init__(self, n_regions, dirs, omega, dt, t0=0.0, scale=0.0, bins=None, window=None, nyquist=0.0,
                 form_factor=None):
        self.win_type, self.win = _window_args(window)
        self.ff_type, self.ff_size = _form_factor_args(form_factor)
        self.nyquist = float(nyquist)
        self.dirs = np.ascontiguousarray(dirs, dtype=np.float64).reshape(-1, 3)
        self.omega = np.ascontiguousarray(omega, dtype=np.float64).reshape(-1)
        self.dt, self.t0, self.scale = float(dt), float(t0), float(scale)
        self.R, self.D, self.W = int(n_regions), self.dirs.shape[0], self.omega.shape[0]
        self.bins = None if bins is None else np.ascontiguousarray(bins, dtype=np.int64)
        self.A = np.zeros((self.R, self.D, self.W, 3, 2), dtype=np.float64)

    def reset(self):
        self.A[...] = 0.0

    def accumulate_step(self, step_index, offsets, rx, ry, rz, bx, by, bz, bdx, bdy, bdz, w):
        offsets = np.ascontiguousarray(offsets, dtype=np.int64)
        if offsets.shape != (self.R + 1,):
            raise ValueError("offsets must have n_regions + 1 entries")
        arrs = [rx, ry, rz, bx, by, bz, bdx, bdy, bdz, w]
        dt0 = np.asarray(arrs[0]).dtype
        if dt0 not in (np.dtype(np.float32), np.dtype(np.float64)):
            raise TypeError("state must be float32 or float64")
        arrs = [np.ascontiguousarray(a, dtype=dt0) for a in arrs]
        n = arrs[0].shape[0]
        if any(a.shape != (n,) for a in arrs) or offsets[-1] > n:
            raise ValueError("state arrays must be 1-D, of equal length >= offsets[-1]")
        nb = 0 if self.bins is None else self.bins.shape[0]
        bp = None if self.bins is None else self.bins.ctypes.data
        rc = _load().oracle_accumulate_step_regions_ff(
            self.D, self.dirs.ctypes.data, self.W, self.omega.ctypes.data, self.dt, self.t0,
            int(step_index), self.R, offsets.ctypes.data, int(dt0 == np.dtype(np.float32)),
            *[a.ctypes.data for a in arrs], nb, bp, self.A.ctypes.data,
            self.win_type, None if self.win is None else self.win.ctypes.data, self.nyquist,
            self.ff_type, self.ff_size.ctypes.data)
        if rc != 0:
            raise ValueError("oracle_accumulate_step_regions: bad argument")

    def amplitude(self):
        """Complex amplitude [R, D, W, 3] (complex128)."""
        return self.A[..., 0] + 1j * self.A[..., 1]

    def spectrum(self):
        """[R, D, W]: every region's own |A_r|^2."""
        S = np.empty((self.R, self.D, self.W), dtype=np.float64)
        rc = _load().oracle_spectrum(self.R * self.D * self.W, self.A.ctypes.data, self.scale,
                                     S.ctypes.data)
        if rc != 0:
            raise ValueError("oracle_spectrum: bad argument")
        return S

    def spectrum_total(self):
        """[D, W]: |sum_r A_r|^2 -- amplitudes, not intensities, add up."""
        S = np.empty((self.D, self.W), dtype=np.float64)
        rc = _load().oracle_spectrum_total(self.R, self.D * self.W, self.A.ctypes.data, self.scale, S.ctypes.data)
        if rc != 0:
            raise ValueError("oracle_spectrum_total: bad argument")
        return S
