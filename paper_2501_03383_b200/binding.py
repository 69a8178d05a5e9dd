"""Thin ctypes binding of include/rad.h -- argument marshalling only.

Same names as the C ABI (rad_create, rad_accumulate_step, rad_spectrum, ...), plus a small
`Detector` convenience class that owns a handle.  torch is used for device memory and
streams only; every step of the path runs in the CUDA kernels of librad.so.  There is no
CPU fallback: if the library is missing or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes
from pathlib import Path
from typing import Optional, Sequence

import numpy as np

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "librad.so"

RAD_OK, RAD_ERR_INVALID_ARG, RAD_ERR_ALLOC, RAD_ERR_CUDA, RAD_ERR_STATE, RAD_ERR_UNSUPPORTED = range(6)
RAD_F32, RAD_F64 = 0, 1
RAD_FLAG_DETERMINISTIC, RAD_FLAG_FORCE_GENERAL, RAD_FLAG_OVERLAP_STEPS, RAD_FLAG_FAST_GRIDDED, RAD_FLAG_PRECISE = 1, 2, 4, 8, 16
RAD_OUT_HOST, RAD_OUT_DEVICE, RAD_OUT_HOST_ASYNC = 0, 1, 2
RAD_WINDOW_NONE, RAD_WINDOW_TRIANGLE, RAD_WINDOW_HAMMING = 0, 1, 2
WINDOW_TYPES = {"none": RAD_WINDOW_NONE, "triangle": RAD_WINDOW_TRIANGLE, "hamming": RAD_WINDOW_HAMMING}
RAD_FF_NONE, RAD_FF_GAUSSIAN, RAD_FF_CIC, RAD_FF_INCOHERENT = 0, 1, 2, 3
FORM_FACTOR_TYPES = {"none": RAD_FF_NONE, "gaussian": RAD_FF_GAUSSIAN, "cic": RAD_FF_CIC,
                     "incoherent": RAD_FF_INCOHERENT}

ABI_SYMBOLS = (
    "rad_create", "rad_accumulate_step", "rad_accumulate_steps", "rad_accumulate_steps_regions",
    "rad_accumulate_step_host",
    "rad_accumulate_step_regions", "rad_accumulate_step_regions_host", "rad_spectrum",
    "rad_spectrum_total", "rad_amplitude", "rad_add_amplitude", "rad_export_accumulator",
    "rad_import_accumulator", "rad_spectrum_of", "rad_reset", "rad_destroy", "rad_launch_count",
    "rad_kernel_variant", "rad_status_string", "rad_last_error", "rad_version",
    "rad_spectrum_static", "rad_static_last_error",
)
RAD_STATIC_MAX_BINS = 65536


class rad_config(ctypes.Structure):
    _fields_ = [
        ("struct_size", ctypes.c_uint32), ("device", ctypes.c_int32),
        ("n_dir", ctypes.c_int32), ("n_omega", ctypes.c_int32),
        ("dirs", ctypes.c_void_p), ("omega", ctypes.c_void_p),
        ("dt", ctypes.c_double), ("t0", ctypes.c_double), ("scale", ctypes.c_double),
        ("state_dtype", ctypes.c_int32), ("flags", ctypes.c_uint32),
        ("n_regions", ctypes.c_int32), ("window_type", ctypes.c_int32),
        ("window_origin", ctypes.c_double * 3), ("window_extent", ctypes.c_double * 3),
        ("nyquist_factor", ctypes.c_double),
        ("form_factor_type", ctypes.c_int32), ("reserved0", ctypes.c_int32),
        ("form_factor_size", ctypes.c_double * 3),
        ("fast_box_min", ctypes.c_double * 3), ("fast_box_max", ctypes.c_double * 3),
        ("fast_step_min", ctypes.c_int64), ("fast_step_max", ctypes.c_int64),
        ("fast_tolerance", ctypes.c_double),
    ]


class RadError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{status_string(status)}: {msg}")
        self.status = status


_lib = None


def load(path: Optional[Path] = None) -> ctypes.CDLL:
    """Load librad.so (built in-tree by paper_2501_03383_b200.build).  Fails loudly."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = Path(path) if path else LIB_PATH
    if not p.exists():
        raise FileNotFoundError(
            f"{p} not found: build it with `python -m paper_2501_03383_b200.build` "
            "(there is no CPU fallback)")
    lib = ctypes.CDLL(str(p))
    vp, i64, dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_double
    lib.rad_create.restype = ctypes.c_int
    lib.rad_create.argtypes = [ctypes.POINTER(rad_config), ctypes.POINTER(vp)]
    for name in ("rad_accumulate_step", "rad_accumulate_step_host"):
        f = getattr(lib, name)
        f.restype = ctypes.c_int
        f.argtypes = [vp, i64, i64] + [vp] * 10 + [vp]
    lib.rad_accumulate_steps.restype = ctypes.c_int
    lib.rad_accumulate_steps.argtypes = [vp, i64, ctypes.c_int32, i64, i64] + [vp] * 10 + [vp]
    lib.rad_accumulate_steps_regions.restype = ctypes.c_int
    lib.rad_accumulate_steps_regions.argtypes = [vp, i64, ctypes.c_int32, i64, ctypes.c_int32, vp] + [vp] * 10 + [vp]
    for name in ("rad_accumulate_step_regions", "rad_accumulate_step_regions_host"):
        f = getattr(lib, name)
        f.restype = ctypes.c_int
        f.argtypes = [vp, i64, ctypes.c_int32, vp] + [vp] * 10 + [vp]
    for name in ("rad_spectrum", "rad_spectrum_total", "rad_amplitude"):
        f = getattr(lib, name)
        f.restype = ctypes.c_int
        f.argtypes = [vp, vp, ctypes.c_int, vp]
    lib.rad_add_amplitude.restype = ctypes.c_int
    lib.rad_add_amplitude.argtypes = [vp, vp, vp]
    lib.rad_reset.restype = ctypes.c_int
    lib.rad_reset.argtypes = [vp, vp]
    for name in ("rad_export_accumulator", "rad_import_accumulator"):
        f = getattr(lib, name)
        f.restype = ctypes.c_int
        f.argtypes = [vp, vp, vp]
    lib.rad_spectrum_of.restype = ctypes.c_int
    lib.rad_spectrum_of.argtypes = [vp, vp, vp, ctypes.c_int, vp]
    lib.rad_destroy.restype = None
    lib.rad_destroy.argtypes = [vp]
    lib.rad_launch_count.restype = i64
    lib.rad_launch_count.argtypes = [vp]
    for name in ("rad_kernel_variant", "rad_last_error"):
        f = getattr(lib, name)
        f.restype = ctypes.c_char_p
        f.argtypes = [vp]
    lib.rad_status_string.restype = ctypes.c_char_p
    lib.rad_status_string.argtypes = [ctypes.c_int]
    lib.rad_version.restype = ctypes.c_char_p
    lib.rad_version.argtypes = []
    lib.rad_spectrum_static.restype = ctypes.c_int
    lib.rad_spectrum_static.argtypes = ([ctypes.c_int32, vp, ctypes.c_int32, vp, dbl, dbl, dbl, ctypes.c_int32, i64,
                                         ctypes.c_int32, i64, i64] + [vp] * 10 + [vp, vp])
    lib.rad_static_last_error.restype = ctypes.c_char_p
    lib.rad_static_last_error.argtypes = []
    if path is None:
        _lib = lib
    return lib


def status_string(status: int) -> str:
    return load().rad_status_string(int(status)).decode()


def rad_version() -> str:
    return load().rad_version().decode()


def _check(status: int, handle) -> None:
    if status != RAD_OK:
        raise RadError(status, (load().rad_last_error(handle) or b"").decode())


# ------------------------------------------------------------------ ABI-named functions
def rad_create(dirs, omega, dt: float, t0: float = 0.0, scale: float = 0.0,
               state_dtype: int = RAD_F32, flags: int = 0, device: int = 0, n_regions: int = 0,
               window=None, nyquist: float = 0.0, form_factor=None, fast=None) -> int:
    """-> opaque handle (int).  dirs [D,3], omega [W]: HOST fp64 (copied by the library).
    window: None or (type name | code, origin[3], extent[3]).
    form_factor: None or (type name | code, size[3] in metres).
    fast (with RAD_FLAG_FAST_GRIDDED): (box_min[3], box_max[3], step_min, step_max, tolerance)."""
    dirs = np.ascontiguousarray(dirs, dtype=np.float64).reshape(-1, 3)
    omega = np.ascontiguousarray(omega, dtype=np.float64).reshape(-1)
    cfg = rad_config(ctypes.sizeof(rad_config), device, dirs.shape[0], omega.shape[0],
                     dirs.ctypes.data, omega.ctypes.data, dt, t0, scale, state_dtype, flags,
                     n_regions, 0)
    cfg.nyquist_factor = float(nyquist)
    if window is not None:
        kind, origin, extent = window
        cfg.window_type = WINDOW_TYPES[kind] if isinstance(kind, str) else int(kind)
        cfg.window_origin = (ctypes.c_double * 3)(*[float(x) for x in origin])
        cfg.window_extent = (ctypes.c_double * 3)(*[float(x) for x in extent])
    if form_factor is not None:
        kind, size = form_factor
        cfg.form_factor_type = FORM_FACTOR_TYPES[kind] if isinstance(kind, str) else int(kind)
        cfg.form_factor_size = (ctypes.c_double * 3)(*[float(x) for x in size])
    if fast is not None:
        bmin, bmax, smin, smax, tol = fast
        cfg.fast_box_min = (ctypes.c_double * 3)(*[float(x) for x in bmin])
        cfg.fast_box_max = (ctypes.c_double * 3)(*[float(x) for x in bmax])
        cfg.fast_step_min, cfg.fast_step_max, cfg.fast_tolerance = int(smin), int(smax), float(tol)
    h = ctypes.c_void_p()
    _check(load().rad_create(ctypes.byref(cfg), ctypes.byref(h)), None)
    return h.value


def rad_accumulate_step(handle: int, step_index: int, n_particles: int, state_ptrs: Sequence[int],
                        stream: int = 0) -> None:
    """state_ptrs: 10 DEVICE pointers (rx ry rz bx by bz bdx bdy bdz w)."""
    _check(load().rad_accumulate_step(handle, step_index, n_particles, *state_ptrs, stream), handle)


def rad_accumulate_steps(handle: int, first_step_index: int, n_steps: int, n_particles: int,
                         step_stride: int, state_ptrs: Sequence[int], stream: int = 0) -> None:
    """state_ptrs: 10 DEVICE pointers to [n_steps][step_stride] arrays (first n_particles of each row)."""
    _check(load().rad_accumulate_steps(handle, first_step_index, n_steps, n_particles, step_stride,
                                       *state_ptrs, stream), handle)


def rad_accumulate_steps_regions(handle: int, first_step_index: int, n_steps: int, step_stride: int,
                                 region_offsets: np.ndarray, state_ptrs: Sequence[int], stream: int = 0) -> None:
    """region_offsets: HOST int64 [R+1], the same for every step; state_ptrs: 10 DEVICE pointers."""
    off = np.ascontiguousarray(region_offsets, dtype=np.int64)
    _check(load().rad_accumulate_steps_regions(handle, first_step_index, n_steps, step_stride,
                                               off.shape[0] - 1, off.ctypes.data, *state_ptrs, stream), handle)


def rad_accumulate_step_host(handle: int, step_index: int, n_particles: int,
                             state_ptrs: Sequence[int], stream: int = 0) -> None:
    """state_ptrs: 10 HOST pointers."""
    _check(load().rad_accumulate_step_host(handle, step_index, n_particles, *state_ptrs, stream), handle)


def rad_accumulate_step_regions(handle: int, step_index: int, region_offsets: np.ndarray,
                                state_ptrs: Sequence[int], stream: int = 0) -> None:
    """region_offsets: HOST int64 [R+1]; state_ptrs: 10 DEVICE pointers."""
    off = np.ascontiguousarray(region_offsets, dtype=np.int64)
    _check(load().rad_accumulate_step_regions(handle, step_index, off.shape[0] - 1, off.ctypes.data,
                                              *state_ptrs, stream), handle)


def rad_accumulate_step_regions_host(handle: int, step_index: int, region_offsets: np.ndarray,
                                     state_ptrs: Sequence[int], stream: int = 0) -> None:
    """region_offsets: HOST int64 [R+1]; state_ptrs: 10 HOST pointers."""
    off = np.ascontiguousarray(region_offsets, dtype=np.int64)
    _check(load().rad_accumulate_step_regions_host(handle, step_index, off.shape[0] - 1, off.ctypes.data,
                                                   *state_ptrs, stream), handle)


def rad_spectrum(handle: int, out_ptr: int, out_on_device: int, stream: int = 0) -> None:
    """out_on_device: RAD_OUT_HOST (False), RAD_OUT_DEVICE (True) or RAD_OUT_HOST_ASYNC."""
    _check(load().rad_spectrum(handle, out_ptr, int(out_on_device), stream), handle)


def rad_spectrum_total(handle: int, out_ptr: int, out_on_device: bool, stream: int = 0) -> None:
    _check(load().rad_spectrum_total(handle, out_ptr, int(out_on_device), stream), handle)


def rad_amplitude(handle: int, out_ptr: int, out_on_device: bool, stream: int = 0) -> None:
    _check(load().rad_amplitude(handle, out_ptr, int(out_on_device), stream), handle)


def rad_add_amplitude(handle: int, amp_device_ptr: int, stream: int = 0) -> None:
    _check(load().rad_add_amplitude(handle, amp_device_ptr, stream), handle)


def rad_export_accumulator(handle: int, out_device_ptr: int, stream: int = 0) -> None:
    """out: DEVICE [(R,) D, W, 4] fp64 = (Re A1, Im A1, Re A2, Im A2) on the handle's transverse basis."""
    _check(load().rad_export_accumulator(handle, out_device_ptr, stream), handle)


def rad_import_accumulator(handle: int, amp4_device_ptr: int, stream: int = 0) -> None:
    _check(load().rad_import_accumulator(handle, amp4_device_ptr, stream), handle)


def rad_spectrum_of(handle: int, amp4_device_ptr: int, out_ptr: int, out_on_device: int, stream: int = 0) -> None:
    _check(load().rad_spectrum_of(handle, amp4_device_ptr, out_ptr, int(out_on_device), stream), handle)


def rad_reset(handle: int, stream: int = 0) -> None:
    _check(load().rad_reset(handle, stream), handle)


def rad_destroy(handle: Optional[int]) -> None:
    load().rad_destroy(handle)


def rad_launch_count(handle: int) -> int:
    return int(load().rad_launch_count(handle))


def rad_kernel_variant(handle: int) -> str:
    return load().rad_kernel_variant(handle).decode()


def rad_spectrum_static(n_dir: int, dirs_device_ptr: int, n_omega: int, omega_device_ptr: int, dt: float, t0: float,
                        scale: float, state_dtype: int, first_step_index: int, n_steps: int, n_particles: int,
                        step_stride: int, state_ptrs: Sequence[int], out_device_ptr: int, stream: int = 0) -> None:
    """The allocation-free one-call detector (include/rad.h): every pointer DEVICE; out [n_dir][n_omega] fp64."""
    lib = load()
    st = lib.rad_spectrum_static(n_dir, dirs_device_ptr, n_omega, omega_device_ptr, dt, t0, scale, state_dtype,
                                 first_step_index, n_steps, n_particles, step_stride, *state_ptrs, out_device_ptr, stream)
    if st != RAD_OK:
        raise RadError(st, (lib.rad_static_last_error() or b"").decode())


# ------------------------------------------------------------------ convenience wrapper
class Detector:
    """Owns one rad_handle.  State may be torch CUDA tensors (device path) or numpy /
    pinned torch CPU tensors (host path, copies inside the library)."""

    def __init__(self, dirs, omega, dt, t0=0.0, scale=0.0, state_dtype=np.float32, flags=0, device=0,
                 n_regions=0, window=None, nyquist=0.0, form_factor=None, fast=None):
        self.D = int(np.asarray(dirs).reshape(-1, 3).shape[0])
        self.W = int(np.asarray(omega).reshape(-1).shape[0])
        self.R = max(1, int(n_regions))
        self.np_dtype = np.dtype(state_dtype)
        code = {np.dtype(np.float32): RAD_F32, np.dtype(np.float64): RAD_F64}[self.np_dtype]
        self.device = device
        self.handle = rad_create(dirs, omega, dt, t0, scale, code, flags, device, n_regions, window, nyquist,
                                 form_factor, fast)

    def _shape(self, *tail):
        return ((self.R,) if self.R > 1 else ()) + (self.D, self.W) + tail

    # -- helpers
    def _stream(self) -> int:
        import torch
        return int(torch.cuda.current_stream(self.device).cuda_stream)

    def _ptrs(self, state, want_cuda: bool):
        import torch
        if len(state) != 10:
            raise ValueError("state must be 10 arrays: rx ry rz bx by bz bdx bdy bdz w")
        n, ptrs = None, []
        for a in state:
            if isinstance(a, torch.Tensor):
                if a.is_cuda != want_cuda or not a.is_contiguous() or a.dim() != 1:
                    raise ValueError("state tensors must be 1-D contiguous and on the expected device")
                if a.element_size() != self.np_dtype.itemsize or not a.dtype.is_floating_point:
                    raise TypeError("state dtype does not match the detector's state_dtype")
                ptrs.append(a.data_ptr()); m = a.numel()
            else:
                if want_cuda or a.dtype != self.np_dtype or not a.flags.c_contiguous or a.ndim != 1:
                    raise ValueError("host state must be 1-D contiguous numpy arrays of state_dtype")
                ptrs.append(a.ctypes.data); m = a.shape[0]
            if n is not None and m != n:
                raise ValueError("state arrays differ in length")
            n = m
        return n, ptrs

    # -- ABI calls
    def accumulate_step(self, step_index: int, state) -> None:
        n, ptrs = self._ptrs(state, want_cuda=True)
        rad_accumulate_step(self.handle, step_index, n, ptrs, self._stream())

    def accumulate_steps(self, first_step_index: int, state, region_offsets=None) -> None:
        """state: 10 torch CUDA tensors [n_steps, n_particles] (contiguous): all steps in one launch.
        region_offsets (per-region handles): HOST int64 [R+1], the same for every step."""
        import torch
        if len(state) != 10:
            raise ValueError("state must be 10 arrays: rx ry rz bx by bz bdx bdy bdz w")
        shp = tuple(state[0].shape)
        for a in state:
            if not (isinstance(a, torch.Tensor) and a.is_cuda and a.dim() == 2 and a.is_contiguous()
                    and tuple(a.shape) == shp and a.element_size() == self.np_dtype.itemsize):
                raise ValueError("state tensors must be contiguous CUDA [n_steps, n_particles] of state_dtype")
        ptrs = [a.data_ptr() for a in state]
        if region_offsets is not None:
            if int(region_offsets[-1]) > shp[1]:
                raise ValueError("region_offsets[-1] exceeds the row length")
            rad_accumulate_steps_regions(self.handle, first_step_index, shp[0], shp[1], region_offsets, ptrs,
                                         self._stream())
        else:
            rad_accumulate_steps(self.handle, first_step_index, shp[0], shp[1], shp[1], ptrs, self._stream())

    def accumulate_step_host(self, step_index: int, state) -> None:
        n, ptrs = self._ptrs(state, want_cuda=False)
        rad_accumulate_step_host(self.handle, step_index, n, ptrs, self._stream())

    def accumulate_step_regions(self, step_index: int, region_offsets, state) -> None:
        """Per-region detectors: state sorted by region, region r = [offsets[r], offsets[r+1])."""
        n, ptrs = self._ptrs(state, want_cuda=True)
        if int(region_offsets[-1]) > n:
            raise ValueError("region_offsets[-1] exceeds the state length")
        rad_accumulate_step_regions(self.handle, step_index, region_offsets, ptrs, self._stream())

    def accumulate_step_regions_host(self, step_index: int, region_offsets, state) -> None:
        n, ptrs = self._ptrs(state, want_cuda=False)
        if int(region_offsets[-1]) > n:
            raise ValueError("region_offsets[-1] exceeds the state length")
        rad_accumulate_step_regions_host(self.handle, step_index, region_offsets, ptrs, self._stream())

    def spectrum(self, out=None):
        """out: optional torch fp64 tensor [(R,) D, W]: CUDA (asynchronous) or pinned CPU
        (RAD_OUT_HOST_ASYNC: valid once the current stream has passed the call); default -> numpy."""
        if out is not None:
            mode = RAD_OUT_DEVICE if out.is_cuda else RAD_OUT_HOST_ASYNC
            rad_spectrum(self.handle, out.data_ptr(), mode, self._stream())
            return out
        res = np.empty(self._shape(), dtype=np.float64)
        rad_spectrum(self.handle, res.ctypes.data, False, self._stream())
        return res

    def spectrum_total(self, out=None):
        """[D, W]: scale * |sum over regions of A_r|^2."""
        if out is not None:
            rad_spectrum_total(self.handle, out.data_ptr(), True, self._stream())
            return out
        res = np.empty((self.D, self.W), dtype=np.float64)
        rad_spectrum_total(self.handle, res.ctypes.data, False, self._stream())
        return res

    def amplitude(self, out=None):
        """Complex amplitude; default -> numpy complex128 [(R,) D, W, 3]."""
        if out is not None:
            rad_amplitude(self.handle, out.data_ptr(), True, self._stream())
            return out
        res = np.empty(self._shape(3, 2), dtype=np.float64)
        rad_amplitude(self.handle, res.ctypes.data, False, self._stream())
        return res[..., 0] + 1j * res[..., 1]

    def add_amplitude(self, amp) -> None:
        rad_add_amplitude(self.handle, amp.data_ptr(), self._stream())

    def export_accumulator(self, out) -> None:
        """out: torch CUDA fp64 tensor [(R,) D, W, 4] (contiguous)."""
        rad_export_accumulator(self.handle, out.data_ptr(), self._stream())

    def import_accumulator(self, amp4) -> None:
        rad_import_accumulator(self.handle, amp4.data_ptr(), self._stream())

    def spectrum_of(self, amp4, out=None):
        """|A|^2 of an exported / all-reduced amplitude buffer; out as in spectrum()."""
        if out is not None:
            mode = RAD_OUT_DEVICE if out.is_cuda else RAD_OUT_HOST_ASYNC
            rad_spectrum_of(self.handle, amp4.data_ptr(), out.data_ptr(), mode, self._stream())
            return out
        res = np.empty(self._shape(), dtype=np.float64)
        rad_spectrum_of(self.handle, amp4.data_ptr(), res.ctypes.data, RAD_OUT_HOST, self._stream())
        return res

    def reset(self) -> None:
        rad_reset(self.handle, self._stream())

    @property
    def launch_count(self) -> int:
        return rad_launch_count(self.handle)

    @property
    def kernel_variant(self) -> str:
        return rad_kernel_variant(self.handle)

    def close(self) -> None:
        if getattr(self, "handle", None):
            rad_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()
