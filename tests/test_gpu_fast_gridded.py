"""GPU parity of the approximate fast path (RAD_FLAG_FAST_GRIDDED):
the oracle stays the EXACT sum; the gridded path must meet the same BASELINE.json north_star
tolerances at its default gridding tolerance, and its measured error must fall with the kernel
width the way the spreading kernel promises."""
import numpy as np
import pytest

from paper_2501_03383_b200 import workloads as wl
from tests import _parity as P

pytestmark = pytest.mark.gpu

L = 10e-6
BOX = ((-0.02 * L,) * 3, (1.02 * L,) * 3)


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    import torch
    from paper_2501_03383_b200 import build
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    build.build()


def _fast(w, steps, tol, step_window=None, flags=0, box=BOX, dtype=None, window=None):
    import torch
    from paper_2501_03383_b200 import binding
    lo, hi = step_window or (min(t for t, _ in steps), max(t for t, _ in steps))
    with binding.Detector(w.dirs, w.omega, w.dt, t0=w.t0, scale=1.0, state_dtype=dtype or w.state_dtype,
                          flags=binding.RAD_FLAG_FAST_GRIDDED | flags, window=window,
                          fast=(box[0], box[1], lo, hi, tol)) as det:
        for t, st in steps:
            det.accumulate_step(t, P.to_device(st))
        torch.cuda.synchronize()
        S = det.spectrum()
        A = det.amplitude()
        return S, A, det.kernel_variant


@pytest.mark.parametrize("D,W,dtype", [(6, 96, np.float32), (33, 64, np.float32), (4, 300, np.float64), (1, 8, np.float32)])
def test_fast_gridded_meets_the_exact_tolerances(oracle_mod, D, W, dtype):
    """Default gridding tolerance (1e-6 -> kernel width 8): spectrum AND complex amplitude against
    the exact oracle; late step indices (the time origin of the grid is the window's)."""
    w = wl.Workload("fast", 4000, 4, 1e-17, wl.dirs_fibonacci(max(D, 2))[:D], wl.omega_log(max(W, 2))[:W], dtype,
                    wl.BASE_SEED + 90, "khi")
    steps = [(600 + 3 * t, st) for t, st in w.steps()]
    o = P.run_oracle(oracle_mod, w, steps)
    S, A, variant = _fast(w, steps, 0.0)
    assert variant == "gridded"
    ref = o.spectrum()
    l2, mr = P.assert_parity(S, ref, what=f"fast gridded {D}x{W}")
    for d in range(D):
        P.assert_parity(S[d], ref[d], what=f"fast gridded {D}x{W} dir {d}")
    Aref = o.amplitude()
    assert np.abs(A - Aref).max() <= 2e-5 * np.abs(Aref).max()
    print(f"fast gridded {D}x{W} {np.dtype(dtype).name}: relL2={l2:.2e} maxrel={mr:.2e}")


def test_fast_gridded_error_falls_with_the_kernel_width(oracle_mod):
    """Accuracy vs width: tolerance 1e-3 ... 1e-9 selects widths 4 ... 10.  Error
    measure: |A - A_ref| per bin relative to max(|A_ref| of the bin, rms |A_ref| of its direction) --
    the gridding error of a bin scales with the bin's own amplitude where the sum is coherent and
    with the rms where it is not.  It must stay below ~20x the requested tolerance until it meets
    the fp32 floor that the direct GPU path has too."""
    w = wl.Workload("fastw", 3000, 3, 1e-17, wl.dirs_fibonacci(5), wl.omega_log(128), np.float32,
                    wl.BASE_SEED + 91, "khi")
    steps = list(w.steps())
    Aref = P.run_oracle(oracle_mod, w, steps).amplitude()
    rms = np.sqrt(np.mean(np.abs(Aref) ** 2, axis=(1, 2), keepdims=True))
    den = np.maximum(np.sqrt((np.abs(Aref) ** 2).sum(axis=2, keepdims=True)), rms)

    def err(A):
        return float((np.abs(A - Aref) / den).max())

    _, A_direct, _ = P.run_gpu(w, steps, want_amplitude=True)
    floor = err(A_direct)
    errs = {}
    for tol in (1e-3, 1e-5, 1e-7, 1e-9):
        S, A, _ = _fast(w, steps, tol)
        errs[tol] = err(A)
        assert errs[tol] <= max(20 * tol, 5 * floor), f"tol {tol}: error {errs[tol]:.2e} (direct path {floor:.2e})"
    assert errs[1e-3] > 10 * errs[1e-7]      # the width really matters
    print("fast gridded error vs tolerance:", {k: f"{v:.1e}" for k, v in errs.items()}, f"direct path: {floor:.1e}")


def test_fast_gridded_equals_direct_path_window_reset_and_many_folds(oracle_mod):
    """More accumulate calls than the fold interval (the fp32 delta grid is folded into the fp64
    master every 32 calls), a spatial window, rad_reset, a spectrum between steps (re-evaluation
    after more deposits)."""
    import torch
    from paper_2501_03383_b200 import binding
    w = wl.Workload("fastm", 1500, 70, 1e-17, wl.dirs_fibonacci(3), wl.omega_log(64), np.float32,
                    wl.BASE_SEED + 92, "khi")
    steps = list(w.steps())
    win = ("hamming", (0.1 * L, 0.0, 0.0), (0.8 * L, 0.0, 0.0))
    o = oracle_mod.Oracle(w.dirs, w.omega, w.dt, scale=1.0, window=win)
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, flags=binding.RAD_FLAG_FAST_GRIDDED, window=win,
                          fast=(BOX[0], BOX[1], 0, 69, 1e-6)) as det:
        det.accumulate_step(5, P.to_device(steps[5][1]))
        det.reset()
        assert np.all(det.spectrum() == 0.0)
        for i, (t, st) in enumerate(steps):
            det.accumulate_step(t, P.to_device(st))
            o.accumulate_step(t, *st)
            if i in (0, 40):
                P.assert_parity(det.spectrum(), o.spectrum(), what=f"fast gridded after step {i}")
        P.assert_parity(det.spectrum(), o.spectrum(), what="fast gridded 70 steps")
        assert np.array_equal(det.spectrum(), det.spectrum())        # cached evaluation, non-destructive


def test_fast_gridded_errors():
    from paper_2501_03383_b200 import binding
    w = wl.Workload("faste", 500, 2, 1e-17, wl.dirs_fibonacci(3), wl.omega_log(32), np.float32, wl.BASE_SEED + 93, "khi")
    steps = list(w.steps())
    F = binding.RAD_FLAG_FAST_GRIDDED
    fast = (BOX[0], BOX[1], 0, 1, 1e-6)
    for kw in (dict(n_regions=3), dict(nyquist=0.5), dict(form_factor=("gaussian", (1e-8,) * 3)),
               dict(flags=F | binding.RAD_FLAG_DETERMINISTIC)):
        args = dict(flags=F, fast=fast)
        args.update(kw)
        with pytest.raises(binding.RadError, match="UNSUPPORTED"):
            binding.Detector(w.dirs, w.omega, w.dt, **args)
    with pytest.raises(binding.RadError, match="fast_box"):
        binding.Detector(w.dirs, w.omega, w.dt, flags=F, fast=((0, 0, 0), (1, -1, 1), 0, 1, 0))
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, flags=F, fast=fast) as det:
        with pytest.raises(binding.RadError, match="step_index outside"):
            det.accumulate_step(7, P.to_device(steps[0][1]))
        st = [a.copy() for a in steps[0][1]]
        st[0][17] = 5.0                                   # 5 m away: outside the box
        det.accumulate_step(0, P.to_device(st))
        with pytest.raises(binding.RadError, match="fell outside"):
            det.spectrum()
        import torch
        buf = torch.empty(3, 32, 4, dtype=torch.float64, device="cuda")
        with pytest.raises(binding.RadError, match="UNSUPPORTED"):
            det.export_accumulator(buf)


def test_fast_gridded_host_buffers_and_multi_step_entry(oracle_mod):
    """The other entry points on a fast handle: rad_accumulate_step_host (state in host memory, staged through the
    handle's double buffer) and rad_accumulate_steps (runs as one spreading pass per step); spectrum to pinned host
    memory with RAD_OUT_HOST_ASYNC."""
    import torch
    from paper_2501_03383_b200 import binding
    w = wl.Workload("fasth", 2500, 4, 1e-17, wl.dirs_fibonacci(4), wl.omega_log(80), np.float32, wl.BASE_SEED + 94, "khi")
    steps = list(w.steps())
    ref = P.run_oracle(oracle_mod, w, steps).spectrum()
    fast = (BOX[0], BOX[1], 0, 3, 0.0)
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, flags=binding.RAD_FLAG_FAST_GRIDDED, fast=fast) as det:
        for t, st in steps:
            det.accumulate_step_host(t, st)
        pinned = torch.empty(4, 80, dtype=torch.float64).pin_memory()
        det.spectrum(out=pinned)
        torch.cuda.synchronize()
        P.assert_parity(pinned.numpy(), ref, what="fast gridded, host buffers")
    stacked = [torch.from_numpy(np.stack([st[c] for _, st in steps])).cuda() for c in range(10)]
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, flags=binding.RAD_FLAG_FAST_GRIDDED, fast=fast) as det:
        det.accumulate_steps(0, stacked)
        P.assert_parity(det.spectrum(), ref, what="fast gridded, multi-step entry")
