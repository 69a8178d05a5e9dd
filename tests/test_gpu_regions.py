"""GPU parity of the per-region (sub-volume) detectors:
rad_accumulate_step_regions through the C ABI vs oracle.RegionOracle, element by element,
same seeded inputs, BASELINE.json north_star tolerances applied to every region's spectrum."""
import numpy as np
import pytest

from paper_2501_03383_b200 import workloads as wl
from tests import _parity as P

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    import torch
    from paper_2501_03383_b200 import build
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    build.build()


def _oracle(oracle_mod, w, R, off, steps, bins=None):
    o = oracle_mod.RegionOracle(R, w.dirs, w.omega, w.dt, t0=w.t0, scale=1.0, bins=bins)
    for t, st in steps:
        o.accumulate_step(t, off, *st)
    return o


def _gpu(w, R, off, steps, flags=0, host=False):
    import torch
    from paper_2501_03383_b200 import binding
    with binding.Detector(w.dirs, w.omega, w.dt, t0=w.t0, scale=1.0, state_dtype=w.state_dtype,
                          flags=flags, n_regions=R) as det:
        for t, st in steps:
            if host:
                det.accumulate_step_regions_host(t, off, st)
            else:
                det.accumulate_step_regions(t, off, P.to_device(st))
        torch.cuda.synchronize()
        return det.spectrum(), det.spectrum_total(), det.amplitude(), det.kernel_variant


def _assert_regions(S, Sref, what):
    worst = (0.0, 0.0)
    for r in range(Sref.shape[0]):
        if Sref[r].max() == 0.0:
            assert np.all(S[r] == 0.0), f"{what}: empty region {r} must be exactly zero"
            continue
        l2, mr = P.assert_parity(S[r], Sref[r], what=f"{what} region {r}")
        worst = (max(worst[0], l2), max(worst[1], mr))
    return worst


@pytest.mark.parametrize("D,W,dtype,uniform", [(1, 512, np.float32, False), (3, 100, np.float32, False),
                                                (4, 64, np.float64, False), (2, 96, np.float32, True)])
def test_regions_ragged_sizes_all_bins(oracle_mod, D, W, dtype, uniform):
    """Region sizes span empty, 1, a ragged batch tail, several chunks; all bins compared."""
    omega = np.linspace(2e14, 5e16, W) if uniform else wl.omega_log(W)
    w = wl.Workload("reg", 0, 3, 1e-17, wl.dirs_fibonacci(D) if D > 1 else np.array([[1.0, 0.0, 0.0]]),
                    omega, dtype, wl.BASE_SEED + 30, "khi")
    sizes = [700, 0, 1, 33, 1500, 0, 64, 257]
    off = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    w.n_particles = int(off[-1])
    steps = [(t * 37, st) for t, st in w.steps(n_steps=3)]
    S, Stot, A, variant = _gpu(w, len(sizes), off, steps)
    assert P.base_variant(variant) == ("uniform" if uniform else "general")
    o = _oracle(oracle_mod, w, len(sizes), off, steps)
    l2, mr = _assert_regions(S, o.spectrum(), f"regions {D}x{W}")
    P.assert_parity(Stot, o.spectrum_total(), what="total spectrum")
    Aref = o.amplitude()
    assert np.abs(A - Aref).max() <= 2e-5 * np.abs(Aref).max()
    print(f"regions {D}x{W} {np.dtype(dtype).name} relL2={l2:.2e} maxrel={mr:.2e}")


def test_regions_match_independent_plain_detectors_and_global(oracle_mod):
    """A per-region handle gives, region by region, what a plain detector fed only that
    region's particles gives, and its total is the plain detector of all particles."""
    w = wl.make_workload("5r")
    n = 9000
    off = w.region_offsets(n)
    steps = list(w.steps(n_steps=2, n_particles=n))
    S, Stot, _, _ = _gpu(w, w.n_regions, off, steps)
    for r in (0, 5, 11):
        sub = [(t, [a[off[r]:off[r + 1]] for a in st]) for t, st in steps]
        Sr, _ = P.run_gpu(w, sub)
        assert P.rel_l2(S[r], Sr) < 1e-6
    Sall, _ = P.run_gpu(w, steps)
    assert P.rel_l2(Stot, Sall) < 1e-6


def test_regions_offsets_gaps_host_path_deterministic_and_errors(oracle_mod):
    from paper_2501_03383_b200 import binding
    w = wl.Workload("reg", 3000, 2, 1e-17, wl.dirs_fibonacci(6), wl.omega_log(80), np.float32,
                    wl.BASE_SEED + 31, "khi")
    steps = list(w.steps())
    off = np.array([100, 900, 900, 2100, 2990], dtype=np.int64)   # head and tail belong to no region
    R = len(off) - 1
    ref = _oracle(oracle_mod, w, R, off, steps).spectrum()
    S, _, _, _ = _gpu(w, R, off, steps)
    _assert_regions(S, ref, "gaps")
    Sh, _, _, _ = _gpu(w, R, off, steps, host=True)
    _assert_regions(Sh, ref, "host path")
    Sd1, _, _, _ = _gpu(w, R, off, steps, flags=binding.RAD_FLAG_DETERMINISTIC)
    Sd2, _, _, _ = _gpu(w, R, off, steps, flags=binding.RAD_FLAG_DETERMINISTIC)
    _assert_regions(Sd1, ref, "deterministic")
    assert np.array_equal(Sd1, Sd2)
    # offsets may change from call to call (the chunk table is rebuilt)
    off2 = np.array([0, 10, 1500, 1500, 3000], dtype=np.int64)
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, n_regions=R) as det:
        det.accumulate_step_regions(0, off, P.to_device(steps[0][1]))
        det.accumulate_step_regions(1, off2, P.to_device(steps[1][1]))
        o = oracle_mod.RegionOracle(R, w.dirs, w.omega, w.dt, scale=1.0)
        o.accumulate_step(0, off, *steps[0][1])
        o.accumulate_step(1, off2, *steps[1][1])
        _assert_regions(det.spectrum(), o.spectrum(), "changing offsets")
        # error paths
        with pytest.raises(binding.RadError, match="INVALID_ARG"):
            det.accumulate_step(0, P.to_device(steps[0][1]))
        with pytest.raises(binding.RadError, match="INVALID_ARG"):
            det.accumulate_step_regions(0, off[:-1], P.to_device(steps[0][1]))
        with pytest.raises(binding.RadError, match="non-decreasing"):
            det.accumulate_step_regions(0, np.array([0, 50, 40, 60, 70]), P.to_device(steps[0][1]))
        det.reset()
        assert np.all(det.spectrum() == 0.0)
        det.accumulate_step_regions(0, np.zeros(R + 1, dtype=np.int64), P.to_device(steps[0][1]))  # all empty
        assert np.all(det.spectrum() == 0.0)
    # a plain handle accepts the region call with one region (a sub-range of the arrays)
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0) as det:
        det.accumulate_step_regions(0, np.array([100, 2000]), P.to_device(steps[0][1]))
        sub = [a[100:2000] for a in steps[0][1]]
        P.assert_parity(det.spectrum(), P.run_oracle(oracle_mod, w, [(0, sub)]).spectrum(), what="R=1 sub-range")


def test_cfg5r_full_particles_sampled_bins(oracle_mod):
    """cfg 5r at its full particle count (331 776 in 12 sub-volumes, the launch configuration
    bench.py --config 5r times), 2 steps; oracle on sampled bins of every region."""
    w = wl.make_workload("5r")
    off = w.region_offsets()
    steps = list(w.steps(n_steps=2))
    S, Stot, _, variant = _gpu(w, w.n_regions, off, steps)
    js = np.unique(np.concatenate([np.linspace(0, w.n_omega - 1, 10).round().astype(int),
                                   [int(np.argmax(S.max(axis=(0, 1))))]])).astype(np.int64)
    o = _oracle(oracle_mod, w, w.n_regions, off, steps, bins=js)
    Sref = o.spectrum()
    for r in range(w.n_regions):
        P.assert_parity(S[r][:, js], Sref[r][:, js], peak=S[r].max(), what=f"cfg5r region {r}")
    P.assert_parity(Stot[:, js], o.spectrum_total()[:, js], peak=Stot.max(), what="cfg5r total")
    assert P.base_variant(variant) == "general"


@pytest.mark.parametrize("flags", [0, 1])
def test_regions_multi_step_one_launch(oracle_mod, flags):
    """rad_accumulate_steps_regions == the per-step region calls: 4 steps, ragged regions incl.
    empty ones and an unassigned head/tail, row stride > n (NaN padding must not be read)."""
    import torch
    from paper_2501_03383_b200 import binding
    w = wl.Workload("reg", 2500, 4, 1e-17, wl.dirs_fibonacci(3), wl.omega_log(200), np.float32,
                    wl.BASE_SEED + 32, "khi")
    steps = [(50 + t, st) for t, st in w.steps()]
    off = np.array([40, 700, 700, 1733, 1734, 2490], dtype=np.int64)
    R = len(off) - 1
    ref = _oracle(oracle_mod, w, R, off, steps).spectrum()
    stride = 2500 + 12
    state = []
    for c in range(10):
        a = np.full((4, stride), np.nan, dtype=np.float32)
        for i, (_, st) in enumerate(steps):
            a[i, :2500] = st[c]
        state.append(torch.from_numpy(a).cuda())
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, n_regions=R, flags=flags) as det:
        l0 = det.launch_count
        det.accumulate_steps(50, state, region_offsets=off)
        if flags == 0:
            assert det.launch_count - l0 == 1
        _assert_regions(det.spectrum(), ref, "regions multi-step")
        with pytest.raises(binding.RadError, match="step_stride"):
            binding.rad_accumulate_steps_regions(det.handle, 0, 2, 100, off, [a.data_ptr() for a in state], 0)
