"""GPU parity: CUDA path (through the C ABI) vs the fp64 oracle, element by element, on the
same seeded inputs.  Tolerances are BASELINE.json north_star's (tests/_parity.py)."""
import numpy as np
import pytest

from paper_2501_03383_b200 import workloads as wl
from tests import _parity as P

pytestmark = pytest.mark.gpu

C = 299792458.0


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    import torch
    from paper_2501_03383_b200 import build
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    build.build()


def test_cfg0_tiny_helical_full(oracle_mod):
    """BASELINE.json configs[0] in full: 256 e-, 128 steps, 8 x 64 bins, fp64 state."""
    w = wl.make_workload("0")
    steps = list(w.steps())
    S, A, variant = P.run_gpu(w, steps, want_amplitude=True)
    o = P.run_oracle(oracle_mod, w, steps)
    l2, mr = P.assert_parity(S, o.spectrum(), what="cfg0")
    Aref = o.amplitude()
    assert np.abs(A - Aref).max() <= 2e-5 * np.abs(Aref).max()
    print(f"cfg0 variant={variant} relL2={l2:.2e} maxrel={mr:.2e}")
    assert P.base_variant(variant) == "uniform"      # linear grid -> rotation-recurrence kernel (a2')
    # the general kernel must give the same answer on the same grid
    from paper_2501_03383_b200 import binding
    Sg, vg = P.run_gpu(w, steps, flags=binding.RAD_FLAG_FORCE_GENERAL)
    assert P.base_variant(vg) == "general"
    P.assert_parity(Sg, o.spectrum(), what="cfg0 general kernel")


@pytest.mark.parametrize("D,W,dtype", [(37, 300, np.float32), (5, 1024, np.float32), (64, 64, np.float64)])
def test_uniform_grid_recurrence_kernel(oracle_mod, D, W, dtype):
    """a2': linear frequency grids (any tile shape, ragged W) use the recurrence kernel and
    match the oracle; high frequencies (up to 2e17 rad/s) stress the rotator phase."""
    w = wl.Workload("lin", 1500, 3, 1e-17, wl.dirs_fibonacci(D), np.linspace(2e14, 2e17, W), dtype,
                    wl.BASE_SEED + 20, "khi")
    steps = [(t * 400, st) for t, st in w.steps(n_steps=3)]
    S, variant = P.run_gpu(w, steps)
    assert P.base_variant(variant) == "uniform"
    l2, mr = P.assert_parity(S, P.run_oracle(oracle_mod, w, steps).spectrum(), what=f"uniform {D}x{W}")
    print(f"uniform {D}x{W} relL2={l2:.2e} maxrel={mr:.2e}")


@pytest.mark.parametrize("D,W", [(1, 40), (3, 16), (2, 20), (4, 24), (1, 100), (8, 70), (1, 17), (1, 31), (5, 257)])
@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_uniform_grid_padded_anchor_shapes(oracle_mod, D, W, dtype):
    """Linear grids whose width is not a multiple of the frequency tile: a thread's chain anchor
    (its middle bin) is then a PADDED bin while lower bins of its strip are valid, so the padded
    part of the frequency tables must continue the grid (round-1 bug: every bin of 1x40, 3x16,
    2x20, 4x24 was wrong).  W = 17, 31 with one direction also make the rotator step exceed
    2^32 f_unit (32 lanes along frequency, lw > W - 1)."""
    w = wl.Workload("lin_pad", 700, 2, 1e-17, wl.dirs_fibonacci(max(D, 2))[:D], np.linspace(3e14, 3e17, W), dtype,
                    wl.BASE_SEED + 21, "khi")
    steps = [(t * 300 + 1, st) for t, st in w.steps(n_steps=2)]
    S, variant = P.run_gpu(w, steps)
    assert P.base_variant(variant) == "uniform"
    ref = P.run_oracle(oracle_mod, w, steps).spectrum()
    l2, mr = P.assert_parity(S, ref, what=f"uniform padded {D}x{W}")
    for d in range(D):
        P.assert_parity(S[d], ref[d], what=f"uniform padded {D}x{W} dir {d}")
    from paper_2501_03383_b200 import binding
    Sg, vg = P.run_gpu(w, steps, flags=binding.RAD_FLAG_FORCE_GENERAL)
    assert P.base_variant(vg) == "general" and P.rel_l2(S, Sg) < 1e-5


@pytest.mark.parametrize("frac", [0.0, 1.0 / 64.0, 0.5, 0.25 + 1e-4])
def test_uniform_grid_recurrence_degenerate_angles(oracle_mod, frac):
    """The uniform-grid kernel reaches the bins of a strip by the three-term recurrence z(i+1) = 2 cos(theta) z(i) - z(i-1)
    with theta = LW dw tau, whose error growth is worst at the double root sin(theta) = 0.  Here
    every particle sits where dw tau = 2 pi (m + frac) with an integer m of up to 3000 turns, so that all chains of the
    sweep run at one angle: theta = 0 (frac 0; 1/2 with an even LW), pi (1/64 with 32 lanes along frequency), or close to
    pi / 2's multiples; fp64 state so that the positions carry the angle.  All bins against the oracle."""
    W, n = 256, 900
    omega = np.linspace(2e15, 4e17, W)
    dw = omega[1] - omega[0]
    w = wl.Workload("uni_deg", n, 1, 1e-17, np.array([[0.0, 0.6, 0.8]]), omega, np.float64, wl.BASE_SEED + 31, "khi")
    (_, st), = list(w.steps(n_steps=1))
    st = [np.array(a, dtype=np.float64) for a in st]
    rng = np.random.default_rng(4242)
    tau = 2.0 * np.pi * (rng.integers(0, 3000, size=n) + frac) / dw      # retarded time of each particle at t = 0
    for c in range(3):
        st[c] = -wl.C_LIGHT * tau * w.dirs[0, c]                          # tau = t0 + t dt - n.r / c with t0 = t = 0
    steps = [(0, st)]
    S, variant = P.run_gpu(w, steps)
    assert P.base_variant(variant) == "uniform"
    ref = P.run_oracle(oracle_mod, w, steps).spectrum()
    P.assert_parity(S, ref, what=f"uniform degenerate angle frac={frac}")


def test_precise_flag_all_polynomial_sincos(oracle_mod):
    """RAD_FLAG_PRECISE: every sin/cos by the fp32 polynomial on the general-grid kernel, whatever the grid (log,
    linear, few bins).  (a) parity on the usual shapes; (b) the dark-bin case a 1200-case random hunt found
    (33 directions x 17 linear frequencies, three sub-volumes of 210 / 768 / 2022 particles,
    a bin at 2.8e-6 of the peak where the default kernels reach 1.2e-3 / 1.6e-3): within the tolerance with the
    flag, and at least 2x closer to the oracle than the default general kernel; (c) unsupported combinations."""
    from paper_2501_03383_b200 import binding
    for D, W, om in ((5, 96, wl.omega_log(96)), (3, 40, np.linspace(2e14, 2e17, 40)), (1, 8, wl.omega_log(8))):
        w = wl.Workload("prec", 1500, 2, 1e-17, wl.dirs_fibonacci(max(D, 2))[:D], om, np.float32, wl.BASE_SEED + 27, "khi")
        steps = list(w.steps())
        S, variant = P.run_gpu(w, steps, flags=binding.RAD_FLAG_PRECISE)
        assert variant == "general+precise"
        P.assert_parity(S, P.run_oracle(oracle_mod, w, steps).spectrum(), what=f"precise {D}x{W}")
    rng = np.random.default_rng(7700 + 148)          # the drawn case 148 of a 1200-case run of tests/test_gpu_fuzz.py
    om = np.linspace(3.71364082e14, 2.12037748e17, 17)
    w = wl.Workload("dark", 3000, 3, 1e-17, wl.dirs_fibonacci(33), om, np.float64, 169478, "khi")
    steps = list(w.steps())
    off = np.array([0, 210, 978, 3000], dtype=np.int64)
    o = oracle_mod.RegionOracle(3, w.dirs, w.omega, w.dt, scale=1.0)
    for t, st in steps:
        o.accumulate_step(t, off, *st)
    ref = o.spectrum()
    err = {}
    for name, flags in (("default", binding.RAD_FLAG_FORCE_GENERAL), ("precise", binding.RAD_FLAG_PRECISE)):
        with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, state_dtype=np.float64, flags=flags, n_regions=3) as det:
            for t, st in steps:
                det.accumulate_step_regions(t, off, P.to_device(st))
            err[name] = P.max_rel(det.spectrum(), ref)
    print(f"dark-bin case: maxrel default general kernel {err['default']:.2e}, RAD_FLAG_PRECISE {err['precise']:.2e}")
    assert err["precise"] <= P.MAX_REL_TOL and err["precise"] < 0.5 * err["default"]
    for kw in (dict(nyquist=0.5), dict(form_factor=("gaussian", (1e-8,) * 3)),
               dict(flags=binding.RAD_FLAG_FAST_GRIDDED, fast=((0, 0, 0), (1e-5, 1e-5, 1e-5), 0, 1, 0.0))):
        kw["flags"] = kw.get("flags", 0) | binding.RAD_FLAG_PRECISE
        with pytest.raises(binding.RadError, match="UNSUPPORTED"):
            binding.Detector(w.dirs, w.omega, w.dt, **kw)


@pytest.mark.parametrize("D,W,grid,dtype", [(1, 64, "log", np.float32), (1, 128, "log", np.float32), (2, 64, "log", np.float64),
                                            (1, 100, "log", np.float32), (3, 24, "log", np.float32), (1, 40, "linear", np.float32),
                                            (2, 60, "linear", np.float64), (1, 17, "log", np.float32)])
def test_particle_split_few_directions(oracle_mod, D, W, grid, dtype):
    """Detectors with fewer directions than a warp's frequency tile leaves room for: the lane groups of a
    warp share a direction and split the particles of a batch (variant "+split"); partial sums meet in a
    shuffle reduction before the fold.  All bins against the oracle, ragged particle counts, late steps,
    deterministic mode bit-reproducible, multi-step launch."""
    import torch
    from paper_2501_03383_b200 import binding
    om = wl.omega_log(W) if grid == "log" else np.linspace(2e14, 2e17, W)
    w = wl.Workload("split", 2077, 3, 1e-17, wl.dirs_fibonacci(max(D, 2))[:D], om, dtype, wl.BASE_SEED + 26, "khi")
    steps = [(t * 300 + 1, st) for t, st in w.steps()]
    ref = P.run_oracle(oracle_mod, w, steps).spectrum()
    S, variant = P.run_gpu(w, steps)
    assert variant == ("uniform+split" if grid == "linear" else "general+split")
    P.assert_parity(S, ref, what=f"split {D}x{W} {grid}")
    for d in range(D):
        P.assert_parity(S[d], ref[d], what=f"split {D}x{W} {grid} dir {d}")
    runs = [P.run_gpu(w, steps, flags=binding.RAD_FLAG_DETERMINISTIC)[0] for _ in range(2)]
    assert np.array_equal(runs[0], runs[1])
    P.assert_parity(runs[0], ref, what=f"split {D}x{W} deterministic")
    stacked = [torch.from_numpy(np.stack([st[c] for _, st in steps])).cuda() for c in range(10)]
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, state_dtype=dtype) as det:
        det.accumulate_step(1, P.to_device(steps[0][1]))
        det.reset()
        for i in range(3):      # steps 1, 301, 601 are not consecutive: three one-step multi-step calls
            det.accumulate_steps(steps[i][0], [a[i:i + 1] for a in stacked])
        P.assert_parity(det.spectrum(), ref, what=f"split {D}x{W} multi-step entry")


@pytest.mark.parametrize("D,W,b,dtype", [(6, 300, 32, np.float32), (3, 512, 64, np.float32), (33, 100, 8, np.float32),
                                         (9, 70, 16, np.float64), (16, 40, 4, np.float32), (2, 1000, 64, np.float64)])
def test_dyadic_log_grid_squaring_chains(oracle_mod, D, W, b, dtype):
    """SURVEY.md section 8(f) NEXT-4, second half: log grids with an integer number b of bins per octave
    run the squaring-chain variant (z(2w) = z(w)^2, every third bin of a chain anchored by a direct
    sincos) -- every tile shape (b = 4 ... 64 = lanes x chain stride), ragged W (padded anchors), late
    steps; same tolerances, per direction too; the plain general kernel on the same grid agrees."""
    from paper_2501_03383_b200 import binding
    w = wl.Workload("dyad", 1500, 3, 1e-17, wl.dirs_fibonacci(max(D, 2))[:D], wl.omega_dyadic(W, b), dtype,
                    wl.BASE_SEED + 23, "khi")
    steps = [(t * 350 + 2, st) for t, st in w.steps(n_steps=3)]
    S, variant = P.run_gpu(w, steps)
    assert variant == "general+dyadic"
    ref = P.run_oracle(oracle_mod, w, steps).spectrum()
    l2, mr = P.assert_parity(S, ref, what=f"dyadic {D}x{W} b={b}")
    for d in range(D):
        P.assert_parity(S[d], ref[d], what=f"dyadic {D}x{W} b={b} dir {d}")
    Sg, vg = P.run_gpu(w, steps, flags=binding.RAD_FLAG_FORCE_GENERAL)
    assert P.base_variant(vg) == "general" and P.rel_l2(S, Sg) < 1e-5
    l2g, mrg = P.assert_parity(Sg, ref, what=f"general on the dyadic grid {D}x{W}")
    print(f"dyadic {D}x{W} b={b} {np.dtype(dtype).name}: relL2={l2:.2e} maxrel={mr:.2e} (plain general kernel: {l2g:.2e} / {mrg:.2e})")


def test_dyadic_grid_with_regions_multi_step_deterministic_and_overlap(oracle_mod):
    """The squaring-chain variant under the other call forms: per-region handle (ragged regions, one
    launch), rad_accumulate_steps (one launch for all steps), deterministic mode (bit-reproducible),
    RAD_FLAG_OVERLAP_STEPS with a spectrum between steps."""
    import torch
    from paper_2501_03383_b200 import binding
    w = wl.Workload("dyad2", 2600, 4, 1e-17, wl.dirs_fibonacci(5), wl.omega_dyadic(200, 16), np.float32,
                    wl.BASE_SEED + 25, "khi")
    steps = list(w.steps())
    ref = P.run_oracle(oracle_mod, w, steps).spectrum()
    off = np.array([0, 700, 700, 701, 1500, 2600], dtype=np.int64)
    ro = oracle_mod.RegionOracle(5, w.dirs, w.omega, w.dt, scale=1.0)
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, n_regions=5) as det:
        for t, st in steps:
            det.accumulate_step_regions(t, off, P.to_device(st))
            ro.accumulate_step(t, off, *st)
        assert det.kernel_variant == "general+dyadic"
        Sr, St = det.spectrum(), det.spectrum_total()
    P.assert_parity(St, ref, what="dyadic regions total")
    Rr = ro.spectrum()
    for r in (0, 3, 4):
        P.assert_parity(Sr[r], Rr[r], what=f"dyadic region {r}")
    assert np.all(Sr[1] == 0.0)
    stacked = [torch.from_numpy(np.stack([st[c] for _, st in steps])).cuda() for c in range(10)]
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0) as det:
        det.accumulate_steps(0, stacked)
        assert det.kernel_variant == "general+dyadic"
        P.assert_parity(det.spectrum(), ref, what="dyadic multi-step")
    runs = []
    for _ in range(2):
        S, v = P.run_gpu(w, steps, flags=binding.RAD_FLAG_DETERMINISTIC)
        assert v == "general+dyadic"
        runs.append(S)
    assert np.array_equal(runs[0], runs[1])
    P.assert_parity(runs[0], ref, what="dyadic deterministic")
    devs = [P.to_device(st) for _, st in steps]
    torch.cuda.synchronize()
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, flags=binding.RAD_FLAG_OVERLAP_STEPS) as det:
        mids = []
        for (t, _), dev in zip(steps, devs):
            det.accumulate_step(t, dev)
            mids.append(det.spectrum())
        o = oracle_mod.Oracle(w.dirs, w.omega, w.dt, scale=1.0)
        for (t, st), S in zip(steps, mids):
            o.accumulate_step(t, *st)
            P.assert_parity(S, o.spectrum(), what=f"dyadic overlap after step {t}")


def test_dyadic_detection_falls_back(oracle_mod):
    """Not dyadic (BASELINE.json's own log grids: 38.46 bins per octave), bins per octave the tile shapes
    cannot divide (12), or a dyadic grid with one perturbed bin: the plain general kernel."""
    for om in (wl.omega_log(512), wl.omega_dyadic(200, 12), wl.omega_dyadic(300, 32) * (1 + 1e-9 * (np.arange(300) == 77))):
        w = wl.Workload("nodyad", 300, 1, 1e-17, wl.dirs_fibonacci(4), om, np.float32, wl.BASE_SEED + 24, "khi")
        steps = list(w.steps())
        S, variant = P.run_gpu(w, steps)
        assert P.base_variant(variant) == "general"
        P.assert_parity(S, P.run_oracle(oracle_mod, w, steps).spectrum(), what="non-dyadic log grid")


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("shape", ["general", "uniform", "stream"])
def test_non_finite_particle_state_propagates(dtype, shape):
    """include/rad.h: particle values are not scanned; NaN/Inf in the state give NaN/Inf in the
    result.  One NaN (or Inf) particle among 500 must poison every bin it contributes to, on every
    kernel, for fp32 and fp64 state alike (round 1 mapped fp32 Inf/NaN positions to finite numbers)."""
    from paper_2501_03383_b200 import binding
    if shape == "stream":
        dirs, omega = wl.dirs_fibonacci(2)[:1], wl.omega_log(8)
    elif shape == "uniform":
        dirs, omega = wl.dirs_fibonacci(3), np.linspace(2e14, 4e16, 48)
    else:
        dirs, omega = wl.dirs_fibonacci(3), wl.omega_log(40)
    w = wl.Workload("nonfinite", 500, 1, 1e-17, dirs, omega, dtype, wl.BASE_SEED + 60, "khi")
    (t, st), = list(w.steps())
    for col, bad in ((0, np.nan), (1, np.inf), (4, np.nan), (7, np.nan), (9, np.inf)):
        st2 = [a.copy() for a in st]
        st2[col][123] = bad
        with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, state_dtype=dtype) as det:
            det.accumulate_step(0, P.to_device(st2))
            S, variant = det.spectrum(), det.kernel_variant
        assert P.base_variant(variant) == shape
        assert not np.isfinite(S).any(), f"column {col} = {bad}: finite bins remain"
    S_ok, _ = P.run_gpu(w, [(0, st)])
    assert np.isfinite(S_ok).all()


@pytest.mark.parametrize("cfg", ["1", "2", "3a", "3b", "3c", "3d", "4"])
def test_reduced_particles_all_bins(oracle_mod, cfg):
    """Every bin / tile path of configs 1-4 on a reduced workload (first 1000 particles --
    a ragged tail for the 32-particle batches -- x 3 steps, incl. a late step index)."""
    w = wl.make_workload(cfg)
    n = 1000 if w.n_dir * w.n_omega <= 65536 else 300
    steps = [(t if i < 2 else w.n_steps - 1, st) for i, (t, st) in enumerate(w.steps(n_steps=3, n_particles=n))]
    S, variant = P.run_gpu(w, steps)
    o = P.run_oracle(oracle_mod, w, steps)
    l2, mr = P.assert_parity(S, o.spectrum(), what=f"cfg{cfg} reduced")
    print(f"cfg{cfg} reduced variant={variant} relL2={l2:.2e} maxrel={mr:.2e}")


def test_cfg1_many_particles_bin_subset(oracle_mod):
    """Config 1 particle count (65 536, spans many chunks/blocks) x 4 steps; oracle on a
    stratified bin subset plus the GPU arg-max bin (bins are independent sums)."""
    w = wl.make_workload("1")
    steps = list(w.steps(n_steps=4))
    S, _ = P.run_gpu(w, steps)
    bins = P.stratified_bins(w.n_dir, w.n_omega, 4, 8, extra=[int(np.argmax(S))])
    o = P.run_oracle(oracle_mod, w, steps, bins=bins)
    Sref = o.spectrum().ravel()[bins]
    P.assert_parity(S.ravel()[bins], Sref, peak=S.max(), what="cfg1 subset")
    assert S.ravel()[int(np.argmax(S))] == pytest.approx(o.spectrum().ravel()[int(np.argmax(S))], rel=1e-4)


def test_closed_form_pins_on_gpu():
    """The oracle's closed forms hold for the CUDA path too (Dirichlet kernel incl. complex
    phase, Doppler shift): a direct GPU-vs-mathematics check, no oracle involved."""
    dirs = np.array([[1.0, 0, 0], [0, 0, 2.0], [0.3, -0.5, 0.8], [-0.6, 0.64, 0.48]])
    unit = dirs / np.linalg.norm(dirs, axis=1, keepdims=True)
    omega = np.array([3.0e14, 1.0e15, 2.7e15, 8.1e15, 3.3e16])
    dt, T, wgt, t0 = 2.0e-17, 31, 0.8, 3.7e-16
    r0 = np.array([0.4e-6, 0.9e-6, -0.3e-6]); beta = np.array([0.31, -0.12, 0.22])
    b = np.array([-1.0e12, 3.0e12, 2.0e12])
    w = wl.Workload("pin", 1, T, dt, dirs, omega, np.float64, 0, "helix", t0=t0)
    steps = [(t, [np.array([v]) for v in list(r0 + C * beta * t * dt) + list(beta) + list(b) + [wgt]])
             for t in range(T)]
    S, A, _ = P.run_gpu(w, steps, want_amplitude=True)
    for i, n in enumerate(unit):
        d = 1.0 - n @ beta
        vec = (n - beta) * (n @ b) - b * d
        for j, om in enumerate(omega):
            x = om * d * dt
            dk = np.sin(T * x / 2) / np.sin(x / 2)
            assert S[i, j] == pytest.approx(wgt ** 2 * (vec @ vec) / d ** 4 * dt ** 2 * dk ** 2, rel=2e-5)
            ph = np.exp(1j * om * (t0 - (n @ r0) / C)) * np.exp(1j * x * (T - 1) / 2.0)
            a_ref = wgt * dt * vec / d ** 2 * ph * dk
            assert np.abs(A[i, j] - a_ref).max() <= 2e-5 * np.abs(a_ref).max()


def test_zero_for_unaccelerated_motion_and_linearity():
    w = wl.make_workload("3c")
    (t, st), = list(w.steps(n_steps=1, n_particles=777))
    zero = st[:6] + [np.zeros_like(st[6])] * 3 + [st[9]]
    S, _ = P.run_gpu(w, [(0, zero)])
    assert np.all(S == 0.0)
    S1, _ = P.run_gpu(w, [(0, st)])
    S3, _ = P.run_gpu(w, [(0, st[:9] + [3.0 * st[9]])])
    m = S1 > 1e-9 * S1.max()
    assert np.allclose(S3[m], 9.0 * S1[m], rtol=1e-4)
    # same particles split over two calls with the same step index
    Ssplit, _ = P.run_gpu(w, [(0, [a[:300] for a in st]), (0, [a[300:] for a in st])])
    assert P.rel_l2(Ssplit, S1) < 1e-6


def test_api_semantics_reset_add_amplitude_host_path_deterministic(oracle_mod):
    import torch
    from paper_2501_03383_b200 import binding
    w = wl.make_workload("3b")
    steps = list(w.steps(n_steps=2, n_particles=2500))
    ref = P.run_oracle(oracle_mod, w, steps).spectrum()
    # host-buffer entry point (library stages the copies)
    S_host, _ = P.run_gpu(w, steps, host=True)
    P.assert_parity(S_host, ref, what="host path")
    # deterministic flag: parity and bit-reproducibility
    Sd1, _ = P.run_gpu(w, steps, flags=binding.RAD_FLAG_DETERMINISTIC)
    Sd2, _ = P.run_gpu(w, steps, flags=binding.RAD_FLAG_DETERMINISTIC)
    P.assert_parity(Sd1, ref, what="deterministic")
    assert np.array_equal(Sd1, Sd2)
    # reset + add_amplitude: two detectors on particle halves, amplitudes summed (multi-GPU path)
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0) as a, \
            binding.Detector(w.dirs, w.omega, w.dt, scale=1.0) as b:
        for t, st in steps:
            a.accumulate_step(t, P.to_device([x[:1200] for x in st]))
            b.accumulate_step(t, P.to_device([x[1200:] for x in st]))
        amp_a = torch.empty(w.n_dir, w.n_omega, 3, 2, dtype=torch.float64, device="cuda")
        amp_b = torch.empty_like(amp_a)
        a.amplitude(out=amp_a); b.amplitude(out=amp_b)
        total = amp_a + amp_b
        a.reset()
        assert np.all(a.spectrum() == 0.0)
        a.add_amplitude(total)
        P.assert_parity(a.spectrum(), ref, what="add_amplitude")
        out_dev = torch.empty(w.n_dir, w.n_omega, dtype=torch.float64, device="cuda")
        a.spectrum(out=out_dev)
        torch.cuda.synchronize()
        assert np.array_equal(out_dev.cpu().numpy(), a.spectrum())
        assert a.launch_count > 0


def test_edge_cases(oracle_mod):
    from paper_2501_03383_b200 import binding
    # single direction, single frequency, single particle; default SI scale
    w = wl.Workload("edge", 1, 1, 1e-17, np.array([[0.0, 1.0, 0.0]]), np.array([5e15]), np.float32, 0, "khi")
    st = [np.array([v], dtype=np.float32) for v in (1e-6, 2e-6, 3e-6, 0.1, 0.2, 0.0, 1e12, -2e12, 5e11, 2.0)]
    S, _ = P.run_gpu(w, [(5, st)], scale=0.0)
    ref = P.run_oracle(oracle_mod, w, [(5, st)], scale=0.0).spectrum()
    assert S[0, 0] == pytest.approx(ref[0, 0], rel=1e-5)
    # empty input is a no-op; ragged sizes 1, 31, 33; awkward grid 5 x 37
    w2 = wl.Workload("ragged", 33, 1, 1e-17, wl.dirs_fibonacci(5), wl.omega_log(37), np.float32,
                     wl.BASE_SEED + 9, "khi")
    (t, full), = list(w2.steps(n_steps=1))
    with binding.Detector(w2.dirs, w2.omega, w2.dt, scale=1.0) as det:
        det.accumulate_step(0, P.to_device([a[:0] for a in full]))
        assert np.all(det.spectrum() == 0.0)
    for n in (1, 31, 33):
        sub = [a[:n] for a in full]
        S, _ = P.run_gpu(w2, [(0, sub)])
        P.assert_parity(S, P.run_oracle(oracle_mod, w2, [(0, sub)]).spectrum(), what=f"ragged n={n}")
    # large |tau|: late time and far-away particles (integer phase path wraps exactly)
    w3 = wl.Workload("far", 64, 1, 1e-17, wl.dirs_fibonacci(8), wl.omega_log(64), np.float64,
                     wl.BASE_SEED + 10, "khi", t0=1e-10)
    (t, st3), = list(w3.steps(n_steps=1))
    st3 = [a.copy() for a in st3]
    st3[0] += 0.5; st3[2] -= 2.0   # metres away from the origin (fp64 state)
    S, _ = P.run_gpu(w3, [(12345, st3)])
    P.assert_parity(S, P.run_oracle(oracle_mod, w3, [(12345, st3)]).spectrum(), what="far/late")


# ------------------------------------------------------------------ full sizes, sampled bins
def _full_size_sampled(oracle_mod, cfg, n_steps, bins, flag_sets=None, check_argmax=True, fast=False):
    """BASELINE.json's full particle count in the launch configurations bench.py times: the same
    handle set-up and per-step call, once with flags = 0 and once with RAD_FLAG_OVERLAP_STEPS
    (bench.py's default).  The oracle computes the sampled `bins` one by one (bins are independent
    sums) ONCE; both GPU runs are compared with it, and the GPU arg-max bin (the S_peak of the
    maxrel criterion) is verified by a second, one-bin oracle pass."""
    import torch
    from paper_2501_03383_b200 import binding
    w = wl.make_workload(cfg)
    flag_sets = (0, binding.RAD_FLAG_OVERLAP_STEPS) if flag_sets is None else flag_sets
    o = oracle_mod.Oracle(w.dirs, w.omega, w.dt, t0=w.t0, scale=1.0, bins=bins)
    dets = [binding.Detector(w.dirs, w.omega, w.dt, t0=w.t0, scale=1.0, state_dtype=w.state_dtype, flags=f)
            for f in flag_sets]
    if fast:    # the approximate fast path rides along: same inputs, same oracle bins, same tolerances
        L = 10e-6
        flag_sets = tuple(flag_sets) + ("RAD_FLAG_FAST_GRIDDED",)
        dets.append(binding.Detector(w.dirs, w.omega, w.dt, t0=w.t0, scale=1.0, state_dtype=w.state_dtype,
                                     flags=binding.RAD_FLAG_FAST_GRIDDED,
                                     fast=((-0.02 * L,) * 3, (1.02 * L,) * 3, 0, n_steps - 1, 0.0)))
    kept = []
    try:
        block = []                              # steps are queued in blocks, back to back, so that the
        def flush():                            # kernels of consecutive steps really overlap under the flag
            devs = [P.to_device(st) for _, st in block]
            torch.cuda.synchronize()            # the flag's input contract: inputs complete before the calls
            for det in dets:
                for (t, _), dev in zip(block, devs):
                    det.accumulate_step(t, dev)
            for t, st in block:                 # the oracle works while the GPU does
                o.accumulate_step(t, *st)
            torch.cuda.synchronize()            # inputs stay alive until the kernels are done
            block.clear()
        for t, st in w.steps(n_steps=n_steps):
            block.append((t, st))
            if check_argmax and n_steps <= 4:
                kept.append((t, st))
            if len(block) == 50:
                flush()
        if block:
            flush()
        spectra = [det.spectrum() for det in dets]
    finally:
        for det in dets:
            det.close()
    Sref = o.spectrum().ravel()[bins]
    for f, S in zip(flag_sets, spectra):
        l2, mr = P.assert_parity(S.ravel()[bins], Sref, peak=S.max(), what=f"cfg{cfg} full-size sample flags={f}")
        print(f"cfg{cfg} full-size flags={f}: {len(bins)} bins relL2={l2:.2e} maxrel={mr:.2e}")
    if kept:       # the arg-max bin itself
        jmax = int(np.argmax(spectra[0]))
        om = oracle_mod.Oracle(w.dirs, w.omega, w.dt, t0=w.t0, scale=1.0, bins=np.array([jmax]))
        for t, st in kept:
            om.accumulate_step(t, *st)
        for S in spectra:
            assert int(np.argmax(S)) == jmax or S.ravel()[jmax] == pytest.approx(S.max(), rel=1e-5)
            assert S.ravel()[jmax] == pytest.approx(om.spectrum().ravel()[jmax], rel=1e-4)


def test_cfg1_full_workload_all_1000_steps(oracle_mod):
    """All 1000 steps of config 1 (late step indices, t up to 1e-14 s) on 64 + 4 sampled bins."""
    w = wl.make_workload("1")
    bins = P.tile_cover_bins(w.n_dir, w.n_omega, block=512, n_random=0, seed=11)[::2]
    _full_size_sampled(oracle_mod, "1", 1000, bins, check_argmax=False, fast=True)


def test_cfg1_full_particles_every_tile(oracle_mod):
    """Config 1 at its full particle count x 4 steps: >= 2048 oracle-checked bins, one in every
    (direction, 32-frequency block) -> every warp tile, every chunk of the tapered schedule."""
    w = wl.make_workload("1")
    bins = P.tile_cover_bins(w.n_dir, w.n_omega, block=32, n_random=2048, seed=12)
    assert len(bins) >= 2048
    _full_size_sampled(oracle_mod, "1", 4, bins, fast=True)


@pytest.mark.parametrize("cfg", ["3a", "3b", "3c", "3d"])
def test_cfg3_full_particles(oracle_mod, cfg):
    w = wl.make_workload(cfg)
    bins = P.tile_cover_bins(w.n_dir, w.n_omega, block=32, n_random=64, seed=13)
    assert len(bins) >= 2048
    _full_size_sampled(oracle_mod, cfg, 4, bins, fast=cfg in ("3a", "3c"))


def test_cfg2_full_particles(oracle_mod):
    """The headline configuration: 1 048 576 particles, 256 x 1024 bins (lw = 32: warp tile = one
    direction x 256 frequencies, so a 64-frequency block puts 4 samples into every tile)."""
    w = wl.make_workload("2")
    bins = P.tile_cover_bins(w.n_dir, w.n_omega, block=64, n_random=64, seed=14)
    assert len(bins) >= 4096
    _full_size_sampled(oracle_mod, "2", 2, bins, fast=True)


def test_cfg4_full_particles(oracle_mod):
    w = wl.make_workload("4")
    bins = P.tile_cover_bins(w.n_dir, w.n_omega, block=32, n_random=64, seed=15)
    _full_size_sampled(oracle_mod, "4", 1, bins)


# --------------------------------------------------------------- particle-streaming kernel
@pytest.mark.parametrize("D,W,dtype,n", [(1, 8, np.float32, 5000), (1, 8, np.float32, 4096), (2, 8, np.float32, 3001),
                                         (2, 3, np.float32, 1025), (1, 1, np.float32, 100), (1, 13, np.float32, 1537),
                                         (1, 8, np.float64, 2077), (2, 7, np.float64, 513)])
def test_stream_kernel_few_bins(oracle_mod, D, W, dtype, n):
    """<= 2 directions x <= 8 frequencies (or 1 x <= 16) -> particle-owner streaming kernel (bulk-copy staged tiles, ragged tail via
    plain loads, warp-shuffle reduction); parity incl. the deterministic mode."""
    from paper_2501_03383_b200 import binding
    w = wl.Workload("stream", n, 2, 1e-17, wl.dirs_fibonacci(max(D, 2))[:D], wl.omega_log(max(W, 2))[:W], dtype,
                    wl.BASE_SEED + 30, "khi")
    steps = [(t * 700, st) for t, st in w.steps(n_steps=2)]
    ref = P.run_oracle(oracle_mod, w, steps).spectrum()
    S, variant = P.run_gpu(w, steps)
    assert variant == "stream"
    P.assert_parity(S, ref, what=f"stream {D}x{W}")
    Sd, _ = P.run_gpu(w, steps, flags=binding.RAD_FLAG_DETERMINISTIC)
    Sd2, _ = P.run_gpu(w, steps, flags=binding.RAD_FLAG_DETERMINISTIC)
    P.assert_parity(Sd, ref, what=f"stream deterministic {D}x{W}")
    assert np.array_equal(Sd, Sd2)


def test_stream_kernel_unaligned_arrays_use_plain_loads(oracle_mod):
    """State arrays that are not 16-byte aligned (views at an odd offset) must not take the
    bulk-copy path; result still matches."""
    import torch
    from paper_2501_03383_b200 import binding
    w = wl.Workload("stream_unaligned", 4099, 1, 1e-17, wl.dirs_fibonacci(2)[:1], wl.omega_log(8), np.float32,
                    wl.BASE_SEED + 31, "khi")
    (t, st), = list(w.steps(n_steps=1))
    ref = P.run_oracle(oracle_mod, w, [(3, st)]).spectrum()
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0) as det:
        dev = []
        for a in st:
            buf = torch.empty(a.shape[0] + 1, dtype=torch.float32, device="cuda")
            buf[1:] = torch.from_numpy(a).cuda()
            dev.append(buf[1:])                      # 4-byte offset: not 16-B aligned
        assert dev[0].data_ptr() % 16 != 0
        det.accumulate_step(3, dev)
        S = det.spectrum()
    P.assert_parity(S, ref, what="stream unaligned")


def test_cfg4b_full_particles(oracle_mod):
    _full_size_sampled(oracle_mod, "4b", 1, np.arange(8, dtype=np.int64))


# ------------------------------------------------------------------ multi-step calls
def _stacked(steps, stride=None):
    """[(t, state)] with consecutive t -> 10 CUDA tensors [T, stride] (rows padded with NaN)."""
    import torch
    T, n = len(steps), steps[0][1][0].shape[0]
    stride = n if stride is None else stride
    out = []
    for c in range(10):
        a = np.full((T, stride), np.nan, dtype=steps[0][1][c].dtype)
        for i, (_, st) in enumerate(steps):
            a[i, :n] = st[c]
        out.append(torch.from_numpy(a).cuda())
    return out, n, stride


def test_accumulate_steps_cfg0_all_128_steps_in_one_launch(oracle_mod):
    """rad_accumulate_steps == the loop of rad_accumulate_step calls (rad.h): config 0 in full
    as ONE launch (uniform-grid kernel, fp64 state) against the oracle."""
    from paper_2501_03383_b200 import binding
    w = wl.make_workload("0")
    steps = list(w.steps())
    ref = P.run_oracle(oracle_mod, w, steps).spectrum()
    state, n, stride = _stacked(steps)
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, state_dtype=w.state_dtype) as det:
        l0 = det.launch_count
        det.accumulate_steps(0, state)
        assert det.launch_count - l0 == 1 and P.base_variant(det.kernel_variant) == "uniform"
        l2, mr = P.assert_parity(det.spectrum(), ref, what="cfg0 one launch")
    print(f"cfg0 128 steps in one launch relL2={l2:.2e} maxrel={mr:.2e}")


@pytest.mark.parametrize("cfg,n,T,pad,flags", [("3c", 1000, 5, 24, 0), ("1", 4100, 3, 0, 0), ("3d", 333, 4, 3, 0),
                                                ("3c", 500, 3, 0, 1), ("4b", 3000, 3, 8, 0),
                                                ("3c", 40, 50, 8, 0), ("0", 7, 100, 1, 0), ("3b", 33, 64, 0, 0)])
def test_accumulate_steps_matches_oracle_and_per_step_calls(oracle_mod, cfg, n, T, pad, flags):
    """Late first step index, row stride > n_particles (padding rows hold NaN and must not be
    read), ragged chunk tails; deterministic handles and few-bin detectors take the per-step
    fallback inside the library.  Also steps with very few particles (7, 33, 40) over many steps."""
    from paper_2501_03383_b200 import binding
    w = wl.make_workload(cfg)
    first = 700 if w.n_steps > 800 else 1
    steps = [(first + t, st) for t, st in w.steps(n_steps=T, n_particles=n)]
    ref = P.run_oracle(oracle_mod, w, steps).spectrum()
    state, n_, stride = _stacked(steps, stride=n + pad)
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, state_dtype=w.state_dtype, flags=flags) as det:
        binding.rad_accumulate_steps(det.handle, first, T, n, stride, [a.data_ptr() for a in state],
                                     det._stream())
        S = det.spectrum()
    P.assert_parity(S, ref, what=f"steps cfg{cfg}")
    S_loop, _ = P.run_gpu(w, steps, flags=flags)
    assert P.rel_l2(S, S_loop) < 1e-6


def test_accumulate_steps_argument_errors():
    import torch
    from paper_2501_03383_b200 import binding
    w = wl.make_workload("3c")
    z = [torch.zeros(2, 64, device="cuda") for _ in range(10)]
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0) as det:
        with pytest.raises(binding.RadError, match="step_stride"):
            binding.rad_accumulate_steps(det.handle, 0, 2, 64, 32, [a.data_ptr() for a in z], 0)
        binding.rad_accumulate_steps(det.handle, 0, 0, 64, 64, [a.data_ptr() for a in z], 0)   # no-op
        assert np.all(det.spectrum() == 0.0)
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, n_regions=3) as det:
        with pytest.raises(binding.RadError, match="UNSUPPORTED"):
            det.accumulate_steps(0, z)


def test_spectrum_to_pinned_host_async():
    """RAD_OUT_HOST_ASYNC: the result is in pinned host memory once the stream has passed the call;
    invalid destinations are rejected."""
    import torch
    from paper_2501_03383_b200 import binding
    w = wl.make_workload("3c")
    (t, st), = list(w.steps(n_steps=1, n_particles=500))
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0) as det:
        det.accumulate_step(t, P.to_device(st))
        pinned = torch.zeros(w.n_dir, w.n_omega, dtype=torch.float64).pin_memory()
        det.spectrum(out=pinned)
        torch.cuda.current_stream().synchronize()
        assert np.array_equal(pinned.numpy(), det.spectrum())
        with pytest.raises(binding.RadError, match="INVALID_ARG"):
            binding.rad_spectrum(det.handle, pinned.data_ptr(), 3, 0)


def test_multi_gpu_plumbing_on_one_device(oracle_mod):
    """The path bench.py --gpus N takes (multi.AmplitudeAllReduce: rad_export_accumulator -> all-reduce
    -> rad_spectrum_of on a side stream), emulated on one device: with no process group the
    all-reduce is the identity, so every queued global spectrum must equal the local spectrum of
    that step; and two 'ranks' = two handles on particle shards, whose exported accumulators are
    added (what the all-reduce delivers), must give the oracle's spectrum of all particles.
    rad_import_accumulator folds one rank's amplitude into the other's handle (same result)."""
    import torch
    from paper_2501_03383_b200 import binding, multi
    w = wl.make_workload("3b")
    T = 5
    steps = list(w.steps(n_steps=T, n_particles=1500))
    o = oracle_mod.Oracle(w.dirs, w.omega, w.dt, scale=1.0)
    dets = [binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, flags=binding.RAD_FLAG_OVERLAP_STEPS)
            for _ in range(2)]
    try:
        dev = [[P.to_device([a[slice(*multi.shard_range(1500, r, 2))] for a in st]) for _, st in steps]
               for r in range(2)]
        torch.cuda.synchronize()
        red = multi.AmplitudeAllReduce(dets[0])
        outs = [torch.empty(w.n_dir, w.n_omega, dtype=torch.float64, device="cuda") for _ in range(T)]
        plain = []
        for i, (t, _) in enumerate(steps):          # every step: accumulate, queue the exchange, go on
            dets[0].accumulate_step(t, dev[0][i])
            red.global_spectrum(out=outs[i])
        red.wait()
        torch.cuda.synchronize()
        with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0) as chk:   # rank 0's running spectrum, step by step
            for i, (t, _) in enumerate(steps):
                chk.accumulate_step(t, dev[0][i])
                plain.append(chk.spectrum())
        for i in range(T):
            assert np.allclose(outs[i].cpu().numpy(), plain[i], rtol=1e-9, atol=1e-12 * plain[-1].max()), f"step {i}"
        red.close()
        for t, st in steps:
            o.accumulate_step(t, *st)
        for i, (t, _) in enumerate(steps):
            dets[1].accumulate_step(t, dev[1][i])
        amp = [torch.empty(w.n_dir, w.n_omega, 4, dtype=torch.float64, device="cuda") for _ in range(2)]
        for r in range(2):
            dets[r].export_accumulator(amp[r])
        total = amp[0] + amp[1]                                  # what the all-reduce delivers
        ref = o.spectrum()
        P.assert_parity(dets[0].spectrum_of(total), ref, what="two shards summed")
        P.assert_parity(dets[1].spectrum_of(total), ref, what="two shards summed (other rank's handle)")
        dets[0].import_accumulator(amp[1])
        P.assert_parity(dets[0].spectrum(), ref, what="import_accumulator")
        # the 4-component export carries the whole amplitude: A1 e1 + A2 e2 == rad_amplitude
        A = dets[0].amplitude()
        assert np.abs(A - o.amplitude()).max() <= 2e-5 * np.abs(o.amplitude()).max()
    finally:
        for d in dets:
            d.close()


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_relativistic_beam_small_doppler_factor(oracle_mod, dtype):
    """Degenerate regime of the formula: beta -> 1 along the line of sight, 1 - beta.n down to
    ~1e-4 (gamma ~ 70), amplitudes spanning (1 - beta.n)^-2 ~ 1e8.  The Doppler factor is formed
    in fp64 on the GPU, so parity must hold for fp32 and fp64 state alike."""
    rng = np.random.default_rng(77)
    n = 2000
    gamma = 10.0 ** rng.uniform(0.5, 1.85, n)
    beta = np.sqrt(1.0 - 1.0 / gamma ** 2)
    th, ph = rng.normal(0, 2.0 / gamma), rng.uniform(0, 2 * np.pi, n)       # cone ~ 1/gamma around +x
    bx, by, bz = beta * np.cos(th), beta * np.sin(th) * np.cos(ph), beta * np.sin(th) * np.sin(ph)
    r = rng.uniform(0, 5e-6, (3, n))
    bd = rng.normal(0, 1e13, (3, n))
    st = [np.ascontiguousarray(a, dtype=dtype) for a in (r[0], r[1], r[2], bx, by, bz, bd[0], bd[1], bd[2],
                                                         rng.uniform(0.5, 2.0, n))]
    assert np.all(st[3].astype(np.float64) ** 2 + st[4].astype(np.float64) ** 2 + st[5].astype(np.float64) ** 2 < 1)
    dirs = np.array([[1.0, 0.0, 0.0], [0.9999, 0.01, 0.0], [0.99, 0.1, 0.05], [0.0, 1.0, 0.0], [-1.0, 0.0, 0.0]])
    w = wl.Workload("beam", n, 1, 1e-18, dirs, wl.omega_log(96, 1e15, 1e19), dtype, 0, "khi")
    steps = [(3, st), (4, st)]
    S, variant = P.run_gpu(w, steps)
    ref = P.run_oracle(oracle_mod, w, steps).spectrum()
    dmin = (1 - (dirs[0] / np.linalg.norm(dirs[0])) @ np.stack([st[3], st[4], st[5]]).astype(np.float64)).min()
    l2, mr = P.assert_parity(S, ref, what=f"relativistic beam {np.dtype(dtype).name}")
    for d in range(len(dirs)):      # every direction on its own scale (forward/backward differ by ~1e14)
        P.assert_parity(S[d], ref[d], what=f"beam dir {d}")
    print(f"beam {np.dtype(dtype).name}: min(1-beta.n)={dmin:.2e} relL2={l2:.2e} maxrel={mr:.2e}")


@pytest.mark.parametrize("kind,shape", [("triangle", "general"), ("hamming", "general"), ("hamming", "uniform"),
                                         ("triangle", "stream"), ("hamming", "regions")])
def test_spatial_window(oracle_mod, kind, shape):
    """NEXT-3 window functions (rad.h, reading W1) through every accumulate kernel: KHI particles
    in the 10 um box, window over x and y only (z extent 0), box chosen so that a part of the
    particles lies outside and gets weight exactly 0; fp32 state."""
    from paper_2501_03383_b200 import binding
    L = 10e-6
    win = (kind, (0.1 * L, -0.2 * L, 0.0), (0.7 * L, 1.1 * L, 0.0))
    if shape == "uniform":
        dirs, omega = wl.dirs_fibonacci(6), np.linspace(2e14, 4e16, 128)
    elif shape == "stream":
        dirs, omega = wl.dirs_fibonacci(1), wl.omega_log(8)
    else:
        dirs, omega = wl.dirs_fibonacci(5), wl.omega_log(96)
    w = wl.Workload("win", 3000, 2, 1e-17, dirs, omega, np.float32, wl.BASE_SEED + 40, "khi")
    steps = list(w.steps())
    if shape == "regions":
        off = np.array([0, 1000, 1000, 3000], dtype=np.int64)
        o = oracle_mod.RegionOracle(3, w.dirs, w.omega, w.dt, scale=1.0, window=win)
        for t, st in steps:
            o.accumulate_step(t, off, *st)
        with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, n_regions=3, window=win) as det:
            for t, st in steps:
                det.accumulate_step_regions(t, off, P.to_device(st))
            S = det.spectrum()
        for r in (0, 2):
            P.assert_parity(S[r], o.spectrum()[r], what=f"window regions {r}")
        assert np.all(S[1] == 0.0)
        return
    o = oracle_mod.Oracle(w.dirs, w.omega, w.dt, scale=1.0, window=win)
    for t, st in steps:
        o.accumulate_step(t, *st)
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, window=win) as det:
        for t, st in steps:
            det.accumulate_step(t, P.to_device(st))
        S, variant = det.spectrum(), det.kernel_variant
    assert P.base_variant(variant) == shape
    l2, mr = P.assert_parity(S, o.spectrum(), what=f"window {kind} {shape}")
    plain = P.run_oracle(oracle_mod, w, steps).spectrum()
    assert P.rel_l2(o.spectrum(), plain) > 0.1        # the window really changes the result
    print(f"window {kind}/{shape}: relL2={l2:.2e} maxrel={mr:.2e}")


def test_window_argument_errors_and_identity():
    from paper_2501_03383_b200 import binding
    w = wl.make_workload("3c")
    (t, st), = list(w.steps(n_steps=1, n_particles=400))
    with pytest.raises(binding.RadError, match="window_type"):
        binding.Detector(w.dirs, w.omega, w.dt, window=(7, (0, 0, 0), (1, 1, 1)))
    with pytest.raises(binding.RadError, match="finite"):
        binding.Detector(w.dirs, w.omega, w.dt, window=("hamming", (0, float("nan"), 0), (1, 1, 1)))
    S0, _ = P.run_gpu(w, [(t, st)])
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, window=("triangle", (0, 0, 0), (0, -1, 0))) as det:
        det.accumulate_step(t, P.to_device(st))          # no axis windowed -> identity
        assert np.array_equal(det.spectrum(), S0)


@pytest.mark.parametrize("D,W,dtype,nu", [(6, 300, np.float32, 0.5), (33, 64, np.float32, 1.0), (4, 1024, np.float64, 0.25),
                                          (1, 8, np.float32, 0.5)])
def test_nyquist_limiter(oracle_mod, D, W, dtype, nu):
    """NEXT-3 Nyquist limiter (rad.h, reading N1): at dt = 1e-17 s and w up to 1e18 rad/s the
    cut-off pi nu / (dt (1 - beta.n)) falls inside the grid and differs per particle and
    direction (beta_x = +-0.2 streams); the GPU must take the same keep/drop decisions as the
    oracle (fp64 on both sides), so the usual tolerances apply to every bin."""
    from paper_2501_03383_b200 import binding
    w = wl.Workload("nyq", 2000, 3, 1e-17, wl.dirs_fibonacci(D), wl.omega_log(W), dtype, wl.BASE_SEED + 50, "khi")
    steps = list(w.steps())
    o = oracle_mod.Oracle(w.dirs, w.omega, w.dt, scale=1.0, nyquist=nu)
    for t, st in steps:
        o.accumulate_step(t, *st)
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, state_dtype=dtype, nyquist=nu) as det:
        for t, st in steps:
            det.accumulate_step(t, P.to_device(st))
        S, variant = det.spectrum(), det.kernel_variant
    assert variant == "general+nyquist"
    ref = o.spectrum()
    plain = P.run_oracle(oracle_mod, w, steps).spectrum()
    assert np.array_equal(ref[:, 0], plain[:, 0]) and not np.allclose(ref[:, -1], plain[:, -1], rtol=1e-3)
    # bins every particle is cut from are exactly zero on both sides
    dead = ref == 0.0
    assert np.array_equal(S == 0.0, dead)
    l2, mr = P.assert_parity(S, ref, what=f"nyquist {D}x{W}")
    for d in range(D):
        P.assert_parity(S[d], ref[d], what=f"nyquist dir {d}")
    print(f"nyquist {D}x{W} nu={nu}: dead bins {int(dead.sum())}, relL2={l2:.2e} maxrel={mr:.2e}")


def test_nyquist_linear_grid_regions_and_errors(oracle_mod):
    from paper_2501_03383_b200 import binding
    # a linear grid with the limiter on runs the general kernel (no recurrence variant)
    w = wl.Workload("nyq", 1500, 2, 1e-17, wl.dirs_fibonacci(5), np.linspace(1e16, 9e17, 160), np.float32,
                    wl.BASE_SEED + 51, "khi")
    steps = list(w.steps())
    off = np.array([0, 400, 1500], dtype=np.int64)
    o = oracle_mod.RegionOracle(2, w.dirs, w.omega, w.dt, scale=1.0, nyquist=0.7)
    for t, st in steps:
        o.accumulate_step(t, off, *st)
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, n_regions=2, nyquist=0.7) as det:
        for t, st in steps:
            det.accumulate_step_regions(t, off, P.to_device(st))
        assert det.kernel_variant == "general+nyquist"
        for r in range(2):
            P.assert_parity(det.spectrum()[r], o.spectrum()[r], what=f"nyquist region {r}")
    with pytest.raises(binding.RadError, match="nyquist_factor"):
        binding.Detector(w.dirs, w.omega, w.dt, nyquist=-1.0)


@pytest.mark.parametrize("cfg,n", [("3c", 2000), ("4b", 6000), ("0", 256)])
def test_calls_are_cuda_graph_capturable(oracle_mod, cfg, n):
    """Steady-state calls (accumulate on device state, spectrum to a device buffer) do no
    allocation and no synchronisation, so a caller can capture a block of steps in a CUDA graph
    and replay it (the remedy for launch-bound small steps when the state is produced on the
    fly); the replayed graph must give the oracle's spectrum."""
    import torch
    from paper_2501_03383_b200 import binding
    w = wl.make_workload(cfg)
    steps = list(w.steps(n_steps=4, n_particles=n))
    dev = [P.to_device(st) for _, st in steps]
    out = torch.zeros(w.n_dir, w.n_omega, dtype=torch.float64, device="cuda")
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, state_dtype=w.state_dtype) as det:
        det.accumulate_step(0, dev[0])          # warm-up outside the capture (lazy set-up paths)
        det.spectrum(out=out)
        det.reset()
        torch.cuda.synchronize()
        side = torch.cuda.Stream()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.stream(side):
            with torch.cuda.graph(g, stream=side):
                for i, (t, _) in enumerate(steps):
                    det.accumulate_step(t, dev[i])
                det.spectrum(out=out)
        torch.cuda.synchronize()
        det.reset()
        torch.cuda.synchronize()
        g.replay()
        torch.cuda.synchronize()
        S = out.cpu().numpy()
    ref = P.run_oracle(oracle_mod, w, steps).spectrum()
    P.assert_parity(S, ref, what=f"graph replay cfg{cfg}")


def test_checkpoint_resume_through_amplitude_export(oracle_mod):
    """SURVEY section 5 (checkpoint / resume): the whole state of a detector is its amplitude.
    Export it after two steps (rad_amplitude to the host), start a fresh handle, import it
    (rad_add_amplitude) and continue: same spectrum as the uninterrupted run and the oracle."""
    import torch
    from paper_2501_03383_b200 import binding
    w = wl.make_workload("3b")
    steps = list(w.steps(n_steps=4, n_particles=1200))
    ref = P.run_oracle(oracle_mod, w, steps).spectrum()
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0) as a:
        for t, st in steps[:2]:
            a.accumulate_step(t, P.to_device(st))
        ckpt = a.amplitude()                                  # numpy complex [D, W, 3] on the host
    saved = np.stack([ckpt.real, ckpt.imag], axis=-1).copy()  # what a checkpoint file would hold
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0) as b:
        b.add_amplitude(torch.from_numpy(saved).cuda())
        for t, st in steps[2:]:
            b.accumulate_step(t, P.to_device(st))
        S_resumed = b.spectrum()
    S_straight, _ = P.run_gpu(w, steps)
    assert P.rel_l2(S_resumed, S_straight) < 1e-12 + 1e-7
    P.assert_parity(S_resumed, ref, what="resumed run")


@pytest.mark.skipif(__import__("os").environ.get("RAD_SLOW") != "1",
                    reason="~10 min: the whole production-like config; run with RAD_SLOW=1")
def test_cfg2_full_workload_all_2000_steps(oracle_mod):
    """BASELINE.json configs[2] in full (1 048 576 particles x 2000 steps x 256 x 1024 bins =
    5.5e14 updates on the GPU); the oracle follows on 12 stratified bins (2.5e10 updates)."""
    w = wl.make_workload("2")
    _full_size_sampled(oracle_mod, "2", 2000, P.stratified_bins(w.n_dir, w.n_omega, 3, 4), flag_sets=(0,),
                       check_argmax=False)


@pytest.mark.parametrize("cfg,n", [("5r", 40000), ("3c", 9000), ("4b", 50000), ("0", 256), ("3d", 3000)])
def test_overlap_steps_flag_keeps_every_intermediate_spectrum(oracle_mod, cfg, n):
    """RAD_FLAG_OVERLAP_STEPS (programmatic dependent launches): kernels of consecutive calls
    overlap, so the spectrum taken after step i must still contain steps 0..i and nothing of
    step i+1 (the accumulate kernels wait before their fold, the result kernels before they
    read A).  Every intermediate spectrum is compared with a run without the flag, the last one
    with the oracle; many short steps back to back make the overlap real."""
    import torch
    from paper_2501_03383_b200 import binding
    w = wl.make_workload(cfg)
    T = 12
    steps = list(w.steps(n_steps=T, n_particles=n))
    dev = [P.to_device(st) for _, st in steps]
    R = w.n_regions
    off = w.region_offsets(n) if R > 1 else None

    def run(flags):
        outs = [torch.zeros(R * w.n_dir, w.n_omega, dtype=torch.float64, device="cuda") for _ in range(T)]
        with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, state_dtype=w.state_dtype, flags=flags,
                              n_regions=R if R > 1 else 0) as det:
            for rep in range(2):                      # second pass: everything warm, launches back to back
                det.reset()
                for i, (t, _) in enumerate(steps):
                    if R > 1:
                        det.accumulate_step_regions(t, off, dev[i])
                    else:
                        det.accumulate_step(t, dev[i])
                    det.spectrum(out=outs[i])
            torch.cuda.synchronize()
        return [o.cpu().numpy() for o in outs]

    plain, over = run(0), run(binding.RAD_FLAG_OVERLAP_STEPS)
    # GPU vs GPU: a step missing from (or leaking into) a spectrum changes it by O(1/T); rounding
    # differences between two runs are ~1e-7 (fp32 partial sums whose grouping depends on timing:
    # fp64 atomics everywhere, work-stealing tile shares in the streaming kernel)
    for i in range(T):
        assert np.allclose(over[i], plain[i], rtol=2e-5, atol=1e-9 * plain[-1].max()), f"step {i}"
    if R > 1:
        o = oracle_mod.RegionOracle(R, w.dirs, w.omega, w.dt, scale=1.0)
        for t, st in steps:
            o.accumulate_step(t, off, *st)
        ref = o.spectrum().reshape(R * w.n_dir, w.n_omega)
    else:
        ref = P.run_oracle(oracle_mod, w, steps).spectrum()
    for r in range(R):
        sl = slice(r * w.n_dir, (r + 1) * w.n_dir)
        P.assert_parity(over[-1][sl], ref[sl], what=f"overlap cfg{cfg} region {r}")


@pytest.mark.parametrize("shape", ["general", "uniform", "stream", "regions"])
def test_overlap_plus_deterministic_is_bit_identical_to_deterministic(oracle_mod, shape):
    """include/rad.h: RAD_FLAG_OVERLAP_STEPS "combines with RAD_FLAG_DETERMINISTIC (results stay
    bit-identical)".  12 short steps back to back, a spectrum after every step, on the general,
    uniform, streaming and per-region handles: every intermediate spectrum of the
    OVERLAP|DETERMINISTIC run equals the DETERMINISTIC run's bit for bit (the workspace of step
    i+1 must not be written before step i's reduction has read it), the last one meets the oracle."""
    import torch
    from paper_2501_03383_b200 import binding
    R, n, T = 1, 20000, 12
    if shape == "general":
        dirs, omega = wl.dirs_fibonacci(6), wl.omega_log(96)
    elif shape == "uniform":
        dirs, omega = wl.dirs_fibonacci(6), np.linspace(2e14, 6e16, 96)
    elif shape == "stream":
        dirs, omega, n = wl.dirs_fibonacci(2)[:1], wl.omega_log(8), 60000
    else:
        dirs, omega, R = wl.dirs_fibonacci(3), wl.omega_log(64), 4
    w = wl.Workload("detov", n, T, 1e-17, dirs, omega, np.float32, wl.BASE_SEED + 70, "khi")
    steps = list(w.steps())
    dev = [P.to_device(st) for _, st in steps]
    off = np.array([0, n // 7, n // 7, n // 2, n], dtype=np.int64) if R > 1 else None

    def run(flags):
        outs = [torch.zeros(R * w.n_dir, w.n_omega, dtype=torch.float64, device="cuda") for _ in range(T)]
        with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, flags=flags, n_regions=R if R > 1 else 0) as det:
            for rep in range(2):
                det.reset()
                torch.cuda.synchronize()
                for i, (t, _) in enumerate(steps):
                    if R > 1:
                        det.accumulate_step_regions(t, off, dev[i])
                    else:
                        det.accumulate_step(t, dev[i])
                    det.spectrum(out=outs[i])
            torch.cuda.synchronize()
            variant = det.kernel_variant
        return [o.cpu().numpy() for o in outs], variant

    det_only, v0 = run(binding.RAD_FLAG_DETERMINISTIC)
    both, v1 = run(binding.RAD_FLAG_DETERMINISTIC | binding.RAD_FLAG_OVERLAP_STEPS)
    assert v0 == v1 == ("general" if shape == "regions" else shape)
    for i in range(T):
        assert np.array_equal(both[i], det_only[i]), f"step {i} differs"
    if R > 1:
        o = oracle_mod.RegionOracle(R, w.dirs, w.omega, w.dt, scale=1.0)
        for t, st in steps:
            o.accumulate_step(t, off, *st)
        ref = o.spectrum().reshape(R * w.n_dir, w.n_omega)
    else:
        ref = P.run_oracle(oracle_mod, w, steps).spectrum()
    for r in range(R):
        sl = slice(r * w.n_dir, (r + 1) * w.n_dir)
        if ref[sl].max() > 0:
            P.assert_parity(both[-1][sl], ref[sl], what=f"overlap+deterministic {shape} region {r}")


@pytest.mark.parametrize("regions", [False, True])
def test_e2e_call_sequence_every_step_spectrum_matches_oracle(oracle_mod, regions):
    """bench.py's `e2e` leg, call for call: RAD_FLAG_OVERLAP_STEPS handle, state in pinned HOST
    memory through rad_accumulate_step(_regions)_host, every step's spectrum delivered to one of
    two pinned host buffers with RAD_OUT_HOST_ASYNC, the host one step behind on an event.  EVERY
    step's host spectrum (the running sum up to that step) is compared with the oracle's."""
    import torch
    from paper_2501_03383_b200 import binding
    R = 3 if regions else 1
    n, T = 30000, 8
    w = wl.Workload("e2e", n, T, 1e-17, wl.dirs_fibonacci(16), wl.omega_log(128), np.float32, wl.BASE_SEED + 71, "khi")
    steps = list(w.steps())
    host = [[torch.from_numpy(a).pin_memory() for a in st] for _, st in steps]
    off = np.array([0, 9000, 9001, n], dtype=np.int64) if regions else None
    o = (oracle_mod.RegionOracle(R, w.dirs, w.omega, w.dt, scale=1.0) if regions
         else oracle_mod.Oracle(w.dirs, w.omega, w.dt, scale=1.0))
    refs = []
    for t, st in steps:
        o.accumulate_step(t, *([off] if regions else []), *st)
        refs.append(o.spectrum().reshape(R * w.n_dir, w.n_omega).copy())
    got = [None] * T
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, flags=binding.RAD_FLAG_OVERLAP_STEPS,
                          n_regions=R if regions else 0) as det:
        pinned = [torch.empty(R * w.n_dir, w.n_omega, dtype=torch.float64).pin_memory() for _ in range(2)]
        arrived = [torch.cuda.Event(), torch.cuda.Event()]
        for i, (t, _) in enumerate(steps):
            if regions:
                det.accumulate_step_regions_host(t, off, host[i])
            else:
                det.accumulate_step_host(t, host[i])
            b = i & 1
            det.spectrum(out=pinned[b])          # RAD_OUT_HOST_ASYNC
            arrived[b].record()
            if i > 0:
                arrived[b ^ 1].synchronize()
                got[i - 1] = pinned[b ^ 1].numpy().copy()
        arrived[(T - 1) & 1].synchronize()
        got[T - 1] = pinned[(T - 1) & 1].numpy().copy()
    for i in range(T):
        for r in range(R):
            sl = slice(r * w.n_dir, (r + 1) * w.n_dir)
            P.assert_parity(got[i][sl], refs[i][sl], what=f"e2e sequence step {i} region {r}")


# ------------------------------------------------- macro-particle form factor (reading FF1)
@pytest.mark.parametrize("kind,size", [("gaussian", (3e-8, 1e-8, 2e-8)), ("cic", (6e-8, 6e-8, 3e-8)),
                                        ("incoherent", (0.0, 0.0, 0.0))])
@pytest.mark.parametrize("shape", ["general", "uniform", "stream", "regions", "nyquist"])
def test_form_factor(oracle_mod, kind, size, shape):
    """NEXT-3 macro-particle form factor (rad.h, reading FF1; "correctly quantify
    coherent and incoherent radiation [39]"): g = sqrt(w + (w^2 - w) F^2(n, w_j)) per update, through
    every accumulate kernel; macro weights log-uniform in [1, 1e4), shape sizes chosen so that F
    passes from 1 to 0 inside the frequency grid; fp32 state."""
    from paper_2501_03383_b200 import binding
    ff = (kind, size)
    kw = {}
    if shape == "uniform":
        dirs, omega = wl.dirs_fibonacci(6), np.linspace(2e14, 6e16, 128)
    elif shape == "stream":
        dirs, omega = wl.dirs_fibonacci(2), wl.omega_log(8, 1e15, 1e17)
    elif shape == "nyquist":
        dirs, omega, kw = wl.dirs_fibonacci(5), wl.omega_log(96), {"nyquist": 0.5}
    else:
        dirs, omega = wl.dirs_fibonacci(5), wl.omega_log(96)
    w = wl.Workload("ff", 3000, 2, 1e-17, dirs, omega, np.float32, wl.BASE_SEED + 80, "khi", extra={"weights": 1e4})
    steps = list(w.steps())
    assert steps[0][1][9].max() > 1e3
    if shape == "regions":
        off = np.array([0, 1000, 1000, 3000], dtype=np.int64)
        o = oracle_mod.RegionOracle(3, w.dirs, w.omega, w.dt, scale=1.0, form_factor=ff)
        for t, st in steps:
            o.accumulate_step(t, off, *st)
        with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, n_regions=3, form_factor=ff) as det:
            for t, st in steps:
                det.accumulate_step_regions(t, off, P.to_device(st))
            S = det.spectrum()
        for r in (0, 2):
            P.assert_parity(S[r], o.spectrum()[r], what=f"form factor regions {r}")
        assert np.all(S[1] == 0.0)
        return
    o = oracle_mod.Oracle(w.dirs, w.omega, w.dt, scale=1.0, form_factor=ff, **kw)
    for t, st in steps:
        o.accumulate_step(t, *st)
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, form_factor=ff, **kw) as det:
        for t, st in steps:
            det.accumulate_step(t, P.to_device(st))
        S, variant = det.spectrum(), det.kernel_variant
    want = {"general": "general+formfactor", "uniform": "uniform+formfactor", "stream": "stream",
            "nyquist": "general+nyquist+formfactor"}[shape]
    if kind == "incoherent":    # F = 0 everywhere: g = sqrt(w) is a per-particle weight, the plain kernels serve it
        want = want.replace("+formfactor", "")
    assert P.base_variant(variant) == want
    ref = o.spectrum()
    l2, mr = P.assert_parity(S, ref, what=f"form factor {kind} {shape}")
    for d in range(len(dirs)):
        P.assert_parity(S[d], ref[d], what=f"form factor {kind} {shape} dir {d}")
    plain = oracle_mod.Oracle(w.dirs, w.omega, w.dt, scale=1.0, **kw)
    for t, st in steps:
        plain.accumulate_step(t, *st)
    Sp = plain.spectrum()                                  # the form factor really changes the result:
    assert np.max(np.abs(ref - Sp)[Sp > 0] / Sp[Sp > 0]) > 0.5   # incoherent bins drop by up to w (relL2 only sees the coherent peak)
    print(f"form factor {kind}/{shape}: relL2={l2:.2e} maxrel={mr:.2e}")


def test_form_factor_identities_and_argument_errors(oracle_mod):
    """w = 1: any shape is the identity (same spectrum as a handle without form factor, to fp32
    rounding of sqrt(1)); zero size = point particle = today's coherent sum; bad arguments."""
    from paper_2501_03383_b200 import binding
    w = wl.make_workload("3c")
    (t, st), = list(w.steps(n_steps=1, n_particles=800))
    S0, _ = P.run_gpu(w, [(t, st)])
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, form_factor=("gaussian", (3e-8, 3e-8, 3e-8))) as det:
        det.accumulate_step(t, P.to_device(st))
        assert P.rel_l2(det.spectrum(), S0) < 1e-6
    stw = st[:9] + [np.full_like(st[9], 37.0)]
    Sw, _ = P.run_gpu(w, [(t, stw)])
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, form_factor=("cic", (0.0, 0.0, 0.0))) as det:
        det.accumulate_step(t, P.to_device(stw))
        assert P.rel_l2(det.spectrum(), Sw) < 1e-6
    with pytest.raises(binding.RadError, match="form_factor_type"):
        binding.Detector(w.dirs, w.omega, w.dt, form_factor=(9, (0, 0, 0)))
    with pytest.raises(binding.RadError, match="form_factor_size"):
        binding.Detector(w.dirs, w.omega, w.dt, form_factor=("gaussian", (1e-8, -1e-8, 0)))
