"""Seeded input generators (paper_2501_03383_b200/workloads.py): determinism and physics sanity."""
import numpy as np
import pytest

from paper_2501_03383_b200 import workloads as wl


def test_rng_is_counter_based_and_prefix_stable():
    a = wl.uniform01(7, 3, 1000)
    b = wl.uniform01(7, 3, 10)
    c = wl.uniform01(7, 3, 10, offset=990)
    assert np.array_equal(a[:10], b) and np.array_equal(a[990:], c)
    assert 0.0 < a.min() and a.max() < 1.0
    assert abs(a.mean() - 0.5) < 0.05
    g = wl.normal01(7, 5, 20000)
    assert abs(g.mean()) < 0.03 and abs(g.std() - 1.0) < 0.03
    assert not np.array_equal(wl.uniform01(7, 4, 10), b)
    assert not np.array_equal(wl.uniform01(8, 3, 10), b)


def test_grids():
    for d in (wl.dirs_fibonacci(256), wl.dirs_seeded_uniform(8, 1)):
        assert np.allclose(np.linalg.norm(d, axis=1), 1.0, atol=1e-14)
    assert np.abs(wl.dirs_fibonacci(1024).mean(axis=0)).max() < 2e-3
    om = wl.omega_log(512)
    assert om[0] == 1e14 and om[-1] == pytest.approx(1e18, rel=1e-12) and np.all(np.diff(om) > 0)
    assert np.allclose(om[1:] / om[:-1], om[1] / om[0], rtol=1e-12)
    dy = wl.omega_dyadic(100, 8)
    assert dy[-1] == 1e18 and np.all(np.diff(dy) > 0) and np.array_equal(dy[8:], 2.0 * dy[:-8])
    assert np.allclose(dy[1:] / dy[:-1], 2.0 ** 0.125, rtol=1e-14)
    lin = wl.omega_linear(64, 4e14)
    assert lin[0] == pytest.approx(6.25e12) and lin[-1] == pytest.approx(4e14)


@pytest.mark.parametrize("cfg", wl.ALL_CONFIGS)
def test_config_shapes(cfg):
    w = wl.make_workload(cfg)
    sizes = {"0": (256, 128, 8, 64), "1": (65536, 1000, 128, 512), "2": (1048576, 2000, 256, 1024),
             "3a": (262144, 200, 16, 4096), "3b": (262144, 200, 64, 1024),
             "3c": (262144, 200, 256, 256), "3d": (262144, 200, 1024, 64),
             "4": (16777216, 4, 16, 128), "4b": (16777216, 4, 1, 8),
             "5r": (331776, 200, 1, 512), "1u": (65536, 1000, 128, 512),
             "1f": (65536, 1000, 128, 512), "1n": (65536, 1000, 128, 512), "1d": (65536, 1000, 128, 512), "5s": (331776, 200, 1, 128), "1p": (65536, 1000, 128, 512)}[cfg]
    assert (w.n_particles, w.n_steps, w.n_dir, w.n_omega) == sizes
    assert w.state_dtype == (np.float64 if cfg == "0" else np.float32)


def test_helix_state_is_self_consistent():
    w = wl.make_workload("0")
    st = {t: s for t, s in w.steps(n_steps=3)}
    assert all(a.dtype == np.float64 and a.shape == (256,) for a in st[0])
    # central difference of r over 2 dt == c beta at the middle step (to O(dt^2))
    for c in range(3):
        v = (st[2][c] - st[0][c]) / (2 * w.dt) / wl.C_LIGHT
        assert np.allclose(v, st[1][3 + c], atol=1e-4)
        bd = (st[2][3 + c] - st[0][3 + c]) / (2 * w.dt)
        assert np.allclose(bd, st[1][6 + c], atol=1e-3 * 1e13)
    assert np.allclose(st[0][3] ** 2 + st[0][4] ** 2, 0.01) and np.all(st[0][5] == 0.05)
    assert np.all(st[0][0] >= 0) and np.all(st[0][0] < 1e-6)


def test_khi_state_physics_and_determinism():
    w = wl.make_workload("1")
    steps = list(w.steps(n_steps=4, n_particles=4096))
    again = list(w.steps(n_steps=4, n_particles=1024))
    for (t, a), (_, b) in zip(steps, again):
        assert all(x.dtype == np.float32 for x in a)
        assert all(np.array_equal(x[:1024], y) for x, y in zip(a, b))   # particle i fixed
    src = wl.KHISource(4096, w.seed, w.dt)
    s0 = [a.copy() for a in src.state()]
    b2_0 = s0[3] ** 2 + s0[4] ** 2 + s0[5] ** 2
    for _ in range(50):
        src.advance()
    s1 = src.state()
    b2_1 = s1[3] ** 2 + s1[4] ** 2 + s1[5] ** 2
    assert np.allclose(b2_0, b2_1, rtol=1e-12)                            # Boris conserves |beta|
    assert np.allclose(s1[3] * s1[6] + s1[4] * s1[7], 0.0, atol=1e-3)     # betadot _|_ beta
    top = s0[1] < 0.5 * 10e-6
    assert abs(s0[3][top].mean() - 0.2) < 2e-3 and abs(s0[3][~top].mean() + 0.2) < 2e-3
    # r advanced by c beta dt
    src2 = wl.KHISource(16, w.seed, w.dt)
    r0 = src2.r.copy()
    src2.advance()
    assert np.allclose(src2.r - r0, wl.C_LIGHT * w.dt * src2.b, rtol=1e-5, atol=0)
    # |betadot| = |q B/(gamma m)| |beta_perp|
    k = np.abs(src2.qm * src2._Bz())
    st = src2.state()
    assert np.allclose(np.hypot(st[6], st[7]), k * np.hypot(st[3], st[4]), rtol=1e-12)


def test_cfg0_oracle_regression_fixture(oracle_mod):
    """The committed oracle spectrum of config 0 (written by tests/golden/make_cfg0_golden.py,
    which calls only oracle/) still comes out of the oracle: guards against silent edits."""
    from pathlib import Path
    gold = np.loadtxt(Path(__file__).parent / "golden" / "cfg0_oracle_spectrum.txt")
    w = wl.make_workload("0")
    o = oracle_mod.Oracle(w.dirs, w.omega, w.dt, scale=1.0)
    for t, st in w.steps():
        o.accumulate_step(t, *st)
    assert np.allclose(o.spectrum(), gold, rtol=1e-12, atol=0)


def test_region_workload_is_sorted_by_sub_volume():
    """cfg 5r: particles come sorted by the (2 x 6) x-y box of their initial position and the
    offsets partition them; the unsorted generator yields the same particle set."""
    w = wl.make_workload("5r")
    assert w.n_regions == 12
    n = 6000
    off = w.region_offsets(n)
    assert off.shape == (13,) and off[0] == 0 and off[-1] == n and np.all(np.diff(off) > 0)
    (_, st), = list(w.steps(n_steps=1, n_particles=n))
    L = 10e-6
    rid = np.minimum((st[0].astype(np.float64) / L * 2).astype(int), 1) * 6 + \
        np.minimum((st[1].astype(np.float64) / L * 6).astype(int), 5)
    assert np.all(np.diff(rid) >= 0)
    for r in range(12):
        assert np.all(rid[off[r]:off[r + 1]] == r)
    plain = wl.Workload("p", n, 1, w.dt, w.dirs, w.omega, np.float32, w.seed, "khi")
    (_, st0), = list(plain.steps())
    assert np.array_equal(np.sort(st0[0]), np.sort(st[0]))
    assert wl.make_workload("1").n_regions == 1
    assert np.array_equal(wl.make_workload("1").region_offsets(10), [0, 10])
