"""Seeded random differential test: detector shapes, frequency-grid kinds, state dtypes, particle
counts, call forms and options drawn at random, every case compared with the fp64 oracle through the
C ABI with BASELINE.json north_star's tolerances (overall and per direction / region).  Complements
the hand-picked shapes of test_gpu_parity.py: the kernel variant (general / uniform / dyadic / stream /
Nyquist / form factor), the tile shape, the chunk schedule and the padding all follow from
the drawn shape, so combinations nobody wrote down get exercised too."""
import numpy as np
import pytest

from paper_2501_03383_b200 import workloads as wl
from tests import _parity as P

pytestmark = pytest.mark.gpu

L = 10e-6
N_CASES = 120


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    import torch
    from paper_2501_03383_b200 import build
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    build.build()


def _draw(case):
    rng = np.random.default_rng(7700 + case)
    D = int(rng.choice([1, 2, 3, 5, 8, 13, 33, 40]))
    W = int(rng.choice([1, 2, 7, 8, 16, 17, 40, 64, 65, 100, 257, 300, 600]))
    kind = rng.choice(["log", "linear", "dyadic", "random"])
    if kind == "log":
        omega = wl.omega_log(max(W, 2))[:W] * rng.uniform(0.5, 2.0)
    elif kind == "linear":
        omega = np.linspace(rng.uniform(1e14, 5e14), rng.uniform(1e17, 6e17), max(W, 2))[:W]
    elif kind == "dyadic":
        omega = wl.omega_dyadic(W, int(rng.choice([4, 8, 12, 16, 32, 64])), hi=rng.uniform(2e17, 1e18))
    else:
        omega = np.sort(10.0 ** rng.uniform(14, 18, W)) * (1 + 1e-3 * np.arange(W))   # strictly increasing
    dtype = np.float64 if rng.random() < 0.3 else np.float32
    n = int(rng.choice([1, 31, 33, 500, 1000, 2049, 3000]))
    T = int(rng.integers(1, 4))
    t_first = int(rng.choice([0, 1, 250, 900]))
    opts = {}
    r = rng.random()
    if r < 0.15:
        opts["nyquist"] = float(rng.choice([0.3, 0.7, 1.0, 2.5]))
    elif r < 0.30:
        opts["form_factor"] = (str(rng.choice(["gaussian", "cic", "incoherent"])), tuple(rng.uniform(0, 6e-8, 3)))
    elif r < 0.42:
        opts["window"] = (str(rng.choice(["triangle", "hamming"])), (0.1 * L, 0.0, 0.2 * L), (0.7 * L, 0.0, 0.6 * L))
    form = str(rng.choice(["step", "step", "host", "steps", "regions"]))
    flags = int(rng.choice([0, 0, 1, 4, 5, 2]))      # DETERMINISTIC = 1, FORCE_GENERAL = 2, OVERLAP_STEPS = 4
    weights = 1e3 if "form_factor" in opts else None
    # RAD_FLAG_PRECISE = 16 on some of the cases it combines with (its own generator: the other draws stay as they were)
    if "nyquist" not in opts and opts.get("form_factor", ("incoherent",))[0] == "incoherent" \
            and np.random.default_rng(8800 + case).random() < 0.15:
        flags |= 16
    return dict(D=D, W=W, kind=str(kind), omega=omega, dtype=dtype, n=n, T=T, t_first=t_first, opts=opts, form=form,
                flags=flags, weights=weights, seed=int(rng.integers(1, 10 ** 6)))


@pytest.mark.parametrize("case", range(N_CASES))
def test_random_case_matches_oracle(oracle_mod, case):
    import torch
    from paper_2501_03383_b200 import binding
    c = _draw(case)
    extra = {"weights": c["weights"]} if c["weights"] else {}
    w = wl.Workload(f"fuzz{case}", c["n"], c["T"], 1e-17, wl.dirs_fibonacci(max(c["D"], 2))[:c["D"]], c["omega"], c["dtype"],
                    c["seed"], "khi", extra=extra)
    steps = [(c["t_first"] + t, st) for t, st in w.steps()]
    R = 1
    off = None
    if c["form"] == "regions":
        R = 3
        cut = sorted(np.random.default_rng(c["seed"]).integers(0, c["n"] + 1, 2).tolist())
        off = np.array([0, cut[0], cut[1], c["n"]], dtype=np.int64)
    if R > 1:
        o = oracle_mod.RegionOracle(R, w.dirs, w.omega, w.dt, scale=1.0, **c["opts"])
    else:
        o = oracle_mod.Oracle(w.dirs, w.omega, w.dt, scale=1.0, **c["opts"])
    for t, st in steps:
        if R > 1:
            o.accumulate_step(t, off, *st)
        else:
            o.accumulate_step(t, *st)
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, state_dtype=c["dtype"], flags=c["flags"],
                          n_regions=R if R > 1 else 0, **c["opts"]) as det:
        if c["form"] == "regions":
            for t, st in steps:
                det.accumulate_step_regions(t, off, P.to_device(st))
        elif c["form"] == "host":
            for t, st in steps:
                det.accumulate_step_host(t, st)
        elif c["form"] == "steps":
            stacked = [torch.from_numpy(np.stack([st[k] for _, st in steps])).cuda() for k in range(10)]
            det.accumulate_steps(c["t_first"], stacked)
        else:
            devs = [P.to_device(st) for _, st in steps]
            torch.cuda.synchronize()            # RAD_FLAG_OVERLAP_STEPS: inputs complete before the calls
            for (t, _), dev in zip(steps, devs):
                det.accumulate_step(t, dev)
        torch.cuda.synchronize()
        S = det.spectrum()
        variant = det.kernel_variant
    ref = o.spectrum()
    what = (f"fuzz {case}: {c['D']}x{c['W']} {c['kind']} {np.dtype(c['dtype']).name} n={c['n']} T={c['T']} {c['form']} "
            f"flags={c['flags']} {sorted(c['opts'])} -> {variant}")
    assert S.shape == ref.shape, what
    if ref.max() > 0:
        P.assert_parity(S, ref, what=what)
        for k in range(S.reshape(-1, c["W"]).shape[0]):     # every direction (of every region) on its own
            row, rrow = S.reshape(-1, c["W"])[k], ref.reshape(-1, c["W"])[k]
            if rrow.max() > 0:
                # stricter than north_star's criterion: the 1e-6 floor relative to the row's OWN peak; the L2
                # measure only where a row has enough bins to be a spectrum (a 1-bin row's relL2 is its maxrel)
                assert P.max_rel(row, rrow) <= P.MAX_REL_TOL, what + f" row {k}: maxrel {P.max_rel(row, rrow):.3e}"
                if c["W"] >= 16:
                    assert P.rel_l2(row, rrow) <= P.REL_L2_TOL, what + f" row {k}: relL2 {P.rel_l2(row, rrow):.3e}"
            else:
                assert np.all(row == 0.0), what
    else:
        assert np.all(S == 0.0), what
    if ref.max() > 0:
        rows = [(S.reshape(-1, c["W"])[k], ref.reshape(-1, c["W"])[k]) for k in range(S.reshape(-1, c["W"]).shape[0])]
        print(f"{what}: maxrel {P.max_rel(S, ref):.2e} worst row {max(P.max_rel(a, b) for a, b in rows if b.max() > 0):.2e}")
    if "nyquist" in c["opts"]:                              # the keep/drop decision is exact: identical zero sets
        assert np.array_equal(S == 0.0, ref == 0.0), what


@pytest.mark.parametrize("case", range(24))
def test_random_case_fast_gridded_matches_exact_oracle(oracle_mod, case):
    """The approximate fast path (RAD_FLAG_FAST_GRIDDED, default gridding tolerance) on drawn shapes, grids,
    dtypes and step windows against the EXACT oracle with the exact path's tolerances."""
    import torch
    from paper_2501_03383_b200 import binding
    rng = np.random.default_rng(9900 + case)
    D = int(rng.choice([1, 3, 8, 33]))
    W = int(rng.choice([8, 40, 64, 100, 300]))
    kind = str(rng.choice(["log", "linear", "random", "dyadic"]))
    omega = {"log": lambda: wl.omega_log(W) * rng.uniform(0.5, 2.0),
             "linear": lambda: np.linspace(2e14, rng.uniform(1e17, 6e17), W),
             "random": lambda: np.sort(10.0 ** rng.uniform(14, 18, W)) * (1 + 1e-3 * np.arange(W)),
             "dyadic": lambda: wl.omega_dyadic(W, 16, hi=rng.uniform(2e17, 1e18))}[kind]()
    dtype = np.float64 if rng.random() < 0.3 else np.float32
    n, T, t_first = int(rng.choice([33, 1000, 3000])), int(rng.integers(1, 5)), int(rng.choice([0, 40, 700]))
    window = ("hamming", (0.1 * L, 0.0, 0.0), (0.8 * L, 0.0, 0.0)) if rng.random() < 0.25 else None
    w = wl.Workload(f"fuzzfast{case}", n, T, 1e-17, wl.dirs_fibonacci(max(D, 2))[:D], omega, dtype,
                    int(rng.integers(1, 10 ** 6)), "khi")
    steps = [(t_first + t, st) for t, st in w.steps()]
    o = oracle_mod.Oracle(w.dirs, w.omega, w.dt, scale=1.0, window=window)
    for t, st in steps:
        o.accumulate_step(t, *st)
    box = ((-0.02 * L,) * 3, (1.02 * L,) * 3)
    with binding.Detector(w.dirs, w.omega, w.dt, scale=1.0, state_dtype=dtype, flags=binding.RAD_FLAG_FAST_GRIDDED,
                          window=window, fast=(box[0], box[1], t_first, t_first + T - 1, 0.0)) as det:
        for t, st in steps:
            det.accumulate_step(t, P.to_device(st))
        torch.cuda.synchronize()
        S = det.spectrum()
        assert det.kernel_variant == "gridded"
    l2, mr = P.assert_parity(S, o.spectrum(), what=f"fuzz fast {case}: {D}x{W} {kind} {np.dtype(dtype).name} n={n} T={T} t0={t_first}")
    print(f"fuzz fast {case}: {D}x{W} {kind} {np.dtype(dtype).name} n={n} T={T}: relL2 {l2:.2e} maxrel {mr:.2e}")
