"""rad_spectrum_static (include/rad.h): the allocation-free one-call detector, whose fp64 amplitude
accumulator is a static __device__ array inside librad.so, against the existing handle-based path
(rad_create / rad_accumulate_steps / rad_spectrum) on the same device arrays, with BASELINE.json
north_star's tolerances (tests/_parity.py), on calls in a row that share the array: a larger detector
first, then a smaller one whose bins overlap the first call's leftovers, then the first again, then one of
exactly the maximum size.
Named test_zz_* so that pytest collects it last (the round's end runs pytest -x)."""
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


def _case(D, W, kind, dtype, n, T, seed):
    omega = wl.omega_log(W) if kind == "log" else np.linspace(2e14, 4e17, W)
    return wl.Workload(f"static{seed}", n, T, 1e-17, wl.dirs_fibonacci(max(D, 2))[:D], omega, dtype, seed, "khi")


def _both_paths(w, t_first, scale=1.0, check_free_memory=False):
    """-> (spectrum of the existing path, spectrum of rad_spectrum_static), both numpy [D, W].
    check_free_memory (for a call whose kernels are loaded already): cudaMemGetInfo's free bytes do not drop."""
    import torch
    from paper_2501_03383_b200 import binding
    steps = [st for _, st in w.steps()]
    T, n = len(steps), steps[0][0].shape[0]
    stacked = [torch.from_numpy(np.stack([st[k] for st in steps])).cuda() for k in range(10)]
    D, W = w.dirs.shape[0], w.omega.shape[0]
    code = {np.dtype(np.float32): binding.RAD_F32, np.dtype(np.float64): binding.RAD_F64}[np.dtype(w.state_dtype)]
    with binding.Detector(w.dirs, w.omega, w.dt, t0=w.t0, scale=scale, state_dtype=w.state_dtype) as det:
        det.accumulate_steps(t_first, stacked)
        torch.cuda.synchronize()
        S_ref = det.spectrum()
    dirs_d = torch.from_numpy(np.ascontiguousarray(w.dirs, dtype=np.float64)).cuda()
    omega_d = torch.from_numpy(np.ascontiguousarray(w.omega, dtype=np.float64)).cuda()
    out = torch.full((D, W), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    binding.rad_spectrum_static(D, dirs_d.data_ptr(), W, omega_d.data_ptr(), w.dt, w.t0, scale, code, t_first, T, n, n,
                                [a.data_ptr() for a in stacked], out.data_ptr(),
                                int(torch.cuda.current_stream().cuda_stream))
    torch.cuda.synchronize()
    if check_free_memory:
        assert torch.cuda.mem_get_info()[0] >= free_before, "rad_spectrum_static took device memory"
    return S_ref, out.cpu().numpy()


def test_static_scratch_entry_matches_existing_path_on_calls_in_a_row(oracle_mod):
    big = _case(13, 300, "log", np.float32, 3000, 3, 4101)       # ragged chunk tail (3000 = 5 * 512 + 440), 3 bin sweeps
    small = _case(3, 40, "linear", np.float64, 700, 2, 4102)    # its 120 bins lie inside the first call's 3900
    limit = _case(128, 512, "log", np.float32, 1100, 1, 4104)   # n_dir * n_omega = RAD_STATIC_MAX_BINS exactly
    results = []
    for call, (w, t_first) in enumerate(((big, 0), (small, 250), (big, 0), (limit, 900))):
        S_ref, S = _both_paths(w, t_first, check_free_memory=call >= 2)
        assert S.shape == S_ref.shape and S_ref.max() > 0
        l2, mr = P.assert_parity(S, S_ref, what=f"rad_spectrum_static {w.name} vs existing path")
        print(f"rad_spectrum_static {w.name} {S.shape}: relL2 {l2:.2e} maxrel {mr:.2e} against the existing path")
        results.append(S)
    # the same inputs again after another detector used the array: the same spectrum (up to the order of the atomics)
    P.assert_parity(results[2], results[0], what="rad_spectrum_static repeated call")
    # and against the fp64 oracle, the tolerance every other path is held to
    o = P.run_oracle(oracle_mod, small, [(250 + t, st) for t, st in small.steps()])
    P.assert_parity(results[1], o.spectrum(), what="rad_spectrum_static vs oracle")


@pytest.mark.parametrize("case", range(10))
def test_static_scratch_entry_drawn_shapes(case):
    """Drawn detector shapes (one bin, one direction, bin counts around the 128-lane tile), particle counts around the
    512-particle chunk, both state dtypes, the SI default scale: against the existing path."""
    rng = np.random.default_rng(6600 + case)
    D = int(rng.choice([1, 2, 5, 40]))
    W = int(rng.choice([1, 3, 17, 64, 127, 129, 300]))
    n = int(rng.choice([1, 31, 512, 513, 1500]))
    T = int(rng.integers(1, 4))
    dtype = np.float64 if case % 2 else np.float32
    w = _case(D, max(W, 2), str(rng.choice(["log", "linear"])), dtype, n, T, 6600 + case)
    w.omega = w.omega[:W]
    scale = 0.0 if case % 3 == 0 else 1.0
    S_ref, S = _both_paths(w, int(rng.choice([0, 40, 900])), scale=scale)
    assert S.shape == (D, W) and S_ref.max() > 0
    what = f"rad_spectrum_static drawn case {case}: {D}x{W} n={n} T={T} {np.dtype(dtype).name}"
    l2, mr = P.assert_parity(S, S_ref, what=what)
    print(f"{what}: relL2 {l2:.2e} maxrel {mr:.2e} worst direction {max(P.max_rel(S[k], S_ref[k]) for k in range(D)):.2e}")
    for k in range(D):                                   # every direction on its own (its own peak)
        assert P.max_rel(S[k], S_ref[k]) <= P.MAX_REL_TOL, f"case {case} direction {k}"


def test_static_scratch_entry_empty_input_and_limits():
    import torch
    from paper_2501_03383_b200 import binding
    w = _case(2, 8, "log", np.float32, 33, 1, 4103)
    dirs_d = torch.from_numpy(np.ascontiguousarray(w.dirs)).cuda()
    omega_d = torch.from_numpy(np.ascontiguousarray(w.omega)).cuda()
    out = torch.full((2, 8), float("nan"), dtype=torch.float64, device="cuda")
    args = lambda D, W, n: (D, dirs_d.data_ptr(), W, omega_d.data_ptr(), w.dt, 0.0, 1.0, binding.RAD_F32, 0, 1, n, n,
                            [0] * 10, out.data_ptr(), 0)
    binding.rad_spectrum_static(*args(2, 8, 0))          # no particles: the spectrum is zero (the array was cleared)
    torch.cuda.synchronize()
    assert np.all(out.cpu().numpy() == 0.0)
    with pytest.raises(binding.RadError) as ei:           # beyond the static array: a clear error, nothing launched
        binding.rad_spectrum_static(*args(257, 256, 0))
    assert ei.value.status == binding.RAD_ERR_UNSUPPORTED and "RAD_STATIC_MAX_BINS" in str(ei.value)
    with pytest.raises(binding.RadError) as ei:
        binding.rad_spectrum_static(*args(2, 8, 5))      # particles but NULL arrays
    assert ei.value.status == binding.RAD_ERR_INVALID_ARG
