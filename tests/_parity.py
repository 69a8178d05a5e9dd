"""Helpers shared by the GPU parity tests: error metrics (SURVEY.md Q13 / BASELINE.json
north_star tolerances) and runners that feed the SAME seeded arrays to both sides."""
import numpy as np

REL_L2_TOL = 1e-4      # north_star: relative L2 error <= 1e-4 on the spectrum
MAX_REL_TOL = 1e-3     # north_star: max relative error <= 1e-3 on bins above 1e-6 of the peak
PEAK_FLOOR = 1e-6


def rel_l2(S, S_ref):
    S, S_ref = np.asarray(S, float).ravel(), np.asarray(S_ref, float).ravel()
    den = np.linalg.norm(S_ref)
    return float(np.linalg.norm(S - S_ref) / den) if den > 0 else float(np.linalg.norm(S))


def max_rel(S, S_ref, peak=None):
    """max |S-S_ref|/S_ref over bins with S_ref >= 1e-6 * peak (peak defaults to max S_ref)."""
    S, S_ref = np.asarray(S, float).ravel(), np.asarray(S_ref, float).ravel()
    peak = float(S_ref.max()) if peak is None else float(peak)
    m = S_ref >= PEAK_FLOOR * peak
    if not m.any():
        return 0.0
    return float(np.max(np.abs(S[m] - S_ref[m]) / S_ref[m]))


def assert_parity(S, S_ref, peak=None, what=""):
    l2, mr = rel_l2(S, S_ref), max_rel(S, S_ref, peak)
    assert np.all(np.isfinite(S)), f"{what}: non-finite spectrum"
    assert l2 <= REL_L2_TOL, f"{what}: relL2 {l2:.3e} > {REL_L2_TOL}"
    assert mr <= MAX_REL_TOL, f"{what}: maxrel {mr:.3e} > {MAX_REL_TOL}"
    return l2, mr


def base_variant(v):
    """Kernel variant name without the "+split" suffix (few-direction detectors: lane groups of a warp
    share a direction and split the particles; same sweep, same results)."""
    return v.replace("+split", "")


def to_device(state):
    import torch
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in state]


def run_gpu(workload, steps, scale=1.0, flags=0, host=False, want_amplitude=False):
    """steps: list of (t, state arrays).  Returns spectrum (and amplitude) as numpy."""
    import torch
    from paper_2501_03383_b200 import binding
    with binding.Detector(workload.dirs, workload.omega, workload.dt, t0=workload.t0, scale=scale,
                          state_dtype=workload.state_dtype, flags=flags) as det:
        for t, st in steps:
            if host:
                det.accumulate_step_host(t, st)
            else:
                det.accumulate_step(t, to_device(st))
        torch.cuda.synchronize()
        S = det.spectrum()
        A = det.amplitude() if want_amplitude else None
        variant = det.kernel_variant
    return (S, A, variant) if want_amplitude else (S, variant)


def run_oracle(oracle_mod, workload, steps, scale=1.0, bins=None):
    o = oracle_mod.Oracle(workload.dirs, workload.omega, workload.dt, t0=workload.t0, scale=scale, bins=bins)
    for t, st in steps:
        o.accumulate_step(t, *st)
    return o


def stratified_bins(D, W, n_dir=4, n_om=8, extra=()):
    """Flat indices of a stratified subset of bins incl. the first and last frequency."""
    ds = np.unique(np.linspace(0, D - 1, min(n_dir, D)).round().astype(int))
    js = np.unique(np.linspace(0, W - 1, min(n_om, W)).round().astype(int))
    flat = (ds[:, None] * W + js[None, :]).ravel()
    return np.unique(np.concatenate([flat, np.asarray(extra, dtype=np.int64)])).astype(np.int64)


def tile_cover_bins(D, W, block=32, n_random=0, seed=1, extra=()):
    """Flat indices of a bin sample that reaches every warp tile of the accumulate kernels: in
    EVERY direction, one bin (seeded random position) in every block of `block` consecutive
    frequencies -- a warp tile is 32/lw directions x lw*8 frequencies with lw in {4, 8, 16, 32},
    i.e. >= 1 direction x >= 32 frequencies, so block = 32 puts a sample into every (direction
    group, frequency tile) pair whatever tile shape rad_create picked (block = 64 does for
    lw >= 8).  Plus `n_random` bins drawn uniformly, the first and last frequency of the first
    and last direction, and `extra` (e.g. the GPU arg-max bin)."""
    rng = np.random.default_rng(seed)
    starts = np.arange(0, W, block)
    width = np.minimum(block, W - starts)
    pos = starts[None, :] + (rng.random((D, starts.shape[0])) * width[None, :]).astype(np.int64)
    flat = (np.arange(D, dtype=np.int64)[:, None] * W + pos).ravel()
    rnd = rng.integers(0, D * W, size=n_random, dtype=np.int64)
    corners = np.array([0, W - 1, (D - 1) * W, D * W - 1], dtype=np.int64)
    return np.unique(np.concatenate([flat, rnd, corners, np.asarray(extra, dtype=np.int64)])).astype(np.int64)
