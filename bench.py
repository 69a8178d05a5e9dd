#!/usr/bin/env python
"""bench.py -- throughput of the radiation-detector hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl ours|reference]

A "step" is one pass of the whole hot path over one PIC step of synthetic input:
rad_accumulate_step (stage + accumulate + fold) followed by
rad_spectrum (a4).  Metric (BASELINE.json): particle*direction*frequency updates per second,
in G/s, whole job.  Headline workload = BASELINE.json configs[2] ("production-like": 1 048 576
electrons x 256 directions x 1024 log-spaced frequencies, fp32 state), the largest single-GPU
configuration.  The same invocation also runs short legs of every other configuration (1, 3a-d,
4, 4b, 5r, 5s, 0, 1u, 1f, 1n, 1d, 1p) and reports them under "configs", runs the pipe microbenchmarks
(librad_ubench.so) and reports the measured ALU peaks under "alu_peaks", and compares the
spectrum left by the timed region with the fp64 oracle on sampled bins ("parity").

`--impl reference` times the fp64 CPU oracle (oracle/) as it stands on the host cores, on a
bounded sample of the same workload (the paper has no code to install: DESIGN.md).
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

from paper_2501_03383_b200 import workloads as wl  # noqa: E402

METRIC = "particle*direction*frequency updates/sec"
UNIT = "Gupdates/s"
HEADLINE = "2"
# nominal pipe widths per SM per clock (B200: 4 sub-partitions x 4 MUFU lanes, x 32 FP32 lanes);
# the measured rates come from the microbenchmarks ("alu_peaks")
MUFU_LANES_PER_SM = 16
FP32_LANES_PER_SM = 128
MUFU_PER_UPDATE = 2         # sin + cos: no recurrence exists on a non-uniform grid
FP32_PER_UPDATE_UNIFORM = 6  # 2 (three-term recurrence of the rotation: one packed FMA) + 4 (accumulate) FP32 FMAs
FP32_PER_UPDATE_UNIFORM_SURVEY = 8  # SURVEY.md section 8(d)'s R_lin: a 4-FMA complex rotation + 4 accumulate FMAs
L2_BYTES = 126 * 2 ** 20
# short legs run after the headline: (config, timed steps, warm-up steps)
LEGS = (("1", 50, 3), ("3a", 10, 3), ("3b", 10, 3), ("3c", 10, 3), ("3d", 10, 3), ("4", 3, 1), ("4b", 200, 3),
        ("5r", 200, 5), ("5s", 200, 5), ("0", 500, 5), ("1u", 50, 3), ("1f", 50, 3), ("1n", 50, 3), ("1d", 50, 3), ("1p", 30, 3))


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", default=HEADLINE, choices=wl.ALL_CONFIGS)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--particles", type=int, default=None, help="override particle count (debug)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-legs", action="store_true", help="headline configuration only")
    ap.add_argument("--no-overlap", action="store_true", help="create the detector without RAD_FLAG_OVERLAP_STEPS")
    return ap.parse_args()


def measured_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            return json.loads(p.read_text()), "measured"
        except Exception:
            pass
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while a timed region runs."""

    def __init__(self, index: int, period: float = 0.005):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop_evt = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.dev = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.dev, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {
            nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
            nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
            nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake",
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.dev, nv.NVML_CLOCK_SM)))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.dev)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop_evt.wait(self.period)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2.0)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


# ------------------------------------------------------------------------- oracle legs
def oracle_for(w, bins):
    from oracle import oracle
    if w.n_regions > 1:
        return oracle.RegionOracle(w.n_regions, w.dirs, w.omega, w.dt, t0=w.t0, scale=0.0, bins=bins,
                                   form_factor=w.form_factor, nyquist=w.nyquist)
    return oracle.Oracle(w.dirs, w.omega, w.dt, t0=w.t0, scale=0.0, bins=bins,   # scale 0 = SI default, as the detector
                         form_factor=w.form_factor, nyquist=w.nyquist)


def oracle_step(o, w, step_index, state, n):
    if w.n_regions > 1:
        o.accumulate_step(step_index, w.region_offsets(n), *state)
    else:
        o.accumulate_step(step_index, *state)


def time_oracle(w, state, n_bins_target=None, budget_s=15.0):
    """Oracle rate (updates/s) on one PIC step of `state`, all particles, a bin subset sized
    for about `budget_s` seconds (or exactly n_bins_target bins).  -> (rate, seconds, bins)."""
    from oracle import oracle
    n = state[0].shape[0]
    total = w.n_dir * w.n_omega

    def run(nb):
        bins = np.unique(np.linspace(0, total - 1, nb).round().astype(np.int64))
        o = oracle_for(w, bins)
        t0 = time.perf_counter()
        oracle_step(o, w, 0, state, n)
        dt = time.perf_counter() - t0
        return bins.shape[0] * n / dt, dt, bins.shape[0]

    if n_bins_target is None:
        cores = oracle.num_threads()
        rate, _, _ = run(min(total, max(cores * 2, 16)))       # calibration
        n_bins_target = int(min(total, max(cores, rate * budget_s / max(n, 1))))
    return run(max(1, n_bins_target))


def parity_vs_oracle(w, n, host_states, ring, n_steps_done, S_gpu, budget_updates=1.5e9):
    """The spectrum the timed region left on the device (steps 0 .. n_steps_done-1, step i fed with
    ring state i % ring) against the oracle on a stratified bin sample + the GPU arg-max bin;
    north_star's two error measures.  Runs outside every timed region."""
    total = w.n_regions * w.n_dir * w.n_omega
    per_bin = n * n_steps_done
    nb = int(max(4, min(64, budget_updates // max(per_bin, 1))))
    DW = w.n_dir * w.n_omega
    bins = np.unique(np.concatenate([np.linspace(0, DW - 1, nb).round().astype(np.int64),
                                     [int(np.argmax(S_gpu.reshape(-1, DW).max(axis=0)))]]))
    o = oracle_for(w, bins)
    for i in range(n_steps_done):
        oracle_step(o, w, i, [np.asarray(a) for a in host_states[i % ring]], n)
    ref = o.spectrum().reshape(-1, DW)[:, bins].ravel()
    got = S_gpu.reshape(-1, DW)[:, bins].ravel()
    den = float(np.linalg.norm(ref))
    rel_l2 = float(np.linalg.norm(got - ref) / den) if den > 0 else float(np.linalg.norm(got))
    m = ref >= 1e-6 * float(S_gpu.max())
    maxrel = float(np.max(np.abs(got[m] - ref[m]) / ref[m])) if m.any() else 0.0
    return {"relL2": rel_l2, "maxrel": maxrel, "bins": int(bins.shape[0] * w.n_regions), "of_bins": int(total),
            "steps": int(n_steps_done), "tolerance": {"relL2": 1e-4, "maxrel": 1e-3},
            "ok": bool(rel_l2 <= 1e-4 and maxrel <= 1e-3 and np.isfinite(got).all())}


def run_reference(args):
    """--impl reference: the oracle as it stands, on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    if int(os.environ.get("WORLD_SIZE", "1")) > 1 and "TORCHELASTIC_RUN_ID" in os.environ:
        # torchrun exports OMP_NUM_THREADS=1 to every rank when N > 1; the other ranks do no work here, so rank 0
        # times the oracle on all the host cores it may run on, as at N = 1 (set before the OpenMP runtime loads)
        os.environ["OMP_NUM_THREADS"] = str(len(os.sched_getaffinity(0)))
    from oracle import oracle
    w = wl.make_workload(args.config)
    n = args.particles or w.n_particles
    states = [st for _, st in w.steps(n_steps=min(2, w.n_steps), n_particles=n)]
    cores = oracle.num_threads()
    total_steps = args.steps + args.warmup
    rate, _, _ = time_oracle(w, states[0], n_bins_target=max(cores * 2, 16))
    per_step_s = min(2.0, 90.0 / max(total_steps, 1))
    nb = int(min(w.n_dir * w.n_omega, max(cores, rate * per_step_s / n)))
    for i in range(args.warmup):
        time_oracle(w, states[i % len(states)], n_bins_target=nb)
    t0 = time.perf_counter()
    done = 0
    for i in range(args.steps):
        _, _, b = time_oracle(w, states[i % len(states)], n_bins_target=nb)
        done += b * n
    el = time.perf_counter() - t0
    val = done / el / 1e9
    sample = (f"each step = {nb} of {w.n_dir * w.n_omega} bins (stratified) x all {n} particles of one "
              f"PIC step of {w.name}")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": el / max(args.steps, 1) * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(w, n, 1),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def workload_config(w, n, world):
    """The `config` object: the workload, identical in both arms (what is specific to the GPU run -- handle flags,
    ring size -- is reported under "launch")."""
    return {"workload": w.name, "n_particles_per_gpu": n, "n_regions": w.n_regions, "n_dir": w.n_dir,
            "n_omega": w.n_omega, "state_dtype": np.dtype(w.state_dtype).name,
            "parallelism": f"particle-shard x{world}",
            "l2": "GPU arm: the timed steps cycle through a ring of distinct PIC steps that is either one input per step "
                  "or larger than twice the L2, after an L2 flush (a 252 MiB fill) before the timed region; CPU arm: not "
                  "applicable"}


# ------------------------------------------------------------------------------ our arm
_state_cache = {}


def host_states_for(w, n, ring):
    """Ring of `ring` consecutive PIC steps of workload w (numpy); workloads that share a
    generator (the four sweep shapes; configs 4 and 4b) share the arrays."""
    key = (w.kind, w.seed, n, w.dt, np.dtype(w.state_dtype).name, repr(sorted(w.extra.items())))
    have = _state_cache.get(key, [])
    if len(have) < ring:
        have = [st for _, st in w.steps(n_steps=ring, n_particles=n)]
        _state_cache.clear()                     # one generator's arrays at a time (config 4: 0.7 GB per step)
        _state_cache[key] = have
    return have[:ring]


def alu_peaks(device, sm_mhz_hint):
    """Pipe microbenchmarks (librad_ubench.so): measured results per clock per SM."""
    from paper_2501_03383_b200 import ubench
    res = ubench.run_all(device, blocks_per_sm=4, reps=3)
    g = lambda k: res[k]["per_clk_sm"]      # noqa: E731
    return {
        "mufu_per_clk_sm": g("mufu_ex2"), "sin_per_clk_sm": g("mufu_sin"),
        "sincos_pairs_per_clk_sm": g("sincos_pairs"), "ffma_per_clk_sm": g("ffma"),
        "ffma_imm_per_clk_sm": g("ffma_imm"), "ffma2_instr_per_clk_sm": g("ffma2_instr"),
        "ffma2_fma_per_clk_sm": 2.0 * g("ffma2_instr"), "ffma_var_per_clk_sm": g("ffma_var"),
        "ffma2_var_fma_per_clk_sm": 2.0 * g("ffma2_var_instr"), "ffma2_bcast_fma_per_clk_sm": 2.0 * g("ffma2_bcast_instr"),
        "dfma_per_clk_sm": g("dfma"),
        "f2f_f32_from_f64_per_clk_sm": g("f2f_f32_from_f64"), "f2f_f64_from_f32_per_clk_sm": g("f2f_f64_from_f32"),
        "imad_per_clk_sm": g("imad"),
        "red_v4_f32_per_clk_sm": g("red_v4_f32"), "red_v4_f32_gops": res["red_v4_f32"]["gops"],
        "sincos_pairs_gops": res["sincos_pairs"]["gops"], "ffma_gops": res["ffma"]["gops"],
        "sm_mhz": sm_mhz_hint,
        "how": "librad_ubench.so (csrc/rad_ubench.cu): 8 independent chains per thread, loop unrolled 4x, 4 x 256 threads "
               "per SM; per_clk_sm from clock64() inside the kernel, gops from CUDA events; ffma / ffma2: two loop-invariant "
               "operands (reuse cache), *_var / *_bcast: three different changing registers per instruction",
    }


def measure(cfg, K, W, args, ctx, headline):
    """One leg: W warm-up + K timed steps (accumulate + spectrum) of workload `cfg`, the accumulate
    kernel alone, parity of the spectrum left behind; the headline leg adds multi-step and e2e."""
    import torch
    import torch.distributed as dist
    from paper_2501_03383_b200 import binding, multi
    rank, world, local = ctx["rank"], ctx["world"], ctx["local"]
    peaks, peaks_src, peaks_alu = ctx["peaks"], ctx["peaks_src"], ctx["alu_peaks"]

    w = wl.make_workload(cfg)
    w.seed += 1000 * rank                       # weak scaling: every rank owns its own particles
    n = (args.particles if headline else None) or w.n_particles
    esz = np.dtype(w.state_dtype).itemsize
    bytes_per_step = n * 10 * esz
    # ring of distinct step inputs: either every step of the leg has its own input (read once, after
    # the L2 flush that precedes the timed region), or the ring is more than twice the L2
    ring = int(min(max(K + W, 1), w.n_steps, max(2, 2 * L2_BYTES // bytes_per_step + 1), 256))
    states_np = host_states_for(w, n, ring)
    pin = headline and not args.no_e2e
    host_states = [[torch.from_numpy(a).pin_memory() if pin else torch.from_numpy(a) for a in st] for st in states_np]
    dev_states = [[a.cuda(non_blocking=True) for a in st] for st in host_states]
    torch.cuda.synchronize()

    R = w.n_regions
    off = w.region_offsets(n) if R > 1 else None
    # RAD_FLAG_OVERLAP_STEPS: consecutive calls may overlap on the device (programmatic dependent
    # launches).  Its contract -- a call's input arrays are complete when the call is made -- holds
    # here: device-resident inputs are uploaded and synchronised before the timed region, host inputs
    # reach the kernels through an event of the library's copy stream.
    flags = 0 if args.no_overlap else binding.RAD_FLAG_OVERLAP_STEPS
    if w.precise:
        flags |= binding.RAD_FLAG_PRECISE
    det = binding.Detector(w.dirs, w.omega, w.dt, t0=w.t0, scale=0.0, state_dtype=w.state_dtype,
                           device=local, n_regions=R if R > 1 else 0, flags=flags, form_factor=w.form_factor,
                           nyquist=w.nyquist)
    spec_dev = torch.empty(R * w.n_dir, w.n_omega, dtype=torch.float64, device="cuda")
    reducer = multi.AmplitudeAllReduce(det) if world > 1 else None

    def accumulate(i, host=False):
        st = (host_states if host else dev_states)[i % ring]
        if R > 1:
            (det.accumulate_step_regions_host if host else det.accumulate_step_regions)(i, off, st)
        else:
            (det.accumulate_step_host if host else det.accumulate_step)(i, st)

    def step(i):
        accumulate(i)
        if world > 1:   # the one exchange of the path: sum complex amplitudes over ranks, then |A|^2
            reducer.global_spectrum(out=spec_dev)
        else:
            det.spectrum(out=spec_dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    flush = ctx["flush"]
    for i in range(W):
        step(i)
    flush.fill_(1.0)                            # evict inputs/tables left in L2 by set-up and warm-up
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = det.launch_count
    e0.record()
    for i in range(W, W + K):
        step(i)
    if reducer:
        reducer.wait()                          # the timed region ends when the last exchange has landed
    e1.record()
    barrier()
    clocks = sampler.stop()
    launches = det.launch_count - l0
    ms_total = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(ms_total, op=dist.ReduceOp.MAX)
    ms_total = float(ms_total.item())
    updates_per_step = n * w.n_dir * w.n_omega
    value = world * updates_per_step * K / (ms_total * 1e-3) / 1e9
    S_after = spec_dev.cpu().numpy().copy()     # what the timed region left behind: checked below

    # dominant kernel alone (accumulate), same launch configuration, CUDA events on its stream
    flush.fill_(2.0)
    torch.cuda.synchronize()
    k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    k0.record()
    for i in range(W, W + K):
        accumulate(i)
    k1.record()
    torch.cuda.synchronize()
    kernel_ms = k0.elapsed_time(k1) / K
    achieved = updates_per_step / (kernel_ms * 1e-3) / 1e9
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    n_sm = torch.cuda.get_device_properties(local).multi_processor_count
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    # algorithmic bytes per launch: the particle state read once + one
    # read-modify-write pass over the fp64 accumulator for the fold (D*W*4 doubles = 32 B per bin)
    fold_bytes = R * w.n_dir * w.n_omega * 32
    algorithmic_bytes = bytes_per_step + fold_bytes
    hbm_achieved = algorithmic_bytes / (kernel_ms * 1e-3) / 1e9
    traffic = None
    try:
        traffic = json.loads((ROOT / "profiles" / "traffic.json").read_text()).get(w.name, {}).get("bytes")
    except Exception:
        pass
    variant = det.kernel_variant
    if variant == "stream":      # few bins per particle: the 40 B/particle stream from HBM binds
        roofline = {"bound": "hbm", "achieved": hbm_achieved, "peak": hbm_peak, "unit": "GB/s",
                    "frac": hbm_achieved / hbm_peak, "traffic": traffic,
                    "peak_how": f"MEASURED_PEAKS.json hbm_gbs ({peaks_src})"}
    else:
        if variant == "uniform":  # rotation recurrence: 2 FP32 FMA rotate (three-term) + 4 FMA accumulate per update
            per_clk_sm, pipe = FP32_LANES_PER_SM / FP32_PER_UPDATE_UNIFORM, "FP32 (6 FMAs per update: 3 fma.rn.f32x2)"
            measured = peaks_alu["ffma2_fma_per_clk_sm"] / FP32_PER_UPDATE_UNIFORM if peaks_alu else None
        elif variant == "general+precise":
            # RAD_FLAG_PRECISE: every sincos by the fp32 polynomial: 23 + 4 accumulate + ~1 loop / load instructions per
            # update on the FMA and ALU pipes, no MUFU: bound by issue slots
            per_clk_sm, pipe = FP32_LANES_PER_SM / 28.0, "issue (28 instructions per update: polynomial sincos)"
            measured = None
        elif variant == "general+dyadic":
            # dyadic log grid: per two bins one anchor (phase + sincos: 8 instructions) + one squaring (4) +
            # 2 x 4 accumulates = 10 instructions per update at 1 MUFU per update: bound by issue slots
            per_clk_sm, pipe = FP32_LANES_PER_SM / 10.0, "issue (10 instructions per update: anchor + squaring chains)"
            measured = None
        elif variant.endswith("+formfactor") and not variant.startswith("uniform"):
            # general grid with the macro-particle form factor: sin + cos + sqrt per update
            per_clk_sm, pipe = MUFU_LANES_PER_SM / 3.0, "MUFU (sin+cos+sqrt per update)"
            measured = peaks_alu["mufu_per_clk_sm"] / 3.0 if peaks_alu else None
        else:                     # general grid: sin + cos per update on the 16-lane MUFU
            per_clk_sm, pipe = MUFU_LANES_PER_SM / MUFU_PER_UPDATE, "MUFU (sin+cos per update)"
            measured = peaks_alu["sincos_pairs_per_clk_sm"] if peaks_alu else None
        peak = n_sm * per_clk_sm * sm_max * 1e6 / 1e9
        roofline = {"bound": "alu", "pipe": pipe, "achieved": achieved, "peak": peak, "unit": UNIT,
                    "frac": achieved / peak, "traffic": traffic,
                    "peak_how": f"nominal: {n_sm} SMs x {per_clk_sm:g} updates/clk/SM x {sm_max:.0f} MHz (max SM clock, "
                                f"{peaks_src}); DESIGN.md section 5"}
        if measured:
            peak_m = n_sm * measured * sm_max * 1e6 / 1e9
            roofline.update({"peak_measured_pipe": peak_m, "frac_of_measured_pipe": achieved / peak_m,
                             "peak_measured_how": f"{n_sm} SMs x {measured:.3f} updates/clk/SM (alu_peaks) x {sm_max:.0f} MHz"})
        if variant == "uniform":
            # SURVEY.md section 8(d) defines R_lin with a 4-FMA complex rotation (8 FMAs per update); the kernel's
            # three-term recurrence needs 6, so `peak` above is the (higher) bound of what the kernel computes
            peak_s = n_sm * FP32_LANES_PER_SM / FP32_PER_UPDATE_UNIFORM_SURVEY * sm_max * 1e6 / 1e9
            roofline.update({"peak_survey_r_lin": peak_s, "frac_of_survey_r_lin": achieved / peak_s})
        if variant == "uniform" and peaks_alu and peaks_alu.get("ffma2_var_fma_per_clk_sm"):
            # the sweep's packed FMAs read three different register pairs each: what the register file feeds the
            # FMA pipe without operand reuse (alu_peaks ffma2_var_fma) is the rate the kernel actually sits on
            peak_v = n_sm * peaks_alu["ffma2_var_fma_per_clk_sm"] / FP32_PER_UPDATE_UNIFORM * sm_max * 1e6 / 1e9
            roofline.update({"peak_measured_no_operand_reuse": peak_v, "frac_of_measured_no_operand_reuse": achieved / peak_v})
        if clocks.get("sm_mhz"):
            roofline["frac_at_sampled_clock"] = roofline["frac"] * sm_max / clocks["sm_mhz"]
    roofline.update({"kernel": f"rad_accum_{variant}", "kernel_ms": kernel_ms,
                     "algorithmic_bytes": int(algorithmic_bytes), "state_bytes": int(bytes_per_step),
                     "fold_bytes": int(fold_bytes), "updates_per_launch": int(updates_per_step),
                     "gupdates_per_s": achieved, "hbm_gbs_achieved": hbm_achieved, "hbm_gbs_peak": hbm_peak})
    if traffic:
        roofline["traffic_over_algorithmic"] = traffic / algorithmic_bytes

    out = {"value": value, "unit": UNIT, "steps": K, "warmup": W, "ms_per_step": ms_total / K,
           "kernel": f"rad_accum_{variant}", "roofline": roofline, "clocks": clocks, "gpu_launches": int(launches),
           "config": workload_config(w, n, world),
           "launch": {"flags": ("none" if args.no_overlap else "RAD_FLAG_OVERLAP_STEPS") + (" | RAD_FLAG_PRECISE" if w.precise else ""),
                      "l2": f"ring of {ring} distinct step inputs ({ring * bytes_per_step / 2**20:.0f} MiB) + "
                            f"L2 flush before the timed region"}}

    # parity of what the timed region computed (outside the timed region; rank 0's own shard)
    if world == 1 and not args.no_cpu_baseline:
        out["parity"] = parity_vs_oracle(w, n, states_np, ring, W + K, S_after,
                                         budget_updates=2.0e9 if headline else 5.0e8)

    tiny = updates_per_step < 1e7          # launch-bound steps (config 0): the many-steps-per-launch figure is the one that counts
    if headline or tiny:
        # rad_accumulate_steps: T resident steps in one launch (ramp/tail/launch latency paid once)
        T = int(min(128 if tiny else 16, ring, (2 << 30) // max(bytes_per_step, 1)))
        if T >= 2 and world == 1:
            stacked = [torch.stack([dev_states[i][c] for i in range(T)]).contiguous() for c in range(10)]
            det.accumulate_steps(0, stacked, region_offsets=off)
            torch.cuda.synchronize()
            m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            reps = max(1, min(10, K // T))
            m0.record()
            for r_ in range(reps):
                det.accumulate_steps(r_ * T, stacked, region_offsets=off)
            m1.record()
            torch.cuda.synchronize()
            ms_ms = m0.elapsed_time(m1) / reps
            out["multi_step"] = {"steps_per_launch": T, "ms_per_launch": ms_ms,
                                 "value": updates_per_step * T / (ms_ms * 1e-3) / 1e9, "unit": UNIT,
                                 "note": "rad_accumulate_steps (kernel only, inputs resident); not the headline"}
            del stacked

    if headline:
        # end to end through the public API with HOST buffers: H2D of the step's state and D2H of
        # the step's spectrum inside the timed region, every step
        if not args.no_e2e:
            det.reset()
            # every step's spectrum lands in pinned host memory (RAD_OUT_HOST_ASYNC); the host waits
            # for step i-1's result while step i's copies and kernels are already queued
            spec_pinned = [torch.empty(R * w.n_dir, w.n_omega, dtype=torch.float64).pin_memory() for _ in range(2)]
            arrived = [torch.cuda.Event(), torch.cuda.Event()]
            ke = max(1, min(K, 50))
            we = min(W, 3)
            for i in range(we):
                accumulate(i, host=True)
            barrier()
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a0.record()
            for i in range(we, we + ke):
                accumulate(i, host=True)
                b = i & 1
                if world > 1:
                    reducer.global_spectrum(out=spec_dev)
                    reducer.wait()
                    spec_pinned[b].copy_(spec_dev, non_blocking=True)
                else:
                    det.spectrum(out=spec_pinned[b])
                arrived[b].record()
                if i > we:
                    arrived[b ^ 1].synchronize()
            arrived[(we + ke - 1) & 1].synchronize()
            a1.record()
            barrier()
            S_e2e = spec_pinned[(we + ke - 1) & 1].numpy().copy()
            ms_e = torch.tensor([a0.elapsed_time(a1)], dtype=torch.float64, device="cuda")
            if world > 1:
                dist.all_reduce(ms_e, op=dist.ReduceOp.MAX)
            out["e2e"] = {"value": world * updates_per_step * ke / (float(ms_e.item()) * 1e-3) / 1e9, "unit": UNIT,
                          "h2d_bytes_per_step": int(bytes_per_step),
                          "d2h_bytes_per_step": int(spec_pinned[0].numel() * 8), "steps": ke}
            if world == 1 and not args.no_cpu_baseline:   # the last host-side spectrum of the e2e leg, checked too
                out["e2e"]["parity"] = parity_vs_oracle(w, n, states_np, ring, we + ke, S_e2e, budget_updates=1.0e9)

        if rank == 0 and world == 1 and not args.no_cpu_baseline:
            from oracle import oracle
            rate, secs, nb = time_oracle(w, states_np[0], budget_s=12.0)
            out["cpu_baseline"] = {"value": rate / 1e9, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                                   "sample": f"{nb} of {w.n_dir * w.n_omega} bins (stratified) x all {n} particles of "
                                             f"one PIC step of {w.name}; {secs:.1f} s"}
    det.close()
    if reducer:
        reducer.close()
    del dev_states, host_states
    torch.cuda.empty_cache()
    return out


def measure_fast(cfg, K, W, args, ctx):
    """The approximate fast path (RAD_FLAG_FAST_GRIDDED) on workload `cfg`: W warm-up + K timed
    accumulate calls (spreading + fold), then ONE spectrum (evaluation of the grids), parity of that
    spectrum against the exact oracle.  Reported beside, never instead of, the direct-sum numbers."""
    import torch
    from paper_2501_03383_b200 import binding
    local = ctx["local"]
    w = wl.make_workload(cfg)
    n = w.n_particles
    bytes_per_step = n * 10 * np.dtype(w.state_dtype).itemsize
    ring = int(min(K + W, w.n_steps, max(2, 2 * L2_BYTES // bytes_per_step + 1)))
    states_np = host_states_for(w, n, ring)
    dev_states = [[torch.from_numpy(a).cuda() for a in st] for st in states_np]
    L = 10e-6   # the KHI box of the generators (workloads.py); particles drift < 1 nm over a window
    box = ((-0.02 * L,) * 3, (1.02 * L,) * 3)
    det = binding.Detector(w.dirs, w.omega, w.dt, t0=w.t0, scale=0.0, state_dtype=w.state_dtype, device=local,
                           flags=binding.RAD_FLAG_FAST_GRIDDED, fast=(box[0], box[1], 0, w.n_steps, 0.0))
    spec_dev = torch.empty(w.n_dir, w.n_omega, dtype=torch.float64, device="cuda")
    for i in range(W):
        det.accumulate_step(i, dev_states[i % ring])
    ctx["flush"].fill_(3.0)
    torch.cuda.synchronize()
    e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
    l0 = det.launch_count
    e0.record()
    for i in range(W, W + K):
        det.accumulate_step(i, dev_states[i % ring])
    e1.record()
    det.spectrum(out=spec_dev)
    e2.record()
    torch.cuda.synchronize()
    ms_acc, ms_spec = e0.elapsed_time(e1) / K, e1.elapsed_time(e2)
    launches = det.launch_count - l0
    S = spec_dev.cpu().numpy().copy()
    updates = n * w.n_dir * w.n_omega
    out = {"workload": w.name, "flag": "RAD_FLAG_FAST_GRIDDED", "tolerance": 1e-6, "steps": K, "warmup": W,
           "ms_per_accumulate": ms_acc, "ms_per_spectrum": ms_spec,
           "effective_updates_per_s": {"unit": UNIT, "accumulate_only": updates / (ms_acc * 1e-3) / 1e9,
                                       "spectrum_every_100_steps": updates * 100 / ((100 * ms_acc + ms_spec) * 1e-3) / 1e9,
                                       "spectrum_every_step": updates / ((ms_acc + ms_spec) * 1e-3) / 1e9},
           "gpu_launches": int(launches), "kernel": "rad_spread + rad_grid_fold (per step), rad_accum<GRID> (per spectrum)",
           "roofline": None,
           "note": "effective = direct-sum updates this replaces / time; an approximation (gridding tolerance 1e-6), "
                   "checked against the exact oracle with the exact path's tolerances"}
    # the spreading kernel is bound by the rate at which L2 takes its 16-byte vector reductions: WD/2 = 4 per
    # (particle, direction) term at the default width; peak = the measured rate of the same instruction on
    # scattered places of an L2-resident buffer (alu_peaks red_v4_f32)
    pk = ctx.get("alu_peaks") or {}
    red_per_s = n * w.n_dir * 4 / (ms_acc * 1e-3) / 1e9
    if pk.get("red_v4_f32_gops"):
        out["roofline"] = {"bound": "l2-reductions", "achieved": red_per_s, "peak": pk["red_v4_f32_gops"],
                           "unit": "G red.v4.f32/s", "frac": red_per_s / pk["red_v4_f32_gops"],
                           "kernel": "rad_spread (+ rad_grid_fold)", "reductions_per_term": 4,
                           "peak_how": "alu_peaks red_v4_f32 (csrc/rad_ubench.cu): the same instruction, runs of 4 consecutive "
                                       "chunks at scattered places of a 64 MB L2-resident buffer, CUDA events; the kernel's own "
                                       "deposits are denser (tens of terms per grid point and step), so it can exceed this figure"}
    if not args.no_cpu_baseline:
        out["parity"] = parity_vs_oracle(w, n, states_np, ring, W + K, S, budget_updates=5.0e8)
    det.close()
    del dev_states
    torch.cuda.empty_cache()
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2501_03383_b200 import build as rad_build

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    rad_build.build()
    peaks, peaks_src = measured_peaks()
    ctx = {"rank": rank, "world": world, "local": local, "peaks": peaks, "peaks_src": peaks_src,
           "flush": torch.empty(2 * L2_BYTES // 4, dtype=torch.float32, device="cuda"), "alu_peaks": None}
    t_start = time.perf_counter()
    try:
        ctx["alu_peaks"] = alu_peaks(local, float(peaks.get("sm_max_mhz", 1965.0)))
    except Exception as exc:       # the microbenchmarks are evidence, not the product: report, go on
        ctx["alu_peaks"] = None
        ctx["alu_peaks_error"] = repr(exc)

    head = measure(args.config, args.steps, args.warmup, args, ctx, headline=True)
    legs, fast = {}, {}
    if world == 1 and not args.no_legs and args.config == HEADLINE and args.particles is None:
        def fast_leg(cfg, k, wu):
            try:
                f = measure_fast(cfg, k, wu, args, ctx)
                fast[f["workload"]] = f
            except Exception as exc:
                fast[f"cfg {cfg}"] = {"error": repr(exc)}
        fast_leg(HEADLINE, 10, 3)           # the generator's arrays of the headline are still cached
        for cfg, k, wu in LEGS:
            try:
                leg = measure(cfg, k, wu, args, ctx, headline=False)
                legs[leg["config"]["workload"]] = leg
            except Exception as exc:
                legs[f"cfg {cfg}"] = {"error": repr(exc)}
            if cfg in ("1", "3a"):
                fast_leg(cfg, 20, 3)
    if rank == 0:
        line = {
            "metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": head["ms_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32",
            "dtype_detail": "f32 phase arithmetic, sincos and per-chunk partial sums; f64 phase set-up, Doppler factor and accumulators",
            "data": "synthetic",
            "config": head["config"], "launch": head["launch"], "clocks": head["clocks"], "e2e": head.get("e2e"),
            "gpu_launches": head["gpu_launches"], "roofline": head["roofline"],
            "cpu_baseline": head.get("cpu_baseline"), "parity": head.get("parity"),
            "multi_step": head.get("multi_step"), "alu_peaks": ctx["alu_peaks"], "configs": legs,
            "fast_gridded": fast,
            "bench_wall_s": time.perf_counter() - t_start,
        }
        if "alu_peaks_error" in ctx:
            line["alu_peaks_error"] = ctx["alu_peaks_error"]
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
