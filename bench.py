#!/usr/bin/env python
"""bench.py -- throughput of the radiation-detector hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1] [--impl ours|reference]

A "step" is one pass of the whole hot path over one PIC step of synthetic input:
rad_accumulate_step (stage + accumulate + fold) followed by
rad_spectrum (a4).  Metric (BASELINE.json): particle*direction*frequency updates per second,
in G/s, whole job.  Default workload = BASELINE.json configs[1] ("KHI-like shear", 65 536
electrons x 128 directions x 512 log-spaced frequencies, fp32 state).

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
MUFU_LANES_PER_SM = 16      # B200_PROFILING / microbenchmark: 16 MUFU results per clk per SM
MUFU_PER_UPDATE = 2         # sin + cos: no recurrence exists on a non-uniform grid
L2_BYTES = 126 * 2 ** 20


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", default="1", choices=wl.ALL_CONFIGS)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--particles", type=int, default=None, help="override particle count (debug)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
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
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period: float = 0.05):
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


# ------------------------------------------------------------------------- oracle timing
def time_oracle(w, state, n_bins_target=None, budget_s=15.0):
    """Oracle rate (updates/s) on one PIC step of `state`, all particles, a bin subset sized
    for about `budget_s` seconds (or exactly n_bins_target bins).  -> (rate, seconds, bins)."""
    from oracle import oracle
    n = state[0].shape[0]
    total = w.n_dir * w.n_omega

    def run(nb):
        bins = np.unique(np.linspace(0, total - 1, nb).round().astype(np.int64))
        if w.n_regions > 1:       # per-region detectors: every particle feeds its own region's bins
            o = oracle.RegionOracle(w.n_regions, w.dirs, w.omega, w.dt, t0=w.t0, scale=1.0, bins=bins)
            off = w.region_offsets(n)
            t0 = time.perf_counter()
            o.accumulate_step(0, off, *state)
        else:
            o = oracle.Oracle(w.dirs, w.omega, w.dt, t0=w.t0, scale=1.0, bins=bins)
            t0 = time.perf_counter()
            o.accumulate_step(0, *state)
        dt = time.perf_counter() - t0
        return bins.shape[0] * n / dt, dt, bins.shape[0]

    if n_bins_target is None:
        cores = oracle.num_threads()
        rate, _, _ = run(min(total, max(cores * 2, 16)))       # calibration
        n_bins_target = int(min(total, max(cores, rate * budget_s / max(n, 1))))
    return run(max(1, n_bins_target))


def run_reference(args):
    """--impl reference: the oracle as it stands, on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
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
        "data": "synthetic", "config": {"workload": w.name, "n_particles": n, "n_regions": w.n_regions,
                                        "n_dir": w.n_dir, "n_omega": w.n_omega,
                                        "state_dtype": np.dtype(w.state_dtype).name},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ------------------------------------------------------------------------------ our arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2501_03383_b200 import binding, build as rad_build, multi

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

    w = wl.make_workload(args.config)
    w.seed += 1000 * rank                       # weak scaling: every rank owns its own particles
    n = args.particles or w.n_particles
    K, W = args.steps, args.warmup
    bytes_per_step = n * 10 * np.dtype(w.state_dtype).itemsize
    # ring of distinct step inputs, larger than L2 so that no timed step finds its input cached
    ring = min(max(K + W, 1), w.n_steps, max(8, int(2 * L2_BYTES // bytes_per_step) + 1), 256)
    host_states = []
    for t, st in w.steps(n_steps=ring, n_particles=n):
        host_states.append([torch.from_numpy(a).pin_memory() for a in st])
    dev_states = [[a.cuda(non_blocking=True) for a in st] for st in host_states]
    torch.cuda.synchronize()

    R = w.n_regions
    off = w.region_offsets(n) if R > 1 else None
    # RAD_FLAG_OVERLAP_STEPS: consecutive calls may overlap on the device (programmatic dependent
    # launches).  Its contract -- a call's input arrays are complete when the call is made -- holds
    # here: device-resident inputs are uploaded and synchronised before the timed region, host inputs
    # reach the kernels through an event of the library's copy stream.
    flags = 0 if args.no_overlap else binding.RAD_FLAG_OVERLAP_STEPS
    det = binding.Detector(w.dirs, w.omega, w.dt, t0=w.t0, scale=0.0, state_dtype=w.state_dtype,
                           device=local, n_regions=R if R > 1 else 0, flags=flags)
    spec_dev = torch.empty(R * w.n_dir, w.n_omega, dtype=torch.float64, device="cuda")
    if world > 1:
        det_glob = binding.Detector(w.dirs, w.omega, w.dt, t0=w.t0, scale=0.0,
                                    state_dtype=w.state_dtype, device=local, n_regions=R if R > 1 else 0,
                                    flags=flags)
        amp_buf = torch.empty(R * w.n_dir, w.n_omega, 3, 2, dtype=torch.float64, device="cuda")

    def accumulate(i, host=False):
        st = (host_states if host else dev_states)[i % ring]
        if R > 1:
            (det.accumulate_step_regions_host if host else det.accumulate_step_regions)(i, off, st)
        else:
            (det.accumulate_step_host if host else det.accumulate_step)(i, st)

    def step(i):
        accumulate(i)
        if world > 1:   # the one exchange of the path: sum complex amplitudes, then |A|^2
            multi.global_spectrum(det, det_glob, amp_buf, out=spec_dev)
        else:
            det.spectrum(out=spec_dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    flush = torch.empty(2 * L2_BYTES // 4, dtype=torch.float32, device="cuda")
    for i in range(W):
        step(i)
    flush.fill_(1.0)                            # evict inputs/tables left in L2 by set-up and warm-up
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = det.launch_count + (det_glob.launch_count if world > 1 else 0)
    e0.record()
    for i in range(W, W + K):
        step(i)
    e1.record()
    barrier()
    clocks = sampler.stop()
    launches = det.launch_count + (det_glob.launch_count if world > 1 else 0) - l0
    ms_total = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(ms_total, op=dist.ReduceOp.MAX)
    ms_total = float(ms_total.item())
    updates_per_step = n * w.n_dir * w.n_omega
    value = world * updates_per_step * K / (ms_total * 1e-3) / 1e9
    spectrum_check = float(spec_dev.sum().item())

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
    hbm_achieved = bytes_per_step / (kernel_ms * 1e-3) / 1e9
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
        if variant == "uniform":  # rotation recurrence: 4 FP32 rotate + 4 FMA accumulate per update
            per_clk_sm, pipe = 128.0 / 8.0, "FP32 (8 FMA-pipe instr per update)"
        else:                     # general grid: sin + cos per update on the 16-lane MUFU
            per_clk_sm, pipe = MUFU_LANES_PER_SM / MUFU_PER_UPDATE, "MUFU (sin+cos per update)"
        peak = n_sm * per_clk_sm * sm_max * 1e6 / 1e9
        roofline = {"bound": "alu", "pipe": pipe, "achieved": achieved, "peak": peak, "unit": UNIT,
                    "frac": achieved / peak, "traffic": traffic,
                    "peak_how": f"{n_sm} SMs x {per_clk_sm:g} updates/clk/SM x {sm_max:.0f} MHz (max SM clock, "
                                f"{peaks_src}); DESIGN.md section 5"}
    if variant == "uniform":
        # plain FFMA issues at 84-87 thread-instr/clk/SM on B200 (BASELINE.md note vii), not the nominal 128
        roofline["frac_of_measured_ffma_rate"] = achieved / (n_sm * 87.0 / 8.0 * sm_max * 1e6 / 1e9)
    roofline.update({"kernel": f"rad_accum_{variant}", "kernel_ms": kernel_ms,
                     "algorithmic_bytes": int(bytes_per_step), "updates_per_launch": int(updates_per_step),
                     "gupdates_per_s": achieved, "hbm_gbs_achieved": hbm_achieved, "hbm_gbs_peak": hbm_peak})
    if clocks.get("sm_mhz"):
        if roofline["bound"] == "alu":
            roofline["frac_at_sampled_clock"] = roofline["frac"] * sm_max / clocks["sm_mhz"]

    # rad_accumulate_steps: T resident steps in one launch (ramp/tail/launch latency paid once)
    multi_step = None
    T = int(min(16, ring, (2 << 30) // max(bytes_per_step, 1)))
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
        multi_step = {"steps_per_launch": T, "ms_per_launch": ms_ms,
                      "value": updates_per_step * T / (ms_ms * 1e-3) / 1e9, "unit": UNIT,
                      "note": "rad_accumulate_steps (kernel only, inputs resident); not the headline"}
        del stacked

    # end to end through the public API with HOST buffers: H2D of the step's state and D2H of
    # the step's spectrum inside the timed region, every step
    e2e = None
    if not args.no_e2e:
        det.reset()
        # every step's spectrum lands in pinned host memory (RAD_OUT_HOST_ASYNC); the host waits
        # for step i-1's result while step i's copies and kernels are already queued
        spec_pinned = [torch.empty(R * w.n_dir, w.n_omega, dtype=torch.float64).pin_memory() for _ in range(2)]
        arrived = [torch.cuda.Event(), torch.cuda.Event()]
        ke = max(1, min(K, 50))
        for i in range(min(W, 3)):
            accumulate(i, host=True)
        barrier()
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e2e_check = 0.0
        a0.record()
        for i in range(W, W + ke):
            accumulate(i, host=True)
            b = i & 1
            if world > 1:
                multi.global_spectrum(det, det_glob, amp_buf, out=spec_dev)
                spec_pinned[b].copy_(spec_dev, non_blocking=True)
            else:
                det.spectrum(out=spec_pinned[b])
            arrived[b].record()
            if i > W:
                arrived[b ^ 1].synchronize()
                e2e_check += float(spec_pinned[b ^ 1][0, 0])
        arrived[(W + ke - 1) & 1].synchronize()
        e2e_check += float(spec_pinned[(W + ke - 1) & 1][0, 0])
        a1.record()
        barrier()
        ms_e = torch.tensor([a0.elapsed_time(a1)], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(ms_e, op=dist.ReduceOp.MAX)
        e2e = {"value": world * updates_per_step * ke / (float(ms_e.item()) * 1e-3) / 1e9, "unit": UNIT,
               "h2d_bytes_per_step": int(bytes_per_step), "d2h_bytes_per_step": int(spec_pinned[0].numel() * 8),
               "steps": ke}

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import oracle
        st0 = [a.numpy() for a in host_states[0]]
        rate, secs, nb = time_oracle(w, st0, budget_s=15.0)
        cpu_baseline = {"value": rate / 1e9, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                        "sample": f"{nb} of {w.n_dir * w.n_omega} bins (stratified) x all {n} particles of one "
                                  f"PIC step of {w.name}; {secs:.1f} s"}
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32 phase/amplitude, f64 set-up and accumulators", "data": "synthetic",
            "config": {"workload": w.name, "n_particles_per_gpu": n, "n_regions": R, "n_dir": w.n_dir,
                       "n_omega": w.n_omega,
                       "state_dtype": np.dtype(w.state_dtype).name, "parallelism": f"particle-shard x{world}",
                       "flags": "none" if args.no_overlap else "RAD_FLAG_OVERLAP_STEPS",
                       "l2": f"ring of {ring} distinct step inputs ({ring * bytes_per_step / 2**20:.0f} MiB) + "
                             f"L2 flush before the timed region"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
            "cpu_baseline": cpu_baseline, "multi_step": multi_step, "spectrum_checksum": spectrum_check,
        }))
    det.close()
    if world > 1:
        det_glob.close()
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
