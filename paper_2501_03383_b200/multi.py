"""Multi-GPU plumbing: particles are sharded across ranks (as PIConGPU's
domain decomposition does); each rank accumulates its own amplitude A;
the ranks then sum the COMPLEX AMPLITUDES (never intensities: "sum of the
contributions from all radiating particles in the simulation") with ONE all-reduce over the
accumulator itself -- D*W*4 doubles, the two transverse components (rad_export_accumulator) --
and |A|^2 is taken afterwards (rad_spectrum_of).  torch.distributed only (NCCL on GPUs, gloo in
the CPU tests); no arithmetic of the method lives here.

The exchange runs on a side stream: export (a device-to-device copy on the compute stream) ->
event -> all-reduce + |A|^2 on the side stream, so that the accumulation of step i+1, queued on
the compute stream right after, overlaps the collective of step i.
"""
from __future__ import annotations

from typing import Tuple


def shard_range(n: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous, balanced [begin, end) slice of n particles for `rank` of `world`."""
    if world < 1 or not (0 <= rank < world) or n < 0:
        raise ValueError("bad shard request")
    base, rem = divmod(n, world)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def allreduce_amplitude(amp, group=None):
    """In-place SUM all-reduce of an amplitude buffer (fp64, any layout) over the ranks."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(amp, op=dist.ReduceOp.SUM, group=group)
    return amp


class AmplitudeAllReduce:
    """Spectrum of the sum over ranks for one detector, with the exchange hidden behind the next
    step's accumulation.

        red = AmplitudeAllReduce(det)
        for step: det.accumulate_step(...); red.global_spectrum(out=spec)   # returns at once
        red.wait()            # the compute stream now sees every `out` written so far

    Two amplitude buffers alternate, so the export of step i+1 never overwrites the buffer the
    side stream is still reducing for step i.
    """

    def __init__(self, det, group=None):
        import torch
        self.det, self.group = det, group
        dev = torch.device("cuda", det.device)
        shape = ((det.R,) if det.R > 1 else ()) + (det.D, det.W, 4)
        self.buf = [torch.empty(shape, dtype=torch.float64, device=dev) for _ in range(2)]
        self.side = torch.cuda.Stream(device=dev)
        self.exported = [torch.cuda.Event() for _ in range(2)]
        self.done = [None, None]           # side-stream event of the last use of each buffer
        self.turn = 0

    def global_spectrum(self, out):
        """Queue: export A -> all-reduce (SUM over ranks) -> out = scale * |sum A|^2.  `out` (CUDA
        fp64 [(R,) D, W]) is written on the side stream; call wait() before using it on the
        compute stream."""
        import torch
        b = self.turn
        self.turn ^= 1
        compute = torch.cuda.current_stream(self.det.device)
        if self.done[b] is not None:
            compute.wait_event(self.done[b])          # buffer b is free again
        self.det.export_accumulator(self.buf[b])      # D2D copy, ordered after every fold queued so far
        self.exported[b].record(compute)
        self.side.wait_event(self.exported[b])
        with torch.cuda.stream(self.side):
            allreduce_amplitude(self.buf[b], self.group)
            self.det.spectrum_of(self.buf[b], out=out)
            ev = torch.cuda.Event()
            ev.record(self.side)
        self.done[b] = ev
        return out

    def wait(self):
        """Make the current (compute) stream wait for everything queued on the side stream."""
        import torch
        compute = torch.cuda.current_stream(self.det.device)
        for ev in self.done:
            if ev is not None:
                compute.wait_event(ev)

    def close(self):
        import torch
        self.side.synchronize()
        torch.cuda.current_stream(self.det.device).synchronize()
        self.buf = []
