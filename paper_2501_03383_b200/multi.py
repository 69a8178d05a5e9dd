"""Multi-GPU plumbing: particles are sharded across ranks (as PIConGPU's
domain decomposition does); each rank accumulates its own amplitude A;
the ranks then sum the COMPLEX AMPLITUDES (never intensities: "sum of the
contributions from all radiating particles in the simulation") with one all-reduce of
D*W*6 doubles, and |A|^2 is taken afterwards.  torch.distributed only (NCCL on GPUs, gloo in
the CPU tests); no arithmetic of the method lives here.
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
    """In-place SUM all-reduce of an amplitude buffer [D, W, 3, 2] (fp64) over the ranks."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(amp, op=dist.ReduceOp.SUM, group=group)
    return amp


def global_spectrum(local_det, global_det, amp_buf, out=None, group=None):
    """Spectrum of the sum over ranks: export local A, all-reduce, load into `global_det`
    (a second handle on the same grid) and take |A|^2 there.  All device-side, asynchronous."""
    local_det.amplitude(out=amp_buf)
    allreduce_amplitude(amp_buf, group)
    global_det.reset()
    global_det.add_amplitude(amp_buf)
    return global_det.spectrum(out=out)
