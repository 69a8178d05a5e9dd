"""World-size-2 gloo test (CPU) of the multi-GPU plumbing: shard particles, sum complex
amplitudes with all_reduce, then |A|^2 -- equals the single-process result; summing
intensities instead would not."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2501_03383_b200 import multi, workloads as wl


def test_shard_range_partitions_exactly():
    for n in (0, 1, 7, 64, 1000):
        for world in (1, 2, 3, 8):
            spans = [multi.shard_range(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [e - b for b, e in spans]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        multi.shard_range(10, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import oracle
        w = wl.make_workload("3c")
        dirs, omega = w.dirs[:4], w.omega[::32]
        b, e = multi.shard_range(n, rank, world)
        o = oracle.Oracle(dirs, omega, w.dt, scale=1.0)
        for t, st in w.steps(n_steps=2, n_particles=n):
            o.accumulate_step(t, *[a[b:e] for a in st])
        amp = torch.from_numpy(o.A.copy())
        local_S = torch.from_numpy(o.spectrum())
        multi.allreduce_amplitude(amp)
        dist.all_reduce(local_S)                      # the WRONG way, for contrast
        if rank == 0:
            np.save(os.path.join(out_dir, "amp.npy"), amp.numpy())
            np.save(os.path.join(out_dir, "sum_of_intensities.npy"), local_S.numpy())
    finally:
        dist.destroy_process_group()


def test_two_rank_amplitude_allreduce_matches_single_process(tmp_path, oracle_mod):
    n, world = 301, 2
    mp.spawn(_worker, args=(world, _free_port(), n, str(tmp_path)), nprocs=world, join=True)
    amp = np.load(tmp_path / "amp.npy")
    w = wl.make_workload("3c")
    o = oracle_mod.Oracle(w.dirs[:4], w.omega[::32], w.dt, scale=1.0)
    for t, st in w.steps(n_steps=2, n_particles=n):
        o.accumulate_step(t, *st)
    assert np.allclose(amp, o.A, rtol=0, atol=1e-12 * np.abs(o.A).max())
    S = (amp ** 2).sum(axis=(2, 3))
    assert np.allclose(S, o.spectrum(), rtol=1e-10)
    wrong = np.load(tmp_path / "sum_of_intensities.npy")
    assert not np.allclose(wrong, o.spectrum(), rtol=1e-3)
