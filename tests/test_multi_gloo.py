"""Multi-process gloo tests (CPU, world sizes 2 and 3) of the multi-GPU plumbing: shard the
particles (uneven shards), every rank forms ITS amplitude, the ranks sum the complex amplitudes
with ONE all-reduce over the accumulator layout of rad_export_accumulator (D*W*4 doubles: the two
transverse components), then |A1|^2 + |A2|^2 -- equal to the single-process spectrum; summing
intensities instead would not be (amplitudes add)."""
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


def transverse_basis(dirs):
    """The basis include/rad.h documents for rad_export_accumulator: e1 = normalise(z^ x n)
    (x^ x n if |n_z| > 0.9), e2 = n x e1 -- a function of n alone, so every rank has the same."""
    n = dirs / np.linalg.norm(dirs, axis=1, keepdims=True)
    e1 = np.where(np.abs(n[:, 2:3]) > 0.9, np.cross([1.0, 0.0, 0.0], n), np.cross([0.0, 0.0, 1.0], n))
    e1 /= np.linalg.norm(e1, axis=1, keepdims=True)
    return n, e1, np.cross(n, e1)


def to_amp4(A_xyz, dirs):
    """Cartesian complex amplitude [D, W, 3] -> accumulator layout [D, W, 4] = (Re A1, Im A1, Re A2, Im A2)."""
    _, e1, e2 = transverse_basis(dirs)
    a1 = np.einsum("dwc,dc->dw", A_xyz, e1)
    a2 = np.einsum("dwc,dc->dw", A_xyz, e2)
    return np.stack([a1.real, a1.imag, a2.real, a2.imag], axis=-1)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _grid():
    w = wl.make_workload("3c")
    dirs = np.concatenate([w.dirs[:4], [[0.0, 0.0, 1.0], [0.1, 0.05, -0.99]]])   # incl. |n_z| > 0.9 (x^ x n branch)
    return w, dirs, w.omega[::32]


def _worker(rank, world, port, n, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import oracle
        w, dirs, omega = _grid()
        b, e = multi.shard_range(n, rank, world)
        o = oracle.Oracle(dirs, omega, w.dt, scale=1.0)
        for t, st in w.steps(n_steps=2, n_particles=n):
            o.accumulate_step(t, *[a[b:e] for a in st])
        amp4 = torch.from_numpy(to_amp4(o.amplitude(), dirs))
        local_S = torch.from_numpy(o.spectrum())
        multi.allreduce_amplitude(amp4)               # the one exchange of the path
        dist.all_reduce(local_S)                      # the WRONG way, for contrast
        np.save(os.path.join(out_dir, f"amp4_rank{rank}.npy"), amp4.numpy())
        if rank == 0:
            np.save(os.path.join(out_dir, "sum_of_intensities.npy"), local_S.numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_amplitude_allreduce_matches_single_process(tmp_path, oracle_mod, world):
    n = 301                                           # 3 ranks: shards of 101, 100, 100 particles
    mp.spawn(_worker, args=(world, _free_port(), n, str(tmp_path)), nprocs=world, join=True)
    w, dirs, omega = _grid()
    o = oracle_mod.Oracle(dirs, omega, w.dt, scale=1.0)
    for t, st in w.steps(n_steps=2, n_particles=n):
        o.accumulate_step(t, *st)
    ref4 = to_amp4(o.amplitude(), dirs)
    amps = [np.load(tmp_path / f"amp4_rank{r}.npy") for r in range(world)]
    for a in amps[1:]:
        assert np.array_equal(a, amps[0])             # every rank holds the same sum
    assert np.allclose(amps[0], ref4, rtol=0, atol=1e-12 * np.abs(ref4).max())
    S = (amps[0] ** 2).sum(axis=-1)                   # |A1|^2 + |A2|^2 == |A|^2 because A _|_ n
    assert np.allclose(S, o.spectrum(), rtol=1e-10)
    wrong = np.load(tmp_path / "sum_of_intensities.npy")
    assert not np.allclose(wrong, o.spectrum(), rtol=1e-3)


def test_transverse_basis_is_orthonormal_and_carries_the_whole_amplitude(oracle_mod):
    """A = n x (...) is perpendicular to n, so two components on (e1, e2) lose nothing."""
    w, dirs, omega = _grid()
    n, e1, e2 = transverse_basis(dirs)
    for a, b in ((n, e1), (n, e2), (e1, e2)):
        assert np.abs(np.einsum("dc,dc->d", a, b)).max() < 1e-15
    assert np.allclose(np.cross(e1, e2), n, atol=1e-15)
    o = oracle_mod.Oracle(dirs, omega, w.dt, scale=1.0)
    for t, st in w.steps(n_steps=1, n_particles=50):
        o.accumulate_step(t, *st)
    A = o.amplitude()
    assert np.abs(np.einsum("dwc,dc->dw", A, n)).max() <= 1e-12 * np.abs(A).max()
    a4 = to_amp4(A, dirs)
    back = (a4[..., 0] + 1j * a4[..., 1])[..., None] * e1[:, None, :] + (a4[..., 2] + 1j * a4[..., 3])[..., None] * e2[:, None, :]
    assert np.abs(back - A).max() <= 1e-12 * np.abs(A).max()
