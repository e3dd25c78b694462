"""Host logic of the spaxel-sharded forward (paper_2412_08265_b200/sharded.py) on CPU: the row
partitioner, the routing of particles to row owners, the all-to-all and the halo exchange -- with the fp64 oracle as the
compute backend, against the single-rank oracle cube.  World size 2 over gloo (two processes), and 1-5 ranks as threads."""
import dataclasses
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_2412_08265_b200 import sharded, synth
from sharded_backend import OracleBackend


def workload(n=900, psf=True):
    w = synth.make_workload("tiny", n=n)
    if psf:
        w.telescope = dataclasses.replace(w.telescope.with_psf_lsf(psf_size=7, lsf_size=5), n_channels=64)
    else:
        w.telescope = dataclasses.replace(w.telescope, n_channels=64)
    return w


def run_rank(comm, w, fuse_halo=True):
    p = w.particles
    sl = sharded.slice_for_rank(p.n, comm.rank, comm.world)
    rec = sharded.pack_records(p.subset(np.arange(p.n)[sl]), "cpu")
    return sharded.forward_sharded(comm, OracleBackend(), rec, w.rotation, w.ssp, w.telescope, fuse_halo=fuse_halo)


def check_slabs(slabs, w):
    ref = oracle.forward(w.particles, w.rotation, w.ssp, w.telescope)
    t = w.telescope
    assert slabs[0].x0 == 0 and slabs[-1].x1 == t.n_x
    covered = 0
    for a, b in zip(slabs[:-1], slabs[1:]):
        assert a.x1 == b.x0 and np.array_equal(a.bounds, b.bounds)
    for s in slabs:
        got = s.cube.numpy()
        assert got.shape == (s.x1 - s.x0, t.n_y, t.n_channels)
        assert np.abs(got - ref[s.x0:s.x1]).max() <= 1e-12 * np.abs(ref).max()
        covered += s.x1 - s.x0
    assert covered == t.n_x
    key, _ = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    assert sum(s.n_received for s in slabs) == int((key < t.n_spaxels).sum())      # every in-FoV particle has one owner


# ------------------------------------------------------------------------------------------ partitioner
def test_partition_balances_cost_and_respects_min_rows():
    counts = np.array([0, 0, 5, 40, 300, 900, 280, 35, 6, 0, 0, 0])
    for world in (1, 2, 3, 4):
        for min_rows in (1, 3):
            if world * min_rows > counts.size:
                continue
            b = sharded.partition_rows(counts, world, min_rows=min_rows, row_cost=2.0)
            assert b[0] == 0 and b[-1] == counts.size and (np.diff(b) >= min_rows).all()
    b = sharded.partition_rows(counts, 2)
    left, right = counts[:b[1]].sum(), counts[b[1]:].sum()
    assert abs(left - right) <= counts.max()                      # as even as one row allows
    uniform = sharded.partition_rows(np.full(300, 10.0), 8)
    assert np.diff(uniform).min() >= 37 and np.diff(uniform).max() <= 38
    empty = sharded.partition_rows(np.zeros(16), 4, min_rows=3, row_cost=1.0)
    assert np.array_equal(empty, [0, 4, 8, 12, 16])
    with pytest.raises(ValueError):
        sharded.partition_rows(counts, 5, min_rows=3)


def test_owner_of_rows():
    bounds = np.array([0, 3, 3 + 4, 16])
    rows = torch.arange(16)
    assert sharded.owner_of_rows(rows, bounds).tolist() == [0] * 3 + [1] * 4 + [2] * 9


# ------------------------------------------------------------------------------------------ ranks as threads
@pytest.mark.parametrize("world", [1, 2, 3, 5])
@pytest.mark.parametrize("psf", [True, False])
@pytest.mark.parametrize("fuse_halo", [True, False])
def test_thread_ranks_reproduce_the_single_rank_cube(world, psf, fuse_halo):
    """fuse_halo: the boundary rows reach the neighbours through mirror stores of the build (thread ranks share an address
    space) or through the explicit halo exchange (what separate processes do)."""
    w = workload(psf=psf)
    if psf and world == 5:
        w.telescope = dataclasses.replace(w.telescope, psf_size=5)           # 16 rows / 5 ranks: halo of 2 rows
    slabs = sharded.run_threads(world, lambda comm: run_rank(comm, w, fuse_halo))
    check_slabs(slabs, w)


def test_all_particles_in_one_row_and_an_empty_rank_slice():
    w = workload(n=40)
    w.particles.pos[:] = 0.01                                   # everything in one spaxel; ranks 2.. hold no particles of it
    w.rotation = np.eye(3, dtype=np.float32)
    slabs = sharded.run_threads(2, lambda comm: run_rank(comm, w))
    check_slabs(slabs, w)
    w2 = workload(n=3)                                          # fewer particles than ranks: some slices are empty
    check_slabs(sharded.run_threads(4, lambda comm: run_rank(comm, dataclasses.replace(
        w2, telescope=dataclasses.replace(w2.telescope, psf_size=3)))), dataclasses.replace(
        w2, telescope=dataclasses.replace(w2.telescope, psf_size=3)))


# ------------------------------------------------------------------------------------------ two processes over gloo
def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = workload()
        slab = run_rank(sharded.DistComm(), w)
        out.put((rank, slab.x0, slab.x1, slab.cube.numpy(), slab.bounds, slab.n_received))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_ranks_over_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=300) for _ in range(world)), key=lambda v: v[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    slabs = [sharded.Slab(x0, x1, torch.from_numpy(c), b, n) for _, x0, x1, c, b, n in res]
    check_slabs(slabs, workload())
