"""N > 1 host logic on CPU: world_size-2 gloo (replicas only).

Covers what `bench.py --gpus N` does besides launching kernels: each rank draws its own galaxy,
nothing is exchanged on the data path, the elapsed time is reduced with MAX over ranks and the
whole-job value is world x per-rank units / slowest time.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2412_08265_b200 import replicas, synth


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        seed = replicas.replica_seed(0, rank)
        w = synth.make_workload("tiny", seed=seed)
        # pretend rank r took (10 + 5 r) ms for 4 steps
        mine = 10.0 + 5.0 * rank
        slowest = replicas.max_over_ranks(mine)
        # digest of this rank's galaxy, gathered only to CHECK that replicas differ (not data path)
        digest = torch.tensor([float(np.float64(w.particles.pos).sum())], dtype=torch.float64)
        all_d = [torch.zeros_like(digest) for _ in range(world)]
        dist.all_gather(all_d, digest)
        dist.barrier()
        out.put((rank, seed, slowest, [float(d.item()) for d in all_d], w.particles.n))
    finally:
        dist.destroy_process_group()


def test_two_rank_replicas_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, m0, d0, n0), (r1, s1, m1, d1, n1) = res
    assert (r0, r1) == (0, 1)
    assert s0 == 1000 and s1 == 1010                     # rank 0 = the config's own galaxy
    assert m0 == m1 == 15.0                              # MAX over ranks, same on every rank
    assert d0 == d1 and d0[0] != d0[1]                   # two different galaxies
    assert n0 == n1 == 1000                              # weak scaling: fixed work per rank
    v = replicas.whole_job_value(n0 * 256, world, m0, steps=4)
    assert v == pytest.approx(2 * 1000 * 256 * 4 / 15e-3)


def test_rank0_galaxy_is_the_config_galaxy():
    a = synth.make_workload("tiny")
    b = synth.make_workload("tiny", seed=replicas.replica_seed(0, 0))
    assert np.array_equal(a.particles.pos, b.particles.pos)
    assert np.array_equal(a.particles.mass, b.particles.mass)


def test_single_process_is_identity():
    assert replicas.max_over_ranks(3.25) == 3.25
    with pytest.raises(ValueError):
        replicas.whole_job_value(1.0, 2, 0.0, 1)
    with pytest.raises(ValueError):
        replicas.replica_seed(0, -1)
