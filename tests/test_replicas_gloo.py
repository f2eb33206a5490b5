"""N>1 path on CPU: replicas over random vectors with world_size 2 over gloo.

The GPU compute of a rank is stood in for by the oracle (tests may call it); what is under test is
the host plumbing of paper_1705_01387_b200/replicas.py that bench.py uses at N>1: which vectors a
rank owns, the gather of the moment blocks in global vector order, the average over all vectors and
the max-over-ranks timing.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from workloads import lattices as L

WORLD, BATCH, NM, CONFIG = 2, 2, 24, 61


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _model():
    return L.square(24, 18, W=2.0, seed=11)


def _worker(rank, port, ret):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), LOCAL_RANK=str(rank),
                      WORLD_SIZE=str(WORLD), OMP_NUM_THREADS="1")
    dist.init_process_group("gloo", rank=rank, world_size=WORLD)
    try:
        from oracle import oracle
        from paper_1705_01387_b200 import replicas
        r, _, w = replicas.world()
        assert (r, w) == (rank, WORLD)
        model = _model()
        phi = L.random_phase_vectors(model.N, BATCH, CONFIG, replicas.first_vector(r, BATCH))
        o = oracle.Oracle(model, batch=BATCH, modes=0)
        o.set_state(phi)
        local = torch.from_numpy(o.dos_moments(NM))
        allm = replicas.gather_moments(local)
        mean = replicas.mean_over_vectors(local)
        tmax = replicas.max_over_ranks(10.0 + rank)
        if rank == 0:
            ret["all"], ret["mean"], ret["tmax"] = allm.numpy().copy(), mean.numpy().copy(), tmax
    finally:
        dist.destroy_process_group()


def test_replicas_over_vectors_world2():
    from oracle import oracle
    from paper_1705_01387_b200 import replicas
    oracle.build()
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(_free_port(), ret), nprocs=WORLD, join=True)
    model = _model()
    phi = L.random_phase_vectors(model.N, WORLD * BATCH, CONFIG, 0)
    o = oracle.Oracle(model, batch=WORLD * BATCH, modes=0)
    o.set_state(phi)
    ref = o.dos_moments(NM)
    assert ret["all"].shape == (WORLD * BATCH, NM)
    assert ret["all"].tobytes() == ref.tobytes()            # same vectors, same order, untouched by the gather
    assert np.allclose(ret["mean"], ref.mean(axis=0), rtol=0, atol=1e-12 * model.N)
    assert ret["tmax"] == 11.0
    for v in range(WORLD * BATCH):
        rk, slot = replicas.vector_owner(v, BATCH)
        assert replicas.first_vector(rk, BATCH) + slot == v


def test_single_process_is_identity():
    from paper_1705_01387_b200 import replicas
    t = torch.arange(6, dtype=torch.float64).reshape(2, 3)
    assert replicas.gather_moments(t) is t
    assert replicas.max_over_ranks(3.5) == 3.5
    assert torch.equal(replicas.mean_over_vectors(t), t.mean(dim=0))


def test_vector_streams_are_disjoint():
    """first_vector offsets give every rank different random vectors, and a rank's block is a
    slice of the global sequence."""
    N = 100
    allv = L.random_phase_vectors(N, 4, CONFIG, 0)
    r1 = L.random_phase_vectors(N, 2, CONFIG, 2)
    assert r1.tobytes() == allv[2:4].tobytes()
    assert not np.array_equal(allv[0], allv[2])


def test_bench_starts_its_own_ranks():
    """bench.py --gpus N outside torchrun re-executes itself as N ranks with the contract's launch line."""
    from paper_1705_01387_b200 import replicas
    assert not replicas.needs_launch(1, env={})
    assert replicas.needs_launch(8, env={})
    assert not replicas.needs_launch(8, env={"WORLD_SIZE": "8"})
    cmd = replicas.launch_command("/x/bench.py", ["--gpus", "4", "--steps", "2"], 4, 29512, python="python")
    assert cmd == ["python", "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=4", "--master-addr", "127.0.0.1",
                   "--master-port", "29512", "/x/bench.py", "--gpus", "4", "--steps", "2"]
    assert 1024 < replicas.free_port() < 65536
