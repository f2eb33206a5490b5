"""The cross-GPU half of the row-slab decomposition: two processes, one GPU and one slab each, linked
by slab.connect_ranks (CUDA IPC mappings of the peer's vector buffers and flag array; the halo pushes are stores into
the peer GPU's memory, ordered by st.release.sys / ld.acquire.sys flags), against the CPU oracle of the WHOLE lattice.

Needs two CUDA devices with peer access; skipped otherwise -- which is every box this repository has been run on so
far (gpurun and the round-end driver give one GPU), so this file is the recipe for the first box that has two, not a
record of a run.  The one-GPU emulation of the same decomposition is tests/test_gpu_slab.py.
"""
import os
import socket

import numpy as np
import pytest

from workloads import lattices as L

pytestmark = pytest.mark.gpu
TOL = 1e-10
WORLD, NM, ORDER, DT, BATCH = 2, 40, 20, 0.6, 2


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _model():
    return L.square(64, 33, W=2.0, seed=15)


def _worker(rank, port, ret):
    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), LOCAL_RANK=str(rank),
                      WORLD_SIZE=str(WORLD))
    torch.cuda.set_device(rank)
    dist.init_process_group("gloo", rank=rank, world_size=WORLD)
    try:
        import paper_1705_01387_b200 as gq
        from oracle import oracle
        from paper_1705_01387_b200 import slab
        model = _model()
        phi = L.random_phase_vectors(model.N, BATCH, 87, 0)
        slabs = slab.partition(model, WORLD)
        g = slab.SlabGroup(model, slabs, mine=slab.slabs_of_rank(WORLD, rank, WORLD), batch=BATCH,
                           modes=gq.MODE_VAC | gq.MODE_MSD)
        g.set_wait_budget(300.0)                   # the ranks drift apart while each runs the oracle on its host cores
        slab.connect_ranks(g)
        o = oracle.Oracle(model, batch=BATCH, modes=oracle.MODE_VAC | oracle.MODE_MSD)
        g.set_state(phi)
        o.set_state(phi)
        errs = {"dos": float(np.max(np.abs(g.dos_moments(NM) - o.dos_moments(NM))) / model.N)}
        for step in range(2):
            va, vb = o.get_state(oracle.VAC_A), o.get_state(oracle.VAC_B)
            scale = np.array([np.linalg.norm(o.apply_v(va[b])) * np.linalg.norm(vb[b]) for b in range(BATCH)])
            errs[f"vac{step}"] = float(np.max(np.abs(g.vac(NM) - o.vac(NM)) / scale[:, None]))
            g.evolve(DT, ORDER)
            o.evolve(DT, ORDER)
            chi = o.get_state(oracle.CHI)
            errs[f"msd{step}"] = float(np.max(np.abs(g.msd(NM) - o.msd(NM)) / np.sum(chi * chi, axis=(1, 2))[:, None]))
        mine = slabs[rank]
        for which, ow, name in ((gq.STATE_PSI, oracle.PSI, "psi"), (gq.STATE_CHI, oracle.CHI, "chi"),
                                (gq.STATE_VAC_B, oracle.VAC_B, "vac_b")):
            got = g.get_state(which, model.N)[:, mine.row0:mine.row1]
            ref = o.get_state(ow)[:, mine.row0:mine.row1]
            errs[name] = float(np.max(np.abs(got - ref)) / np.max(np.abs(ref)))
        ret[rank] = errs
        dist.barrier()
        g.close()
        o.close()
    finally:
        dist.destroy_process_group()


def test_two_gpus_one_slab_each_match_the_oracle():
    import torch
    if not torch.cuda.is_available() or torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices (cross-GPU halo exchange over CUDA IPC)")
    if not torch.cuda.can_device_access_peer(0, 1):
        pytest.skip("devices 0 and 1 have no peer access")
    import torch.multiprocessing as mp
    from oracle import oracle
    oracle.build()
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(_free_port(), ret), nprocs=WORLD, join=True)
    assert sorted(ret.keys()) == [0, 1]
    for rank in range(WORLD):
        for name, err in ret[rank].items():
            assert err <= TOL, (rank, name, err)
