"""Row-slab decomposition, host side (no GPU): paper_1705_01387_b200/slab.py.

* the slabs' local tables + halo lists reproduce the global H exactly (dense comparison),
* every send segment fills exactly the halo rows of the receiver that the sender owns,
* world_size 2 over gloo: each rank holds one slab, runs the Chebyshev moment recurrence
  T_m = 2 H~ T_{m-1} - T_{m-2} on its owned rows with numpy, exchanges halo rows following the send segments
  (isend / irecv in the order the library pushes them) and all-reduces its partial inner products with
  slab.sum_over_ranks; the result must equal the oracle's moments of the whole lattice.  The rank-local
  arithmetic here is a stand-in written for the test; what is under test is the decomposition bookkeeping
  that the CUDA slabs use unchanged (tests/test_gpu_slab.py covers those against the oracle on the GPU).
"""
import ctypes as C
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from tests import dense_ref
from workloads import lattices as L


def models():
    return [
        L.cubic(8, W=2.0, seed=3, energy_scale=8.0),
        L.square(24, 18, W=2.0, seed=11),
        L.graphene(12, 9, vacancy_fraction=0.04, vacancy_seed=5),
        L.square_peierls(16, 12, flux_quanta=2, W=1.0, seed=7),
        L.chain(301, W=1.0, seed=8),
    ]


def dense_from_slabs(model, slabs):
    N, K = model.N, model.K
    H = np.zeros((N, N), complex)
    for s in slabs:
        glob = np.concatenate([np.arange(s.row0, s.row1), s.halo_global])
        idx = s.nbr_index.reshape(s.n_own, K)
        for r in range(s.n_own):
            if s.onsite is not None:
                H[s.row0 + r, s.row0 + r] += s.onsite[r]
            for k in range(s.nbr_count[r]):
                h = (-1.0 if s.hop_re is None else s.hop_re[r * K + k]) + 1j * (0.0 if s.hop_im is None else s.hop_im[r * K + k])
                H[s.row0 + r, glob[idx[r, k]]] += h
    return H


@pytest.mark.parametrize("n_slabs", [1, 2, 3, 5])
@pytest.mark.parametrize("model", models(), ids=lambda m: m.name)
def test_slabs_reproduce_the_global_matrix(model, n_slabs):
    from paper_1705_01387_b200 import slab
    slabs = slab.partition(model, n_slabs)
    assert [s.row0 for s in slabs][0] == 0 and slabs[-1].row1 == model.N
    assert all(a.row1 == b.row0 for a, b in zip(slabs, slabs[1:]))
    assert all(s.row0 % 32 == 0 for s in slabs)
    H = dense_ref.dense_H(model)
    assert np.array_equal(dense_from_slabs(model, slabs), H)
    for s in slabs:
        # halo rows are rows of other slabs, ascending, each referenced at least once; x follows the same order
        assert np.all((s.halo_global < s.row0) | (s.halo_global >= s.row1))
        assert np.all(np.diff(s.halo_global) > 0)
        used = s.nbr_index.reshape(s.n_own, model.K)[np.arange(model.K)[None, :] < s.nbr_count[:, None]]
        assert set(used[used >= s.n_own] - s.n_own) == set(range(s.n_halo))
        assert np.array_equal(s.x, np.concatenate([model.x[s.row0:s.row1], model.x[s.halo_global]]))


@pytest.mark.parametrize("model", models(), ids=lambda m: m.name)
def test_send_segments_fill_every_halo_row_once(model):
    from paper_1705_01387_b200 import slab
    slabs = slab.partition(model, 4)
    filled = {s.global_id: np.zeros(s.n_halo, int) for s in slabs}
    for p in slabs:
        for peer, rows, dst0 in p.sends:
            q = slabs[peer]
            assert peer != p.global_id and rows.dtype == np.int32
            assert np.all((rows >= 0) & (rows < p.n_own))
            seg = slice(dst0 - q.n_own, dst0 - q.n_own + rows.size)
            assert np.array_equal(q.halo_global[seg], p.row0 + rows)
            filled[peer][seg] += 1
    for s in slabs:
        assert np.all(filled[s.global_id] == 1)
        # Hermitian H [A10]: the slabs I send to are the slabs that send to me
        senders = {p.global_id for p in slabs for peer, _, _ in p.sends if peer == s.global_id}
        assert senders == {peer for peer, _, _ in s.sends}


def test_partition_rejects_too_many_slabs():
    from paper_1705_01387_b200 import slab
    with pytest.raises(ValueError):
        slab.partition(L.chain(40, W=0.0, seed=1), 3)
    assert slab.slabs_of_rank(5, 1, 2) == [3, 4] and slab.slabs_of_rank(4, 0, 4) == [0]


def test_ipc_handle_survives_nul_bytes():
    """A cudaIpcMemHandle is 64 bytes of binary data; the marshalling in slab.connect_ranks must carry every byte,
    NULs included (a c_char array would cut it at the first NUL), and refuse a handle of another length."""
    from paper_1705_01387_b200 import slab
    raw = bytes([7, 0, 0, 9] + [0] * 28 + list(range(32)))
    assert len(raw) == 64 and raw[1] == 0
    h = slab._handle_from_bytes(raw)
    assert C.sizeof(h) == 64
    assert slab._handle_to_bytes(h) == raw
    assert bytes(h.reserved) == raw
    assert slab._handle_to_bytes(slab._IpcHandle()) == bytes(64)
    with pytest.raises(ValueError):
        slab._handle_from_bytes(raw[:2])


# ------------------------------------------------------------------------------- world_size 2 over gloo
WORLD, NM, CONFIG = 2, 20, 71


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _gloo_model():
    return L.square_peierls(20, 16, flux_quanta=2, W=1.0, seed=9)


def _exchange(me, slabs, vec):
    """vec: complex [n_own + n_halo] of slab `me`; fills its halo rows from the owners, sends what they need."""
    reqs, bufs = [], []
    for peer, rows, _ in me.sends:
        t = torch.from_numpy(np.ascontiguousarray(vec[rows]).view(np.float64).copy())
        reqs.append(dist.isend(t, dst=peer))
    for p in slabs:
        for peer, rows, dst0 in p.sends:
            if peer == me.global_id:
                t = torch.empty(2 * rows.size, dtype=torch.float64)
                reqs.append(dist.irecv(t, src=p.global_id))
                bufs.append((dst0, rows.size, t))
    for r in reqs:
        r.wait()
    for dst0, n, t in bufs:
        vec[dst0:dst0 + n] = t.numpy().view(np.complex128)


def _worker(rank, port, ret):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), LOCAL_RANK=str(rank),
                      WORLD_SIZE=str(WORLD), OMP_NUM_THREADS="1")
    dist.init_process_group("gloo", rank=rank, world_size=WORLD)
    try:
        from paper_1705_01387_b200 import slab
        model = _gloo_model()
        slabs = slab.partition(model, WORLD)
        me = slabs[slab.slabs_of_rank(WORLD, rank, WORLD)[0]]
        K, n, dE = model.K, me.n_own, model.energy_scale
        idx = me.nbr_index.reshape(n, K)
        hop = me.hop_re.reshape(n, K) + 1j * me.hop_im.reshape(n, K)
        mask = np.arange(K)[None, :] < me.nbr_count[:, None]

        def h_tilde(v):          # owned rows of H~ v from the local (owned + halo) vector
            g = np.where(mask, v[np.where(mask, idx, 0)] * hop, 0.0).sum(axis=1)
            return (g + me.onsite * v[:n]) / dE

        phi = L.random_phase_vectors(model.N, 1, CONFIG, 0)[0]
        phi = phi[:, 0] + 1j * phi[:, 1]
        t0 = np.zeros(n + me.n_halo, complex)
        t0[:n] = phi[me.row0:me.row1]
        _exchange(me, slabs, t0)
        t1 = np.zeros_like(t0)
        t1[:n] = h_tilde(t0)
        left = t0[:n].conj()
        part = [np.vdot(t0[:n], t0[:n]).real, (left @ t1[:n]).real]
        for _ in range(2, NM):
            _exchange(me, slabs, t1)
            t2 = np.zeros_like(t0)
            t2[:n] = 2.0 * h_tilde(t1) - t0[:n]
            part.append((left @ t2[:n]).real)
            t0, t1 = t1, t2
        total = slab.sum_over_ranks(np.array([part]))
        if rank == 0:
            ret["moments"] = total.copy()
    finally:
        dist.destroy_process_group()


def test_two_ranks_one_slab_each_match_the_oracle():
    from oracle import oracle
    oracle.build()
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(_free_port(), ret), nprocs=WORLD, join=True)
    model = _gloo_model()
    o = oracle.Oracle(model, batch=1, modes=0)
    o.set_state(L.random_phase_vectors(model.N, 1, CONFIG, 0))
    ref = o.dos_moments(NM)
    assert np.max(np.abs(ret["moments"] - ref)) / model.N <= 1e-12
