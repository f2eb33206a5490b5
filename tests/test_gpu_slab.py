"""GPU parity of the row-slab decomposition: a lattice cut into 1-4 slabs, all resident on the one
GPU (gpuqt_slab_group; the slabs' steps are interleaved with the halo pushes exactly as on several GPUs, only the
cross-GPU flags are not exercised), against the CPU oracle of the WHOLE lattice -- moments, evolved states, VAC and
MSD, at 1e-10 in the A22 norms -- and bit-identical to itself from run to run.
"""
import numpy as np
import pytest

from workloads import lattices as L

pytestmark = pytest.mark.gpu
TOL = 1e-10


@pytest.fixture(scope="module")
def gq():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1705_01387_b200 as g
    return g


def vec_err(a, b):
    return np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300)


CASES = [
    # (model, batch, n_slabs)
    (L.cubic(12, W=16.5, seed=4, energy_scale=16.0), 4, 3),          # constant hopping, K = 6, planes as halos
    (L.square(70, 37, W=2.0, seed=3), 1, 4),                          # B = 1 two-slice tiles, ragged last slice
    (L.graphene(29, 17, vacancy_fraction=0.03, vacancy_seed=9), 2, 2),  # ragged rows (0-3 neighbours)
    (L.square_peierls(45, 31, flux_quanta=3, W=1.5, seed=7), 8, 3),   # complex hoppings, B = 8
    (L.with_bond_disorder(L.square(52, 33, W=1.0, seed=13), 0.5, 21), 4, 2),   # per-entry real hoppings
    (L.chain(3001, W=1.0, seed=8), 2, 4),                             # K = 2, two halo rows per slab
    (L.cubic(12, W=16.5, seed=4, energy_scale=16.0), 4, 1),          # one slab: no halo at all
]
IDS = [f"{m.name}-B{b}-S{s}" for m, b, s in CASES]


@pytest.mark.parametrize("model,batch,n_slabs", CASES, ids=IDS)
def test_slabs_match_the_oracle(gq, oracle_mod, model, batch, n_slabs):
    from paper_1705_01387_b200 import slab
    nm, order, dt = 48, 24, 0.7
    phi = L.random_phase_vectors(model.N, batch, 81, 0)
    slabs = slab.partition(model, n_slabs)
    g = slab.SlabGroup(model, slabs, batch=batch, modes=gq.MODE_VAC | gq.MODE_MSD)
    o = oracle_mod.Oracle(model, batch=batch, modes=oracle_mod.MODE_VAC | oracle_mod.MODE_MSD)
    g.set_state(phi)
    o.set_state(phi)
    assert np.max(np.abs(g.dos_moments(nm) - o.dos_moments(nm))) / model.N <= TOL
    for step in range(3):
        va, vb = o.get_state(oracle_mod.VAC_A), o.get_state(oracle_mod.VAC_B)
        scale = np.array([np.linalg.norm(o.apply_v(va[b])) * np.linalg.norm(vb[b]) for b in range(batch)])
        assert np.max(np.abs(g.vac(nm) - o.vac(nm)) / scale[:, None]) <= TOL, f"VAC moments at step {step}"
        g.evolve(dt, order)
        o.evolve(dt, order)
        chi = o.get_state(oracle_mod.CHI)
        assert np.max(np.abs(g.msd(nm) - o.msd(nm)) / np.sum(chi * chi, axis=(1, 2))[:, None]) <= TOL, f"MSD moments at step {step}"
    for which, ow in ((gq.STATE_PSI, oracle_mod.PSI), (gq.STATE_CHI, oracle_mod.CHI), (gq.STATE_VAC_A, oracle_mod.VAC_A),
                      (gq.STATE_VAC_B, oracle_mod.VAC_B)):
        assert vec_err(g.get_state(which, model.N), o.get_state(ow)) <= TOL, f"state {which}"
    g.close()
    o.close()


def test_slab_count_does_not_change_the_states_beyond_rounding(gq):
    """1, 2 and 4 slabs evolve the same vectors: the owned rows are computed by the same kernel on the same operands
    in the same neighbour order, so the states agree bit for bit; the moments differ only by the order of the partial sums."""
    from paper_1705_01387_b200 import slab
    model = L.cubic(12, W=16.5, seed=4, energy_scale=16.0)
    phi = L.random_phase_vectors(model.N, 4, 82, 0)
    states, moments = [], []
    for n_slabs in (1, 2, 4):
        g = slab.SlabGroup(model, slab.partition(model, n_slabs), batch=4, modes=gq.MODE_MSD)
        g.set_state(phi)
        g.evolve(1.0, 30)
        g.evolve(-0.3, 20)
        states.append((g.get_state(gq.STATE_PSI, model.N), g.get_state(gq.STATE_CHI, model.N)))
        moments.append(g.msd(64))
        again = g.msd(64)
        assert again.tobytes() == moments[-1].tobytes()           # run-to-run identical
        g.close()
    for psi, chi in states[1:]:
        assert psi.tobytes() == states[0][0].tobytes() and chi.tobytes() == states[0][1].tobytes()
    for m in moments[1:]:
        assert np.max(np.abs(m - moments[0])) <= 1e-12 * np.max(np.abs(moments[0]))


def test_slab_group_and_single_handle_agree(gq):
    """The decomposed lattice against the ordinary one-handle path (streaming kernels, one launch per step)."""
    from paper_1705_01387_b200 import slab
    model = L.square(64, 32, W=2.0, seed=15)
    phi = L.random_phase_vectors(model.N, 2, 83, 0)
    h = gq.GpuQT(model, batch=2, modes=gq.MODE_VAC, options={"small": 0, "persistent": 0})
    g = slab.SlabGroup(model, slab.partition(model, 2), batch=2, modes=gq.MODE_VAC)
    h.set_state(phi)
    g.set_state(phi)
    h.evolve(0.5, 16)
    g.evolve(0.5, 16)
    assert g.get_state(gq.STATE_VAC_B, model.N).tobytes() == h.get_state(gq.STATE_VAC_B).tobytes()
    a, b = g.vac(40), h.vac(40)
    assert np.max(np.abs(a - b)) <= 1e-12 * np.max(np.abs(b))
    h.close()
    g.close()


def test_slab_errors(gq):
    from paper_1705_01387_b200 import slab
    model = L.square(64, 32, W=2.0, seed=15)
    g = slab.SlabGroup(model, slab.partition(model, 2), batch=1, modes=gq.MODE_MSD)
    with pytest.raises(gq.GpuqtError):
        g.dos_moments(16)                      # no state yet
    g.set_state(L.random_phase_vectors(model.N, 1, 84, 0))
    with pytest.raises(gq.GpuqtError):
        g.vac(16)                              # created without GPUQT_MODE_VAC
    g.close()
    # a slab whose send target is missing from the group and was never connected
    slabs = slab.partition(model, 2)
    lonely = slab.SlabGroup(model, slabs, mine=[0], batch=1, modes=gq.MODE_PSI)
    lonely.set_state(L.random_phase_vectors(model.N, 1, 84, 0))
    with pytest.raises(gq.GpuqtError, match="not connected"):
        lonely.dos_moments(8, reduce=False)
    lonely.close()


VARIANTS = [
    # (model, batch, n_slabs, options, hop variant expected in every slab or None)
    (L.cubic(12, W=16.5, seed=4, energy_scale=16.0), 4, 3, {"stencil": 2}, 5),     # implicit stencil, columns into halo rows
    (L.square(64, 33, W=2.0, seed=3), 8, 2, {"stencil": 2}, 5),
    (L.cubic(12, W=16.5, seed=4, energy_scale=16.0), 4, 3, {"stencil": 0, "idx16": 0}, 2),   # int32 columns
    (L.cubic(12, W=16.5, seed=4, energy_scale=16.0), 2, 2, {"stencil": 0, "hop_const": 0}, 0),  # per-entry hoppings
    (L.graphene(29, 17, vacancy_fraction=0.03, vacancy_seed=9), 4, 3, {"stencil": 2}, None),  # ragged: stencil must decline
]


@pytest.mark.parametrize("model,batch,n_slabs,options,hop", VARIANTS,
                         ids=[f"{m.name}-B{b}-S{s}-{'-'.join(f'{k}{v}' for k, v in o.items())}" for m, b, s, o, _ in VARIANTS])
def test_slab_storage_variants_match_the_oracle(gq, oracle_mod, model, batch, n_slabs, options, hop):
    """gpuqt_slab_create_with_options: the storage variants of the records (implicit stencil, 16-bit / 32-bit columns,
    per-entry hoppings) on slabs, whose columns reach into the halo rows behind the owned rows."""
    from paper_1705_01387_b200 import slab
    nm, order, dt = 40, 20, 0.6
    phi = L.random_phase_vectors(model.N, batch, 85, 0)
    g = slab.SlabGroup(model, slab.partition(model, n_slabs), batch=batch, modes=gq.MODE_VAC | gq.MODE_MSD, options=options)
    if hop is not None:
        assert g.hop_variants() == [hop] * n_slabs
    o = oracle_mod.Oracle(model, batch=batch, modes=oracle_mod.MODE_VAC | oracle_mod.MODE_MSD)
    g.set_state(phi)
    o.set_state(phi)
    assert np.max(np.abs(g.dos_moments(nm) - o.dos_moments(nm))) / model.N <= TOL
    g.evolve(dt, order)
    o.evolve(dt, order)
    va, vb = o.get_state(oracle_mod.VAC_A), o.get_state(oracle_mod.VAC_B)
    scale = np.array([np.linalg.norm(o.apply_v(va[b])) * np.linalg.norm(vb[b]) for b in range(batch)])
    assert np.max(np.abs(g.vac(nm) - o.vac(nm)) / scale[:, None]) <= TOL
    chi = o.get_state(oracle_mod.CHI)
    assert np.max(np.abs(g.msd(nm) - o.msd(nm)) / np.sum(chi * chi, axis=(1, 2))[:, None]) <= TOL
    for which, ow in ((gq.STATE_PSI, oracle_mod.PSI), (gq.STATE_CHI, oracle_mod.CHI), (gq.STATE_VAC_B, oracle_mod.VAC_B)):
        assert vec_err(g.get_state(which, model.N), o.get_state(ow)) <= TOL, f"state {which}"
    g.close()
    o.close()


def test_vac_only_group_answers_dos_moments(gq, oracle_mod):
    """gpuqt_slab_dos_moments behaves as gpuqt_dos_moments: psi is set in every mode."""
    from paper_1705_01387_b200 import slab
    model = L.square(40, 30, W=2.0, seed=1)
    phi = L.random_phase_vectors(model.N, 2, 86, 0)
    g = slab.SlabGroup(model, slab.partition(model, 2), batch=2, modes=gq.MODE_VAC)
    h = gq.GpuQT(model, batch=2, modes=gq.MODE_VAC)
    o = oracle_mod.Oracle(model, batch=2, modes=oracle_mod.MODE_VAC)
    for x in (g, h, o):
        x.set_state(phi)
    ref = o.dos_moments(32)
    assert np.max(np.abs(g.dos_moments(32) - ref)) / model.N <= TOL
    assert np.max(np.abs(h.dos_moments(32) - ref)) / model.N <= TOL
    g.close()
    h.close()
    o.close()


def test_connect_checks_and_a_peer_that_never_arrives(gq):
    """Two groups on this one GPU, linked with plain device addresses (same process, so no IPC mapping is needed):
    gpuqt_slab_connect refuses segments outside the peer's halo and its own slabs; a group whose peer never makes
    the matching calls gives up after the wait budget with GPUQT_ERR_STATE instead of hanging, and is unusable
    afterwards.  Only ONE group issues work here -- nothing on the GPU waits for another kernel to run."""
    from paper_1705_01387_b200 import slab
    model = L.square(64, 32, W=2.0, seed=15)
    slabs = slab.partition(model, 2)
    a = slab.SlabGroup(model, slabs, mine=[0], batch=1, modes=gq.MODE_PSI)
    b = slab.SlabGroup(model, slabs, mine=[1], batch=1, modes=gq.MODE_PSI)
    bufs, flags, n_own, n_halo = b.export(0)
    assert (n_own, n_halo) == (slabs[1].n_own, slabs[1].n_halo)
    with pytest.raises(gq.GpuqtError) as ei:
        a.connect(1, bufs, flags, n_own + 1, n_halo)              # the first halo row would be an owned row there
    assert ei.value.status == -2
    with pytest.raises(gq.GpuqtError) as ei:
        a.connect(1, bufs, flags, n_own, n_halo - 1)              # the last segment would run past the halo
    assert ei.value.status == -2
    with pytest.raises(gq.GpuqtError) as ei:
        a.connect(0, bufs, flags, n_own, n_halo)                  # slab 0 is a's own
    assert ei.value.status == -1
    with pytest.raises(gq.GpuqtError):
        a.set_wait_budget(0.0)
    a.set_state(L.random_phase_vectors(model.N, 1, 84, 0))
    with pytest.raises(gq.GpuqtError, match="not connected"):
        a.dos_moments(4, reduce=False)                            # refused before any work: the group stays usable
    a.connect(1, bufs, flags, n_own, n_halo)
    a.set_wait_budget(0.05)
    with pytest.raises(gq.GpuqtError, match="did not arrive") as ei:
        a.dos_moments(4, reduce=False)                            # b never publishes its flags
    assert ei.value.status == -6
    with pytest.raises(gq.GpuqtError, match="unusable") as ei:
        a.dos_moments(4, reduce=False)
    assert ei.value.status == -6
    with pytest.raises(gq.GpuqtError, match="unusable"):
        a.evolve(0.1, 4)
    a.close()
    b.close()


def test_duplicate_global_ids_are_refused(gq):
    from paper_1705_01387_b200 import slab
    model = L.square(64, 32, W=2.0, seed=15)
    slabs = slab.partition(model, 2)
    slabs[1].global_id = 0
    with pytest.raises(gq.GpuqtError, match="two local slabs"):
        slab.SlabGroup(model, slabs, batch=1, modes=gq.MODE_PSI)
