"""GPU parity on random sparse Hermitian graphs (workloads/lattices.py::random_graph): rows of 0 .. K neighbours in
random order, random real or complex hoppings, random on-site energies and positions, sizes from 1 row to a few
thousand with ragged tails, every batch size, all three launch forms -- the storage variants and the generic-width walk
get inputs no lattice produces.  Same norms and tolerance as tests/test_gpu_parity.py (1e-10, A22); the table decode
is bit-exact.
"""
import numpy as np
import pytest

from workloads import lattices as L

pytestmark = pytest.mark.gpu
TOL = 1e-10

PATHS = {"streaming": {"small": 0, "persistent": 0}, "small_path": {"small": 1, "persistent": 0},
         "persistent": {"small": 0, "persistent": 1}}

#        N     K  seed complex fill  locality batch
CASES = [(1,    2, 11, False, 0.7, 0,  1),
         (31,   3, 12, True,  0.9, 0,  2),
         (33,   1, 13, False, 1.0, 0,  4),
         (64,   8, 14, True,  0.6, 9,  8),
         (257,  5, 15, False, 0.8, 0,  1),
         (700,  7, 16, True,  0.9, 50, 4),
         (1500, 6, 17, False, 0.7, 33, 8),
         (2049, 4, 18, True,  0.5, 0,  2),
         (3000, 3, 19, False, 0.9, 64, 1),
         (4100, 2, 20, True,  1.0, 5,  8)]


@pytest.fixture(scope="module")
def gq():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1705_01387_b200 as g
    return g


def vec_err(a, b):
    return np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300)


@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("N,K,seed,cplx,fill,loc,batch", CASES, ids=[f"N{c[0]}-K{c[1]}-B{c[6]}{'-c' if c[3] else ''}" for c in CASES])
def test_random_graph_matches_the_oracle(gq, oracle_mod, N, K, seed, cplx, fill, loc, batch, path):
    model = L.random_graph(N, K, seed, complex_hops=cplx, degree_fill=fill, locality=loc, open_x=(seed % 2 == 1))
    phi = L.random_phase_vectors(model.N, batch, 90 + seed, 0)
    g = gq.GpuQT(model, batch=batch, modes=gq.MODE_VAC | gq.MODE_MSD, options=PATHS[path])
    o = oracle_mod.Oracle(model, batch=batch, modes=oracle_mod.MODE_VAC | oracle_mod.MODE_MSD)
    # table: bit-exact decode of whatever storage variant was chosen
    col, re, im, dx = g.get_table()
    oc, ore, oim, odx = o.get_table()
    assert np.array_equal(col, oc) and re.tobytes() == ore.tobytes() and im.tobytes() == oim.tobytes() and dx.tobytes() == odx.tobytes()
    g.set_state(phi)
    o.set_state(phi)
    nm, order, dt = 40, 18, 0.6
    assert np.max(np.abs(g.dos_moments(nm) - o.dos_moments(nm))) / model.N <= TOL
    for step in range(2):
        va, vb = o.get_state(oracle_mod.VAC_A), o.get_state(oracle_mod.VAC_B)
        scale = np.array([np.linalg.norm(o.apply_v(va[b])) * np.linalg.norm(vb[b]) for b in range(batch)])
        scale = np.where(scale > 0, scale, 1.0)                       # a site without bonds has V phi = 0
        assert np.max(np.abs(g.vac(nm) - o.vac(nm)) / scale[:, None]) <= TOL
        g.evolve(dt if step == 0 else -0.3, order)
        o.evolve(dt if step == 0 else -0.3, order)
        chi = o.get_state(oracle_mod.CHI)
        cs = np.sum(chi * chi, axis=(1, 2))
        cs = np.where(cs > 0, cs, 1.0)
        assert np.max(np.abs(g.msd(nm) - o.msd(nm)) / cs[:, None]) <= TOL
    for which, ow in ((gq.STATE_PSI, oracle_mod.PSI), (gq.STATE_CHI, oracle_mod.CHI), (gq.STATE_VAC_A, oracle_mod.VAC_A),
                      (gq.STATE_VAC_B, oracle_mod.VAC_B)):
        ref = o.get_state(ow)
        if np.max(np.abs(ref)) > 0:
            assert vec_err(g.get_state(which), ref) <= TOL
        else:
            assert np.max(np.abs(g.get_state(which))) == 0.0
    g.close()
    o.close()


@pytest.mark.parametrize("n_slabs", [2, 3])
def test_random_graph_in_slabs(gq, oracle_mod, n_slabs):
    """Non-local random bonds: every slab has halo rows from every other slab, in no particular order."""
    from paper_1705_01387_b200 import slab
    model = L.random_graph(1500, 5, 31, complex_hops=True, degree_fill=0.9, locality=0, open_x=True)
    phi = L.random_phase_vectors(model.N, 2, 95, 0)
    g = slab.SlabGroup(model, slab.partition(model, n_slabs), batch=2, modes=gq.MODE_MSD)
    o = oracle_mod.Oracle(model, batch=2, modes=oracle_mod.MODE_MSD)
    g.set_state(phi)
    o.set_state(phi)
    g.evolve(0.5, 16)
    o.evolve(0.5, 16)
    chi = o.get_state(oracle_mod.CHI)
    assert np.max(np.abs(g.msd(32) - o.msd(32)) / np.sum(chi * chi, axis=(1, 2))[:, None]) <= TOL
    assert vec_err(g.get_state(gq.STATE_CHI, model.N), chi) <= TOL
    g.close()
    o.close()


#           N     K  seed fill loc  batch hop   options
OPT_CASES = [(2048, 6, 51, 1.0, 40,  4, -1.0, {"stencil": 2}),                       # forced pattern dictionary on an irregular table
             (1024, 4, 52, 0.6, 0,   1, -1.0, {"stencil": 2, "persistent": 1, "small": 0}),
             (4096, 3, 53, 0.9, 900, 2, -2.7, {"idx16": 1, "small": 0}),              # 16-bit columns with padding sentinels
             (4096, 3, 53, 0.9, 900, 2, -2.7, {"idx16": 0, "small": 0}),
             (70001, 6, 54, 0.8, 0, 8, -1.0, {"small": 0, "stages": 1}),               # column spread beyond 16 bits -> int32
             (1999, 2, 55, 0.7, 3,   4, 0.5,  {"small": 0, "stages": 4, "run": 32}),
             (2500, 4, 56, 0.9, 100, 1, -1.0, {"small": 0, "persistent": 1, "run": 8, "blocks_per_sm": 1, "alternate": 0}),
             (900,  12, 57, 0.9, 0,  8, None, {"small": 0}),                           # wide rows, complex: generic-width walk
             (300,  16, 58, 1.0, 0,  2, None, {"small": 0, "persistent": 1}),
             (128,  10, 59, 0.8, 0,  4, -1.0, {"hop_const": 0}),                       # constant hopping stored per entry
             ]


@pytest.mark.parametrize("N,K,seed,fill,loc,batch,hop,options", OPT_CASES,
                         ids=[f"N{c[0]}-K{c[1]}-B{c[5]}-" + "_".join(f"{k}{v}" for k, v in c[7].items()) for c in OPT_CASES])
def test_random_graph_storage_variants_and_options(gq, oracle_mod, N, K, seed, fill, loc, batch, hop, options):
    model = L.random_graph(N, K, seed, complex_hops=(hop is None), degree_fill=fill, locality=loc, hop_value=hop)
    phi = L.random_phase_vectors(model.N, batch, 190 + seed, 0)
    g = gq.GpuQT(model, batch=batch, modes=gq.MODE_VAC | gq.MODE_MSD, options=options)
    o = oracle_mod.Oracle(model, batch=batch, modes=oracle_mod.MODE_VAC | oracle_mod.MODE_MSD)
    col, re, im, dx = g.get_table()
    oc, ore, oim, odx = o.get_table()
    assert np.array_equal(col, oc) and re.tobytes() == ore.tobytes() and im.tobytes() == oim.tobytes() and dx.tobytes() == odx.tobytes()
    g.set_state(phi)
    o.set_state(phi)
    nm = 64
    assert np.max(np.abs(g.dos_moments(nm) - o.dos_moments(nm))) / model.N <= TOL
    g.evolve(0.8, 22)
    o.evolve(0.8, 22)
    va, vb = o.get_state(oracle_mod.VAC_A), o.get_state(oracle_mod.VAC_B)
    scale = np.array([np.linalg.norm(o.apply_v(va[b])) * np.linalg.norm(vb[b]) for b in range(batch)])
    assert np.max(np.abs(g.vac(nm) - o.vac(nm)) / scale[:, None]) <= TOL
    chi = o.get_state(oracle_mod.CHI)
    assert np.max(np.abs(g.msd(nm) - o.msd(nm)) / np.sum(chi * chi, axis=(1, 2))[:, None]) <= TOL
    assert vec_err(g.get_state(gq.STATE_CHI), chi) <= TOL
    assert vec_err(g.get_state(gq.STATE_VAC_B), vb) <= TOL
    g.close()
    o.close()


def test_live_handles_sharing_a_kernel_with_different_shared_memory_needs(gq, oracle_mod):
    """Two handles alive at once whose tables run the SAME kernel instantiation (generic-width walk, B = 2) with different
    shared-memory sizes (K = 5 and K = 16), used alternately: the dynamic shared-memory limit is a property of the kernel
    in the process, not of a handle (it must only ever be raised)."""
    ma = L.random_graph(800, 16, 61, complex_hops=True, degree_fill=1.0)
    mb = L.random_graph(900, 5, 62, complex_hops=True, degree_fill=0.9)
    ha = gq.GpuQT(ma, batch=2, modes=gq.MODE_PSI, options={"small": 0})
    hb = gq.GpuQT(mb, batch=2, modes=gq.MODE_PSI, options={"small": 0})
    oa, ob = oracle_mod.Oracle(ma, batch=2, modes=0), oracle_mod.Oracle(mb, batch=2, modes=0)
    pa, pb = L.random_phase_vectors(ma.N, 2, 161, 0), L.random_phase_vectors(mb.N, 2, 162, 0)
    for h, o, p in ((ha, oa, pa), (hb, ob, pb)):
        h.set_state(p)
        o.set_state(p)
    for _ in range(2):
        for h, o, m in ((hb, ob, mb), (ha, oa, ma), (hb, ob, mb)):
            assert np.max(np.abs(h.dos_moments(24) - o.dos_moments(24))) / m.N <= TOL
            h.evolve(0.4, 12)
            o.evolve(0.4, 12)
            assert vec_err(h.get_state(gq.STATE_PSI), o.get_state(oracle_mod.PSI)) <= TOL
    for x in (ha, hb, oa, ob):
        x.close()
