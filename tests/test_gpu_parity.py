"""GPU parity: the CUDA path (through the C-ABI) against the CPU oracle, element by element on the
same seeded inputs.  Sizes span several 256-thread tiles, several 32-row slices and a ragged tail.

Tolerances, written here:
  tables / indices / dx : bit-exact
  moments               : max_n |C_gpu - C_cpu| / (||phi_L|| ||phi_R||) <= 1e-10
  vectors               : max_i |d psi_i| / max_i |psi_i|             <= 1e-10
  transform             : max |d| / max |out|                          <= 1e-10
"""
import numpy as np
import pytest

from workloads import lattices as L

pytestmark = pytest.mark.gpu

TOL = 1e-10


PATHS = {
    # one plain launch per recurrence step
    "streaming": {"small": 0, "persistent": 0},
    # the one-CTA whole-recurrence kernel wherever matrix + vectors fit one SM's shared memory
    "small_path": {"small": 1, "persistent": 0},
    # whole recurrences as ONE cooperative launch of the streaming kernel, grid barriers between the steps
    "persistent": {"small": 0, "persistent": 1},
}


@pytest.fixture(autouse=True, params=list(PATHS))
def launch_path(request, monkeypatch):
    """Every case runs on each of the three launch forms of the recurrences (gpuqt_options)."""
    from paper_1705_01387_b200 import binding
    monkeypatch.setattr(binding, "DEFAULT_OPTIONS", dict(PATHS[request.param]))
    return request.param


def opts(**kw):
    """The launch path of this test run plus explicit option overrides."""
    from paper_1705_01387_b200 import binding
    return {**binding.DEFAULT_OPTIONS, **kw}


@pytest.fixture(scope="module")
def gq():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1705_01387_b200 as g
    return g


def vec_err(a, b):
    return np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300)


def norms(v):
    """[B][N][2] -> per-vector 2-norm"""
    return np.sqrt(np.sum(v * v, axis=(1, 2)))


def small_models():
    return [
        ("square_k4", L.square(70, 37, W=2.0, seed=3)),                         # N = 2590, KT = 4 path
        ("cubic_k6", L.cubic(13, W=16.5, seed=4, energy_scale=16.0)),           # N = 2197, KT = 6 path
        ("graphene_k3", L.graphene(29, 17, W=1.0, seed=5)),                     # N = 1972, KT = 3 path
        ("graphene_vac", L.graphene(31, 19, vacancy_fraction=0.03, vacancy_seed=9)),  # ragged rows
        ("square_open", L.square(41, 23, W=1.0, seed=6, periodic=False)),       # generic width path
        ("peierls_cplx", L.square_peierls(45, 31, flux_quanta=3, W=1.5, seed=7)),  # complex hoppings
        ("chain_k2", L.chain(3001, W=1.0, seed=8)),                             # generic K = 2
        # per-entry real hoppings (every model above without Peierls phases has ONE hopping value
        # and is stored in the constant-hopping record variant)
        ("square_bonddis", L.with_bond_disorder(L.square(52, 33, W=1.0, seed=13), 0.5, 21)),
        ("graphene_vac_bonddis", L.with_bond_disorder(L.graphene(23, 17, vacancy_fraction=0.05, vacancy_seed=4), 0.3, 22)),
        ("cubic_bonddis", L.with_bond_disorder(L.cubic(11, W=8.0, seed=14, energy_scale=11.0), 0.2, 23)),
        # N a multiple of 32, no padding, constant hopping: stored with 16-bit columns (kHopConst16)
        ("square_idx16", L.square(64, 32, W=2.0, seed=15)),
        ("cubic_idx16", L.cubic(16, W=16.5, seed=16, energy_scale=16.0)),
        ("graphene_idx16", L.graphene(16, 8, W=1.0, seed=17)),
    ]


@pytest.mark.parametrize("name,model", small_models(), ids=[n for n, _ in small_models()])
def test_table_bit_exact(gq, oracle_mod, name, model):
    o = oracle_mod.Oracle(model)
    g = gq.GpuQT(model, batch=1, modes=0)
    for a, b in zip(g.get_table(), o.get_table()):
        assert a.tobytes() == b.tobytes()
    g.close()


@pytest.mark.parametrize("batch", [1, 2, 4, 8])
@pytest.mark.parametrize("name,model", small_models(), ids=[n for n, _ in small_models()])
def test_dos_moments(gq, oracle_mod, name, model, batch):
    phi = L.random_phase_vectors(model.N, batch, config=50)
    o = oracle_mod.Oracle(model, batch=batch)
    o.set_state(phi)
    g = gq.GpuQT(model, batch=batch, modes=0)
    g.set_state(phi)
    for nm in (64, 33):                                     # even and odd moment counts
        ref = o.dos_moments(nm)
        got = g.dos_moments(nm)
        assert np.max(np.abs(got - ref)) / model.N <= TOL
    assert np.max(np.abs(g.get_state(gq.STATE_PSI) - phi)) == 0.0
    g.close()


@pytest.mark.parametrize("batch", [1, 4])
@pytest.mark.parametrize("name,model", small_models(), ids=[n for n, _ in small_models()])
def test_time_stepping_all_branches(gq, oracle_mod, name, model, batch):
    """psi, chi (fused e-recursion vs the oracle's separate U chi + [X,U] psi), a, b after
    non-uniform steps; VAC = measure-then-evolve, MSD = evolve-then-measure [A4]."""
    phi = L.random_phase_vectors(model.N, batch, config=51)
    modes = gq.MODE_VAC | gq.MODE_MSD
    o = oracle_mod.Oracle(model, batch=batch, modes=modes)
    g = gq.GpuQT(model, batch=batch, modes=modes)
    o.set_state(phi)
    g.set_state(phi)
    nm = 24
    assert vec_err(g.get_state(gq.STATE_VAC_B), o.get_state(oracle_mod.VAC_B)) <= TOL   # V phi
    dE = model.energy_scale
    for dt in (0.4, 1.0, 0.15):
        order = int(dE * dt) + 30
        vac_ref, vac_got = o.vac(nm), g.vac(nm)
        va = o.get_state(oracle_mod.VAC_A)
        vb = o.get_state(oracle_mod.VAC_B)
        scale = np.array([np.linalg.norm(o.apply_v(va[b])) * np.linalg.norm(vb[b]) for b in range(batch)])
        assert np.max(np.abs(vac_got - vac_ref) / scale[:, None]) <= TOL
        o.evolve(dt, order)
        g.evolve(dt, order)
        for which_g, which_o in ((gq.STATE_PSI, oracle_mod.PSI), (gq.STATE_CHI, oracle_mod.CHI),
                                 (gq.STATE_VAC_A, oracle_mod.VAC_A), (gq.STATE_VAC_B, oracle_mod.VAC_B)):
            assert vec_err(g.get_state(which_g), o.get_state(which_o)) <= TOL
        chi = o.get_state(oracle_mod.CHI)
        msd_ref, msd_got = o.msd(nm), g.msd(nm)
        assert np.max(np.abs(msd_got - msd_ref) / (norms(chi) ** 2)[:, None]) <= TOL
    g.close()


def test_negative_dt_and_order_one(gq, oracle_mod):
    model = L.square(33, 21, W=2.0, seed=12)
    phi = L.random_phase_vectors(model.N, 2, config=52)
    o = oracle_mod.Oracle(model, batch=2, modes=oracle_mod.MODE_MSD)
    g = gq.GpuQT(model, batch=2, modes=gq.MODE_MSD)
    o.set_state(phi)
    g.set_state(phi)
    for dt, order in ((-0.7, 40), (0.3, 1), (0.2, 2), (0.9, 3)):
        o.evolve(dt, order)
        g.evolve(dt, order)
        assert vec_err(g.get_state(gq.STATE_PSI), o.get_state(oracle_mod.PSI)) <= TOL
        assert vec_err(g.get_state(gq.STATE_CHI), o.get_state(oracle_mod.CHI)) <= TOL
    g.close()


def test_psi_only_mode(gq, oracle_mod):
    model = L.graphene(20, 11, W=1.0, seed=2)
    phi = L.random_phase_vectors(model.N, 1, config=53)
    o = oracle_mod.Oracle(model, batch=1, modes=0)
    g = gq.GpuQT(model, batch=1, modes=gq.MODE_PSI)
    o.set_state(phi)
    g.set_state(phi)
    o.evolve(1.3, 50)
    g.evolve(1.3, 50)
    assert vec_err(g.get_state(gq.STATE_PSI), o.get_state(oracle_mod.PSI)) <= TOL
    # unitarity: the norm is preserved to rounding
    assert abs(np.linalg.norm(g.get_state(gq.STATE_PSI)) - np.sqrt(model.N)) < 1e-9
    g.close()


def test_transform(gq, oracle_mod):
    model = L.square(40, 30, W=2.0, seed=1)
    phi = L.random_phase_vectors(model.N, 4, config=54)
    o = oracle_mod.Oracle(model, batch=4)
    g = gq.GpuQT(model, batch=4, modes=0)
    o.set_state(phi)
    g.set_state(phi)
    for nm in (1000, 257):
        C = o.dos_moments(nm)
        E = np.linspace(-0.98 * model.energy_scale, 0.98 * model.energy_scale, 601)
        ref = o.kpm_transform(C, E)
        got = g.kpm_transform(C, E)
        assert np.max(np.abs(got - ref)) / np.max(np.abs(ref)) <= TOL
    with pytest.raises(gq.GpuqtError) as ei:
        g.kpm_transform(C, np.array([model.energy_scale]))
    assert ei.value.status == -5
    # the other damping kernels: Lorentz(lambda), none; Jackson through the same entry point
    for kind, lam in ((gq.DAMPING_JACKSON, 0.0), (gq.DAMPING_LORENTZ, 4.0), (gq.DAMPING_LORENTZ, 0.7), (gq.DAMPING_NONE, 0.0)):
        ref = o.kpm_transform(C, E, damping=kind, lam=lam)
        got = g.kpm_transform(C, E, damping=kind, lam=lam)
        assert np.max(np.abs(got - ref)) / np.max(np.abs(ref)) <= TOL
    assert np.array_equal(g.kpm_transform(C, E, damping=gq.DAMPING_JACKSON), g.kpm_transform(C, E))
    for kind, lam in ((gq.DAMPING_LORENTZ, 0.0), (gq.DAMPING_LORENTZ, -1.0), (7, 1.0)):
        with pytest.raises(gq.GpuqtError) as ei:
            g.kpm_transform(C, E, damping=kind, lam=lam)
        assert ei.value.status == -1
    g.close()


def test_prefetched_state_equals_set_state(gq):
    """gpuqt_prefetch_state + gpuqt_set_state_prefetched (upload on the library's copy stream, overlapping compute)
    leave exactly the state gpuqt_set_state does -- also when a prefetch is issued while the previous batch computes."""
    import torch
    model = L.cubic(13, W=16.5, seed=4, energy_scale=16.0)
    a = gq.GpuQT(model, batch=4, modes=gq.MODE_VAC | gq.MODE_MSD, options=opts())
    b = gq.GpuQT(model, batch=4, modes=gq.MODE_VAC | gq.MODE_MSD, options=opts())
    with pytest.raises(gq.GpuqtError):
        b.set_state_prefetched()                         # nothing pending
    batches = [torch.from_numpy(L.random_phase_vectors(model.N, 4, 91, 4 * i)).pin_memory() for i in range(3)]
    b.prefetch_state(batches[0])
    for i, phi in enumerate(batches):
        a.set_state(phi)
        b.set_state_prefetched()
        if i + 1 < len(batches):
            b.prefetch_state(batches[i + 1])             # overlaps the work below
        for g in (a, b):
            g.evolve(0.7, 20)
        assert a.msd(32).tobytes() == b.msd(32).tobytes()
        assert a.vac(32).tobytes() == b.vac(32).tobytes()
        for which in (gq.STATE_PSI, gq.STATE_CHI, gq.STATE_VAC_A, gq.STATE_VAC_B):
            assert a.get_state(which).tobytes() == b.get_state(which).tobytes()
    with pytest.raises(gq.GpuqtError):
        b.set_state_prefetched()                         # consumed
    a.close()
    b.close()


def test_errors_and_call_order(gq):
    model = L.square(10, 10, W=1.0, seed=1)
    g = gq.GpuQT(model, batch=1, modes=gq.MODE_MSD)
    with pytest.raises(gq.GpuqtError) as ei:
        g.dos_moments(16)                                   # before set_state
    assert ei.value.status == -6
    g.set_state(L.random_phase_vectors(model.N, 1, config=55))
    with pytest.raises(gq.GpuqtError) as ei:
        g.vac(16)                                           # VAC mode not enabled
    assert ei.value.status == -6
    with pytest.raises(gq.GpuqtError) as ei:
        g.msd(1)
    assert ei.value.status == -1
    with pytest.raises(gq.GpuqtError):
        gq.GpuQT(model, batch=3)                            # unsupported batch
    g.close()


def test_run_to_run_determinism(gq):
    """Fixed-order reductions: two runs give bit-identical moments."""
    model = L.cubic(24, W=16.5, seed=4, energy_scale=16.0)
    phi = L.random_phase_vectors(model.N, 4, config=56)
    outs = []
    for _ in range(2):
        g = gq.GpuQT(model, batch=4, modes=gq.MODE_MSD)
        g.set_state(phi)
        g.evolve(1.0, 44)
        outs.append((g.dos_moments(100).copy(), g.msd(100).copy()))
        g.close()
    assert outs[0][0].tobytes() == outs[1][0].tobytes()
    assert outs[0][1].tobytes() == outs[1][1].tobytes()


def test_empty_rows_and_tiny_sizes(gq, oracle_mod):
    """Degenerate inputs: N smaller than one slice, sites with no neighbours at all."""
    for model in (L.chain(5, W=0.5, seed=1), L.square(3, 3, periodic=False),
                  L.graphene(4, 3, vacancy_fraction=0.3, vacancy_seed=2)):
        phi = L.random_phase_vectors(model.N, 2, config=57)
        o = oracle_mod.Oracle(model, batch=2)
        g = gq.GpuQT(model, batch=2)
        o.set_state(phi)
        g.set_state(phi)
        o.evolve(0.5, 30)
        g.evolve(0.5, 30)
        assert vec_err(g.get_state(gq.STATE_CHI), o.get_state(oracle_mod.CHI)) <= TOL
        assert np.max(np.abs(g.dos_moments(10) - o.dos_moments(10))) / model.N <= TOL
        g.close()


@pytest.mark.parametrize("key", ["c1", "c2", "c3", "c4", "c5"])
def test_config_families_small(gq, oracle_mod, key):
    """The five BASELINE.json families at sizes the oracle finishes in seconds, with each config's
    own batch, path, dt and N_p: every time step's moments (all N_m' = 96) and final vectors."""
    from paper_1705_01387_b200 import binding
    from workloads import configs
    w = configs.WORKLOADS[key]
    model = configs.small_variant(key)
    order = w.order or binding.choose_order(model.energy_scale, w.dt)
    nm, steps, B = 96, 3, w.batch
    phi = w.phases(model)
    mg = gq.MODE_MSD if w.path == "msd" else gq.MODE_VAC
    mo = oracle_mod.MODE_MSD if w.path == "msd" else oracle_mod.MODE_VAC
    g, o = gq.GpuQT(model, batch=B, modes=mg), oracle_mod.Oracle(model, batch=B, modes=mo)
    for a, b in zip(g.get_table(), o.get_table()):
        assert a.tobytes() == b.tobytes()
    g.set_state(phi)
    o.set_state(phi)
    assert np.max(np.abs(g.dos_moments(nm) - o.dos_moments(nm))) / model.N <= TOL
    for _ in range(steps):
        if w.path == "vac":
            va, vb = o.get_state(oracle_mod.VAC_A), o.get_state(oracle_mod.VAC_B)
            scale = np.array([np.linalg.norm(o.apply_v(va[b])) * np.linalg.norm(vb[b]) for b in range(B)])
            assert np.max(np.abs(g.vac(nm) - o.vac(nm)) / scale[:, None]) <= TOL
            g.evolve(w.dt, order)
            o.evolve(w.dt, order)
        else:
            g.evolve(w.dt, order)
            o.evolve(w.dt, order)
            chi = o.get_state(oracle_mod.CHI)
            assert np.max(np.abs(g.msd(nm) - o.msd(nm)) / (norms(chi) ** 2)[:, None]) <= TOL
    pairs = (((gq.STATE_PSI, oracle_mod.PSI), (gq.STATE_CHI, oracle_mod.CHI)) if w.path == "msd" else
             ((gq.STATE_VAC_A, oracle_mod.VAC_A), (gq.STATE_VAC_B, oracle_mod.VAC_B)))
    for sg, so in pairs:
        assert vec_err(g.get_state(sg), o.get_state(so)) <= TOL
    # energy transform of this run's moments on the paper's 601-point grid (a8)
    C = o.dos_moments(nm)
    E = np.linspace(-0.98 * model.energy_scale, 0.98 * model.energy_scale, 601)
    ref = o.kpm_transform(C, E)
    assert np.max(np.abs(g.kpm_transform(C, E) - ref)) / np.max(np.abs(ref)) <= TOL
    g.close()


def test_deep_recurrences(gq, oracle_mod):
    """Moment sets as deep as the benchmarked configs run them (N_m = 3000 / 2000 / 1000; dots[] indexed
    deep into its buffer, late-moment drift) on the streaming kernels, all moments against the oracle:
    c2's family (VAC, B = 1), c3's (MSD, B = 1, ragged rows), c4's (MSD, B = 4)."""
    from workloads import configs
    for key, nm in (("c2", 3000), ("c3", 2000), ("c4", 1000)):
        w = configs.WORKLOADS[key]
        model = configs.small_variant(key)
        B = w.batch
        phi = w.phases(model)
        mg = gq.MODE_MSD if w.path == "msd" else gq.MODE_VAC
        mo = oracle_mod.MODE_MSD if w.path == "msd" else oracle_mod.MODE_VAC
        g, o = gq.GpuQT(model, batch=B, modes=mg, options=opts(small=0)), oracle_mod.Oracle(model, batch=B, modes=mo)
        g.set_state(phi)
        o.set_state(phi)
        assert np.max(np.abs(g.dos_moments(nm) - o.dos_moments(nm))) / model.N <= TOL
        g.evolve(w.dt, w.order)
        o.evolve(w.dt, w.order)
        if w.path == "vac":
            va, vb = o.get_state(oracle_mod.VAC_A), o.get_state(oracle_mod.VAC_B)
            scale = np.array([np.linalg.norm(o.apply_v(va[b])) * np.linalg.norm(vb[b]) for b in range(B)])
            assert np.max(np.abs(g.vac(nm) - o.vac(nm)) / scale[:, None]) <= TOL
        else:
            chi = o.get_state(oracle_mod.CHI)
            assert np.max(np.abs(g.msd(nm) - o.msd(nm)) / (norms(chi) ** 2)[:, None]) <= TOL
        g.close()
        o.close()


def test_constant_hopping_variant_matches_per_entry(gq, oracle_mod):
    """The constant-hopping record variant (no hop array, padding col = N, the zero row) and the
    per-entry variant (option hop_const = 0) of the same model decode to the same table and give
    moments and vectors within rounding of the oracle."""
    from paper_1705_01387_b200 import binding
    model = L.graphene(31, 19, W=0.5, seed=3, vacancy_fraction=0.2, vacancy_seed=9)   # many padded rows
    phi = L.random_phase_vectors(model.N, 4, config=58)
    o = oracle_mod.Oracle(model, batch=4, modes=oracle_mod.MODE_MSD | oracle_mod.MODE_VAC)
    o.set_state(phi)
    ref_tab = o.get_table()
    ref_dos, ref_vac = o.dos_moments(40), o.vac(40)
    o.evolve(0.8, 45)
    ref_chi = o.get_state(oracle_mod.CHI)
    for flag in (1, 0):
        g = gq.GpuQT(model, batch=4, modes=gq.MODE_MSD | gq.MODE_VAC, options=opts(hop_const=flag))
        assert g.info(binding.INFO_HOP_VARIANT) == (3 if flag else 0)      # constant hopping, 16-bit columns (zero row in reach) / per entry
        for a, b in zip(g.get_table(), ref_tab):
            assert a.tobytes() == b.tobytes()
        g.set_state(phi)
        assert np.max(np.abs(g.dos_moments(40) - ref_dos)) / model.N <= TOL
        assert np.max(np.abs(g.vac(40) - ref_vac)) / np.max(np.abs(ref_vac[:, 0])) <= TOL
        g.evolve(0.8, 45)
        assert vec_err(g.get_state(gq.STATE_CHI), ref_chi) <= TOL
        g.close()


@pytest.mark.parametrize("o", [{"persistent": 0}, {"persistent": 1, "run": 8}, {"persistent": 1, "blocks_per_sm": 1, "stages": 4},
                               {"persistent": 1, "alternate": 0, "run": 32, "stages": 1}],
                         ids=["single_step", "multi_run8", "multi_1cta_4stages", "multi_noalt_run32_1stage"])
def test_multi_step_launches(gq, oracle_mod, o):
    """Whole recurrences in one cooperative launch (grid barrier between the steps, the stage ring and
    the dot partials running on across them) against one launch per step and the oracle, on lattices
    large enough for many runs per CTA: every mode, odd and even term counts, periodic wrap-around."""
    from paper_1705_01387_b200 import binding
    for model, B in ((L.cubic(40, W=16.5, seed=4, energy_scale=16.0), 4),                    # 64000 rows, K = 6
                     (L.graphene(150, 101, vacancy_fraction=0.02, vacancy_seed=9), 1),       # ragged, B = 1
                     (L.square(300, 230, W=1.0, seed=6, periodic=False), 1),                 # open edges: padding entries out of 16-bit reach
                     (L.square(300, 211, W=2.0, seed=3), 1),                                 # two-slice tiles, odd tail
                     (L.chain(50001, W=1.0, seed=8), 2),                                     # K = 2, B = 2
                     (L.square_peierls(240, 130, flux_quanta=5, W=1.5, seed=7), 8)):         # complex, B = 8
        phi = L.random_phase_vectors(model.N, B, config=59)
        modes = gq.MODE_VAC | gq.MODE_MSD
        o_ = oracle_mod.Oracle(model, batch=B, modes=modes)
        stencil = 2 if model.name.startswith("cubic") else 1     # the implicit stencil on multi-step launches too
        g = gq.GpuQT(model, batch=B, modes=modes, options={"small": 0, "stencil": stencil, **o})
        assert g.info(binding.INFO_PERSISTENT) == o["persistent"]
        if model.name.startswith("square") and model.box_length <= 0:
            assert g.info(binding.INFO_HOP_VARIANT) == 4      # 16-bit columns with the 0xffff sentinel for the zero row
        if model.name.startswith("cubic"):
            assert g.info(binding.INFO_HOP_VARIANT) == 5 and g.info(binding.INFO_STENCIL_PATTERNS) == 27
        o_.set_state(phi)
        g.set_state(phi)
        for nm in (37, 64):
            assert np.max(np.abs(g.dos_moments(nm) - o_.dos_moments(nm))) / model.N <= TOL
        for dt, order in ((0.7, 24), (0.35, 17)):
            va, vb = o_.get_state(oracle_mod.VAC_A), o_.get_state(oracle_mod.VAC_B)
            scale = np.array([np.linalg.norm(o_.apply_v(va[b])) * np.linalg.norm(vb[b]) for b in range(B)])
            assert np.max(np.abs(g.vac(33) - o_.vac(33)) / scale[:, None]) <= TOL
            o_.evolve(dt, order)
            g.evolve(dt, order)
            for sg, so in ((gq.STATE_PSI, oracle_mod.PSI), (gq.STATE_CHI, oracle_mod.CHI),
                           (gq.STATE_VAC_A, oracle_mod.VAC_A), (gq.STATE_VAC_B, oracle_mod.VAC_B)):
                assert vec_err(g.get_state(sg), o_.get_state(so)) <= TOL
            chi = o_.get_state(oracle_mod.CHI)
            assert np.max(np.abs(g.msd(30) - o_.msd(30)) / (norms(chi) ** 2)[:, None]) <= TOL
        g.close()
        o_.close()


def test_launch_counts(gq):
    """The multi-step forms really are one launch per recurrence (gpuqt_kernel_stats)."""
    from paper_1705_01387_b200 import binding
    model = L.square(48, 40, W=2.0, seed=2)                  # 1920 orbitals: fits one SM's shared memory
    phi = L.random_phase_vectors(model.N, 1, config=61)
    for o, per_rec in (({"small": 0, "persistent": 1}, 1), ({"small": 1, "persistent": 0}, 1), ({"small": 0, "persistent": 0}, None)):
        g = gq.GpuQT(model, batch=1, modes=gq.MODE_VAC, options=o)
        g.set_state(phi)
        g.reset_stats()
        g.dos_moments(100)
        g.vac(64)
        g.evolve(0.5, 20)
        ms, n = g.kernel_stats(binding.KERNEL_KPM_DOUBLING)
        assert n == (per_rec or 50) and g.kernel_steps(binding.KERNEL_KPM_DOUBLING) == 50
        ms, n = g.kernel_stats(binding.KERNEL_KPM_LEFT)
        assert n == (per_rec or 63) and g.kernel_steps(binding.KERNEL_KPM_LEFT) == 63
        ms, n = g.kernel_stats(binding.KERNEL_EVOLVE)          # two branches; + the scale launch each on the streaming forms
        assert n == (2 if o["small"] else 4 if per_rec else 2 * 20) and g.kernel_steps(binding.KERNEL_EVOLVE) == 2 * 19
        g.close()
        # the (psi, chi) time step (SURVEY 7 hard part 5): one launch on the one-CTA path too
        g = gq.GpuQT(model, batch=1, modes=gq.MODE_MSD, options=o)
        assert g.info(binding.INFO_SMALL_PATH_MSD) == o["small"]
        g.set_state(phi)
        g.reset_stats()
        for _ in range(3):
            g.evolve(0.5, 20)
        ms, n = g.kernel_stats(binding.KERNEL_EVOLVE_MSD)      # + two scale launches per step on the streaming forms
        assert n == 3 * (1 if o["small"] else 3 if per_rec else 2 + 19) and g.kernel_steps(binding.KERNEL_EVOLVE_MSD) == 3 * 19
        g.close()


@pytest.mark.parametrize("model", [L.cubic(16, W=16.5, seed=16, energy_scale=16.0),
                                   L.graphene(40, 24, vacancy_fraction=0.04, vacancy_seed=5)],     # padding entries: delta 0xffff
                         ids=["cubic", "graphene_vacancies"])
def test_16bit_columns_match_32bit(gq, oracle_mod, model):
    """The same table stored with 16-bit (base + delta) and with 32-bit columns decodes to the same
    canonical table and gives the same moments / vectors."""
    from paper_1705_01387_b200 import binding
    phi = L.random_phase_vectors(model.N, 4, config=60)
    o = oracle_mod.Oracle(model, batch=4, modes=oracle_mod.MODE_MSD | oracle_mod.MODE_VAC)
    o.set_state(phi)
    ref_tab, ref_dos, ref_vac = o.get_table(), o.dos_moments(48), o.vac(48)
    o.evolve(1.0, 44)
    ref_chi = o.get_state(oracle_mod.CHI)
    outs = []
    for flag in (1, 0):
        g = gq.GpuQT(model, batch=4, modes=gq.MODE_MSD | gq.MODE_VAC, options=opts(idx16=flag, stencil=0))
        assert g.info(binding.INFO_HOP_VARIANT) == (3 if flag else 2)
        for a, b in zip(g.get_table(), ref_tab):
            assert a.tobytes() == b.tobytes()
        g.set_state(phi)
        dos = g.dos_moments(48)
        assert np.max(np.abs(dos - ref_dos)) / model.N <= TOL
        assert np.max(np.abs(g.vac(48) - ref_vac)) / np.max(np.abs(ref_vac[:, 0])) <= TOL
        g.evolve(1.0, 44)
        assert vec_err(g.get_state(gq.STATE_CHI), ref_chi) <= TOL
        outs.append(dos.copy())
        g.close()
    assert outs[0].tobytes() == outs[1].tobytes()        # same arithmetic, only the column encoding differs


@pytest.mark.parametrize("batch", [1, 2, 4, 8])
@pytest.mark.parametrize("model", [L.cubic(16, W=16.5, seed=16, energy_scale=16.0),      # lines aligned with the slices
                                   L.cubic(13, W=8.0, seed=4, energy_scale=11.0),        # nothing aligned, ragged tail
                                   L.square(70, 37, W=2.0, seed=3),
                                   L.graphene(29, 17, W=1.0, seed=5),                    # 4-atom cell: period 4 in the row index
                                   L.chain(3001, W=1.0, seed=8)],
                         ids=["cubic16", "cubic13", "square70x37", "graphene29x17", "chain3001"])
def test_implicit_stencil_matches_explicit_columns(gq, oracle_mod, model, batch):
    """the same regular lattice stored as an implicit stencil (on-site
    records + pattern dictionary, option stencil = 2: forced) and with an explicit column array decodes to
    the same canonical table, bit for bit the oracle's, and gives the same moments / vectors -- identical
    bits, since only the column encoding differs."""
    from paper_1705_01387_b200 import binding
    phi = L.random_phase_vectors(model.N, batch, config=62)
    modes = gq.MODE_MSD | gq.MODE_VAC
    o = oracle_mod.Oracle(model, batch=batch, modes=modes)
    o.set_state(phi)
    ref_tab, ref_dos, ref_vac = o.get_table(), o.dos_moments(48), o.vac(31)
    va, vb = o.get_state(oracle_mod.VAC_A), o.get_state(oracle_mod.VAC_B)
    scale = np.array([np.linalg.norm(o.apply_v(va[b])) * np.linalg.norm(vb[b]) for b in range(batch)])
    o.evolve(1.0, 44)
    ref_chi, ref_a = o.get_state(oracle_mod.CHI), o.get_state(oracle_mod.VAC_A)
    ref_msd = o.msd(20)
    outs = []
    for flag in (2, 0):
        g = gq.GpuQT(model, batch=batch, modes=modes, options=opts(stencil=flag, idx16=0))
        assert g.info(binding.INFO_HOP_VARIANT) == (5 if flag else 2)
        assert (g.info(binding.INFO_STENCIL_PATTERNS) > 0) == bool(flag)
        for a, b in zip(g.get_table(), ref_tab):
            assert a.tobytes() == b.tobytes()
        g.set_state(phi)
        dos, vac = g.dos_moments(48), g.vac(31)
        assert np.max(np.abs(dos - ref_dos)) / model.N <= TOL
        assert np.max(np.abs(vac - ref_vac) / scale[:, None]) <= TOL
        g.evolve(1.0, 44)
        chi = g.get_state(gq.STATE_CHI)
        assert vec_err(chi, ref_chi) <= TOL and vec_err(g.get_state(gq.STATE_VAC_A), ref_a) <= TOL
        msd = g.msd(20)
        assert np.max(np.abs(msd - ref_msd) / (norms(ref_chi) ** 2)[:, None]) <= TOL
        outs.append((dos.copy(), vac.copy(), chi.copy(), msd.copy()))
        g.close()
    for a, b in zip(*outs):
        assert a.tobytes() == b.tobytes()


@pytest.mark.parametrize("batch", [1, 4, 8])
def test_brick_reordering_is_invisible(gq, oracle_mod, batch):
    """gpuqt_options.reorder: a recognised simple-cubic lattice is stored in bricks of 4 x 4 x 2 sites.  Forced on a
    small lattice (neighbour lists in shuffled order per row): the decoded table is bit-identical to the oracle's in the
    caller's numbering, states and moments agree with the oracle, and with the unreordered handle to rounding."""
    from paper_1705_01387_b200 import binding
    model = L.cubic(16, W=16.5, seed=16, energy_scale=16.0)            # 16 x 16 x 16: Lx, Ly multiples of 4, Lz even
    # shuffle the neighbour order inside every row (the detection must not depend on it)
    idx = model.nbr_index.reshape(model.N, 6).copy()
    perm = np.argsort(L.rng.uniform01(77, model.N * 6).reshape(model.N, 6), axis=1)
    model.nbr_index = np.ascontiguousarray(np.take_along_axis(idx, perm, axis=1).reshape(-1))
    a = gq.GpuQT(model, batch=batch, modes=gq.MODE_VAC | gq.MODE_MSD, options=opts(reorder=2, small=0))
    b = gq.GpuQT(model, batch=batch, modes=gq.MODE_VAC | gq.MODE_MSD, options=opts(reorder=0, small=0))
    assert a.info(binding.INFO_REORDERED) == 1 and b.info(binding.INFO_REORDERED) == 0
    o = oracle_mod.Oracle(model, batch=batch, modes=oracle_mod.MODE_VAC | oracle_mod.MODE_MSD)
    oc, ore, oim, odx = o.get_table()
    for g in (a, b):
        col, re, im, dx = g.get_table()
        assert np.array_equal(col, oc) and re.tobytes() == ore.tobytes() and dx.tobytes() == odx.tobytes()
    phi = L.random_phase_vectors(model.N, batch, 97, 0)
    for g in (a, b, o):
        g.set_state(phi)
    nm = 48
    ref = o.dos_moments(nm)
    assert np.max(np.abs(a.dos_moments(nm) - ref)) / model.N <= TOL
    for g in (a, b, o):
        g.evolve(0.9, 30)
    chi = o.get_state(oracle_mod.CHI)
    for which, ow in ((gq.STATE_PSI, oracle_mod.PSI), (gq.STATE_CHI, oracle_mod.CHI), (gq.STATE_VAC_A, oracle_mod.VAC_A),
                      (gq.STATE_VAC_B, oracle_mod.VAC_B)):
        assert vec_err(a.get_state(which), o.get_state(ow)) <= TOL
        assert a.get_state(which).tobytes() == b.get_state(which).tobytes()     # same operands, same neighbour order per row
    assert np.max(np.abs(a.msd(nm) - o.msd(nm)) / np.sum(chi * chi, axis=(1, 2))[:, None]) <= TOL
    va, vb = o.get_state(oracle_mod.VAC_A), o.get_state(oracle_mod.VAC_B)
    scale = np.array([np.linalg.norm(o.apply_v(va[k])) * np.linalg.norm(vb[k]) for k in range(batch)])
    assert np.max(np.abs(a.vac(nm) - o.vac(nm)) / scale[:, None]) <= TOL
    # not a cubic lattice / dimensions the bricks do not divide: left alone
    for other in (L.cubic(13, W=1.0, seed=4, energy_scale=8.0), L.square(64, 32, W=2.0, seed=15)):
        g = gq.GpuQT(other, batch=batch, modes=gq.MODE_PSI, options=opts(reorder=2))
        assert g.info(binding.INFO_REORDERED) == 0
        g.close()
    for g in (a, b, o):
        g.close()


@pytest.mark.parametrize("size", [4, 8, 12, 20])
def test_brick_reordering_small_and_odd_brick_counts(gq, oracle_mod, size):
    """Cubes whose brick grid is 1 x 1 x 2 (4^3), 2 x 2 x 4, 3 x 3 x 6 and 5 x 5 x 10: every wrap falls on a brick boundary,
    one brick can be its own neighbour in x and y."""
    from paper_1705_01387_b200 import binding
    model = L.cubic(size, W=16.5, seed=size, energy_scale=16.0)
    g = gq.GpuQT(model, batch=4, modes=gq.MODE_MSD, options=opts(reorder=2, small=0))
    assert g.info(binding.INFO_REORDERED) == 1
    o = oracle_mod.Oracle(model, batch=4, modes=oracle_mod.MODE_MSD)
    col, re, im, dx = g.get_table()
    oc, ore, oim, odx = o.get_table()
    assert np.array_equal(col, oc) and re.tobytes() == ore.tobytes() and dx.tobytes() == odx.tobytes()
    phi = L.random_phase_vectors(model.N, 4, 98, 0)
    g.set_state(phi)
    o.set_state(phi)
    g.evolve(1.0, 44)
    o.evolve(1.0, 44)
    chi = o.get_state(oracle_mod.CHI)
    assert vec_err(g.get_state(gq.STATE_CHI), chi) <= TOL
    assert np.max(np.abs(g.msd(64) - o.msd(64)) / np.sum(chi * chi, axis=(1, 2))[:, None]) <= TOL
    g.close()
    o.close()
