"""Pins of the product's simulation loop (paper_1705_01387_b200/transport.py) that are not the loop itself
(-m "not gpu"): driven by the ORACLE as engine it must give (i) the closed forms of a plane wave on a clean
periodic chain at the times reading [A4] assigns to the rows and (ii) the rows of the
independently written test-side loop tests/ref_loop.py.  A wrong row convention (VAC measured after the
step, MSD before it, a skipped or doubled evolution, averaging over the wrong axis) fails (i)."""
import numpy as np

from tests import ref_loop
from workloads import lattices as L


class OracleEngine:
    """The oracle behind the method names transport.run calls."""

    def __init__(self, oracle_mod, model, batch, modes):
        self.o = oracle_mod.Oracle(model, batch=batch, modes=modes)
        self.mod = oracle_mod

    def __getattr__(self, name):
        return getattr(self.o, name)

    def running_conductivity(self, kind, corr, dos, dt):
        return self.mod.running_conductivity(kind, corr, dos, dt)

    def localization_length(self, length):
        return self.mod.localization_length(length)


def test_rows_are_at_the_times_of_reading_a4(oracle_mod):
    """phi = e^{ikx} on a clean ring: rho C_vv(t) = rho v_k^2 at every t, rho dX^2(t) = rho v_k^2 t^2.  With
    non-uniform steps the MSD rows single out the times t_{k+1} = sum_{i<=k} dt_i, and
    sigma^VAC(t_k) = rho v_k^2 t_k singles out the VAC times t_k = sum_{i<k} dt_i."""
    from paper_1705_01387_b200 import transport
    Lc, kq = 64, 5
    model = L.chain(Lc, energy_scale=2.5)
    k = 2 * np.pi * kq / Lc
    phi = np.stack([np.cos(k * model.x), np.sin(k * model.x)], axis=1)[None]
    dts = [0.5, 0.25, 1.0, 0.75]
    E = np.array([-2.0 * np.cos(k)])                                      # eps_k for hopping -1
    eng = OracleEngine(oracle_mod, model, 1, oracle_mod.MODE_VAC | oracle_mod.MODE_MSD)
    res = transport.run(eng, phi, dts, 64, E, lambda dt: 40, vac=True, msd=True)
    vk2 = (2.0 * np.sin(k)) ** 2
    t = np.concatenate([[0.0], np.cumsum(dts)])
    rho = res["dos"][0]
    assert rho > 0
    assert np.allclose(res["times"], t)
    assert res["rho_vac"].shape == (4, 1) and res["rho_msd"].shape == (4, 1)
    assert np.allclose(res["rho_vac"][:, 0], rho * vk2, rtol=1e-9)                       # time independent
    assert np.allclose(res["rho_msd"][:, 0], rho * vk2 * t[1:] ** 2, rtol=1e-9)          # rows at t_1 .. t_4
    assert np.allclose(res["sigma_vac"][:, 0], rho * vk2 * t[:4], rtol=1e-9)             # rows at t_0 .. t_3
    assert np.allclose(res["sigma_msd"][:, 0], rho * vk2 * 0.5 * (t[1:] + t[:-1]), rtol=1e-9)   # mid-step values
    assert np.allclose(res["length"][:, 0], 2.0 * np.sqrt(vk2) * t[1:], rtol=1e-9)       # Eq. 11
    # the last VAC evolution is skipped when MSD is off, and nothing else changes
    eng2 = OracleEngine(oracle_mod, model, 1, oracle_mod.MODE_VAC)
    calls = []
    real_evolve = eng2.o.evolve
    eng2.evolve = lambda dt, order: (calls.append(dt), real_evolve(dt, order))[1]
    res2 = transport.run(eng2, phi, dts, 64, E, lambda dt: 40, vac=True, msd=False)
    assert calls == dts[:3]
    assert np.allclose(res2["rho_vac"], res["rho_vac"], rtol=1e-12)


def test_transport_run_matches_the_independent_loop(oracle_mod):
    """transport.run against tests/ref_loop.simulation_loop on a disordered lattice, two vectors (averaging),
    VAC + MSD and MSD only; transport's per_vector rows against ref_loop.per_vector_rows."""
    from paper_1705_01387_b200 import transport
    model = L.square(12, 10, W=2.0, seed=5, energy_scale=5.1)
    phi = L.random_phase_vectors(model.N, 2, config=77)
    dts = [0.3, 0.6, 0.2]
    E = np.linspace(-4.5, 4.5, 19)
    order_of = lambda dt: ref_loop.order_rule(oracle_mod, model.energy_scale, dt)
    for vac, msd in ((True, True), (False, True), (True, False)):
        modes = (oracle_mod.MODE_VAC if vac else 0) | (oracle_mod.MODE_MSD if msd else 0)
        got = transport.run(OracleEngine(oracle_mod, model, 2, modes), phi, dts, 48, E, order_of, vac=vac, msd=msd)
        ref = ref_loop.simulation_loop(oracle_mod, model, phi, dts, 48, E, vac, msd)
        assert set(ref) <= set(got)
        for name, r in ref.items():
            assert np.allclose(got[name], r, rtol=1e-12, atol=1e-13 * np.max(np.abs(r))), name
    rows = transport.run(OracleEngine(oracle_mod, model, 2, oracle_mod.MODE_VAC | oracle_mod.MODE_MSD), phi, dts, 48, E,
                         order_of, vac=True, msd=True, per_vector=True)
    dos, rv, rm = ref_loop.per_vector_rows(oracle_mod, model, phi, dts, 48, E, True, True)
    assert np.allclose(rows["dos"], dos, rtol=1e-12, atol=1e-15)
    assert np.allclose(rows["rho_vac"], rv.transpose(1, 0, 2), rtol=1e-12, atol=1e-13 * np.max(np.abs(rv)))
    assert np.allclose(rows["rho_msd"], rm.transpose(1, 0, 2), rtol=1e-12, atol=1e-13 * np.max(np.abs(rm)))


def test_order_rule_matches_the_products(oracle_mod):
    """binding.choose_order (Miller table of the product) and the test-side rule (libm jn) pick the same N_p."""
    from paper_1705_01387_b200 import binding, build
    build.build()
    for dE, dt in ((16.0, 1.0), (10.0, 2.0), (5.1, 2.0), (6.1, 0.2), (4.1, 0.1), (4.1, 100.0), (10.7, 1.0)):
        assert binding.choose_order(dE, dt) == ref_loop.order_rule(oracle_mod, dE, dt)
    assert ref_loop.order_rule(oracle_mod, 16.0, 1.0) == 44 and ref_loop.order_rule(oracle_mod, 10.7, 1.0) == 36
