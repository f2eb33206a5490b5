"""GPU parity of the post-processing step and of the paper's whole simulation loop:
gpuqt_running_conductivity against the oracle, and transport.run on the CUDA library against the
test-side loop of tests/ref_loop.py driven through the oracle (no shared code: the row convention
[A4], the averaging and the N_p rule [A5] are restated there), on reduced-size versions of the
paper's two examples.  Tolerance: max |d| / max |ref| <= 1e-10 per output array
(A22)."""
import numpy as np
import pytest

from tests import ref_loop
from workloads import configs

pytestmark = pytest.mark.gpu

TOL = 1e-10


@pytest.fixture(scope="module")
def gq():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1705_01387_b200 as g
    return g


def rel(a, b):
    return np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300)


def test_running_conductivity_parity(gq, oracle_mod):
    from workloads import lattices as L
    rng_ = np.random.default_rng(3)
    g = gq.GpuQT(L.square(8, 8), batch=1, modes=0)
    for n_t, n_e in ((1, 1), (7, 5), (30, 601), (20, 1000)):
        corr = rng_.standard_normal((n_t, n_e)) ** 2
        dos = rng_.random(n_e) + 0.1
        dos[0] = 0.0                                                   # degenerate: no states at this energy
        dt = rng_.random(n_t) + 0.05
        for kind in ("vac", "msd"):
            s_ref, l_ref = oracle_mod.running_conductivity(kind, corr, dos, dt)
            s_got, l_got = g.running_conductivity(kind, corr, dos, dt)
            assert rel(s_got, s_ref) <= 1e-14 or np.max(np.abs(s_ref)) == 0
            if kind == "msd":
                assert rel(l_got, l_ref) <= 1e-14
                assert np.all(l_got[:, 0] == 0.0)
                # Eq. 12 on top of it: xi at the last time and the saturation check, element by element
                xi_ref, gr_ref = oracle_mod.localization_length(l_ref)
                xi_got, gr_got = g.localization_length(l_ref)
                assert np.array_equal(xi_got, xi_ref) and np.allclose(gr_got, gr_ref, rtol=1e-14, atol=0)
                assert xi_got[0] == 0.0 and gr_got[0] == 0.0
    with pytest.raises(gq.GpuqtError):
        g.running_conductivity("msd", np.ones((2, 2)), None, np.array([0.1, -0.1]))
    g.close()


@pytest.mark.parametrize("key,scale", [("e1", 0.04), ("e2", 0.0005)])
def test_paper_examples_reduced(gq, oracle_mod, key, scale):
    from paper_1705_01387_b200 import binding, transport
    ex = configs.EXAMPLES[key]
    model = ex.build(scale)                                             # e1: 80 x 80, e2: chain of 2000
    dts = ex.dts[:8] if key == "e1" else ex.dts[:14]                   # oracle cost control
    nm = 200
    phi = ex.phases(model)
    mg = (gq.MODE_VAC if ex.vac else 0) | (gq.MODE_MSD if ex.msd else 0)
    order_of = lambda dt: binding.choose_order(model.energy_scale, dt)
    for dt in set(dts):                                                 # the product's N_p rule against the oracle-side one
        assert order_of(dt) == ref_loop.order_rule(oracle_mod, model.energy_scale, dt)
    g = gq.GpuQT(model, batch=ex.batch, modes=mg)
    got = transport.run(g, phi, dts, nm, ex.energies(), order_of, vac=ex.vac, msd=ex.msd)
    ref = ref_loop.simulation_loop(oracle_mod, model, phi, dts, nm, ex.energies(), ex.vac, ex.msd)
    for name in ("dos", "rho_vac", "sigma_vac", "rho_msd", "sigma_msd"):
        if name in ref:
            assert rel(got[name], ref[name]) <= TOL, name
    if "length" in ref:
        # L = 2 sqrt(rho dX^2 / rho) is a ratio: where the DOS vanishes (band tails, |E| -> dE) it divides two
        # rounding-level numbers, so it is compared where it is conditioned, rho > 1e-3 max rho
        ok = ref["dos"] > 1e-3 * np.max(ref["dos"])
        assert rel(got["length"][:, ok], ref["length"][:, ok]) <= TOL
        assert rel(got["xi"][ok], ref["xi"][ok]) <= TOL                     # Eq. 12 at the last time [A27]
        assert np.max(np.abs(got["xi_growth"][ok] - ref["xi_growth"][ok])) <= 1e-8      # a difference of two lengths / L
    # what the paper says about its figures, on quantities that are exact for any size:
    E = ex.energies()
    assert abs(np.trapezoid(got["dos"], E) - 2.0) < 0.02                    # int rho dE = 2 per site (spin factor, Eq. 4)
    if ex.msd:
        j0 = int(np.argmin(np.abs(E)))
        x2 = got["rho_msd"][:, j0] / got["dos"][j0]
        t = transport.time_axis(dts)[1:]
        assert np.all(np.diff(x2[:4]) > 0)                              # the MSD grows from zero ...
        assert abs(x2[0] / t[0] ** 2 / (x2[1] / t[1] ** 2) - 1.0) < 0.2  # ... quadratically at short times (ballistic)
    g.close()


def test_file_front_end_matches_oracle(gq, oracle_mod, tmp_path):
    """The paper's workflow: a simulation folder run through the CUDA library writes
    the dos.out / vac.out / msd.out rows the oracle gives for the same model and vectors, each vector
    run alone through tests/ref_loop.py (no product code on the expected side)."""
    from paper_1705_01387_b200 import frontend as F
    from workloads import lattices as L
    model = L.square(40, 32, W=4.0, seed=3, energy_scale=6.1)
    E = np.linspace(-6.0, 6.0, 121)
    dts = [0.2, 0.2, 0.5, 1.0]
    para = {"calculate_vac": True, "calculate_msd": True, "number_of_random_vectors": 3, "number_of_moments": 128}
    F.write_folder(str(tmp_path / "gpu"), model, E, dts, para)
    F.run_folder(str(tmp_path / "gpu"), seed=11)
    phi = F.random_phase_vectors(model.N, 3, 11)                      # the front-end's input generator (no method arithmetic)
    dos, vac, msd = ref_loop.per_vector_rows(oracle_mod, model, phi, dts, 128, E, True, True)
    for out, ref in (("dos.out", dos), ("vac.out", vac.reshape(12, 121)), ("msd.out", msd.reshape(12, 121))):
        a = np.loadtxt(tmp_path / "gpu" / out)
        assert a.shape == ref.shape
        assert rel(a, ref) <= TOL, out
