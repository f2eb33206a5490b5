"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (default
tuning knobs, the config's own batch B, N_m and N_p).

The oracle cannot run a whole config in seconds, so it follows the parity schedule of SURVEY.md
8(d): ONE sampled random vector (the last slot of the batch, so the [N][B] interleave is exercised)
at full N; every evolved state vector of that sample is compared element by element; moments are
compared on the prefix n < P of the GPU's full N_m run (C_n does not depend on N_m [A19]).
Properties that hold at any size cover the other B - 1 vectors: C_0 = <phi|phi> = N, norm
conservation of U, |C_n| <= ||phi_L|| ||phi_R||, run-to-run bit identity.

Tolerances as in test_gpu_parity.py (north_star: 1e-10 in the norms of A22; tables bit-exact).
"""
import numpy as np
import pytest

from workloads import configs

pytestmark = pytest.mark.gpu

TOL = 1e-10
PREFIX = 32


@pytest.fixture(scope="module")
def gq():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1705_01387_b200 as g
    return g


def vec_err(a, b):
    return np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300)


def norm(v):
    return float(np.sqrt(np.sum(v * v)))


@pytest.mark.parametrize("key", ["c1", "c2", "c3", "c4", "c5"])
def test_full_size_config(gq, oracle_mod, key):
    from paper_1705_01387_b200 import binding
    w = configs.WORKLOADS[key]
    model = w.build()
    order = w.order or binding.choose_order(model.energy_scale, w.dt)
    B, nm = w.batch, w.n_moments
    P = nm if key == "c1" else PREFIX                 # c1 is small: the oracle runs all of it
    sb = B - 1                                        # sampled vector
    phi = w.phases(model)
    modes_g = gq.MODE_MSD if w.path == "msd" else gq.MODE_VAC
    modes_o = oracle_mod.MODE_MSD if w.path == "msd" else oracle_mod.MODE_VAC
    g = gq.GpuQT(model, batch=B, modes=modes_g)
    o = oracle_mod.Oracle(model, batch=1, modes=modes_o)

    # a1: the device table decodes to the oracle's padded ELL, bit for bit (col, re, im, dx)
    for a, b in zip(g.get_table(), o.get_table()):
        assert a.tobytes() == b.tobytes()

    g.set_state(phi)
    o.set_state(phi[sb:sb + 1])

    # a6 (DOS), full N_m on the GPU, prefix on the oracle
    dos = g.dos_moments(nm)
    assert dos.shape == (B, nm)
    assert np.max(np.abs(dos[:, 0] - model.N)) <= TOL * model.N            # C_0 = <phi|phi> = N  [A7]
    assert np.max(np.abs(dos)) <= model.N * (1 + 1e-9)                     # |T_n| <= 1 on the spectrum
    assert np.max(np.abs(dos[sb, :P] - o.dos_moments(P)[0])) / model.N <= TOL

    n_rounds = 1 if key == "c5" else 2
    if w.path == "vac":
        for rnd in range(n_rounds + 1):                                   # measure, evolve, measure ... [A4]
            vac = g.vac(nm)
            va, vb = o.get_state(oracle_mod.VAC_A)[0], o.get_state(oracle_mod.VAC_B)[0]
            scale = norm(o.apply_v(va)) * norm(vb)
            assert np.max(np.abs(vac[sb, :P] - o.vac(P)[0])) / scale <= TOL
            if rnd == n_rounds:
                break
            g.evolve(w.dt, order)
            o.evolve(w.dt, order)
            ga, gb = g.get_state(gq.STATE_VAC_A), g.get_state(gq.STATE_VAC_B)
            assert vec_err(ga[sb], o.get_state(oracle_mod.VAC_A)[0]) <= TOL
            assert vec_err(gb[sb], o.get_state(oracle_mod.VAC_B)[0]) <= TOL
            na = np.sqrt(np.sum(ga * ga, axis=(1, 2)))                    # U(-dt) is unitary: every vector
            assert np.max(np.abs(na - np.sqrt(model.N))) <= 1e-9 * np.sqrt(model.N)
            del ga, gb
    else:
        for rnd in range(n_rounds):                                       # evolve, measure ... [A4]
            g.evolve(w.dt, order)
            o.evolve(w.dt, order)
            gpsi, gchi = g.get_state(gq.STATE_PSI), g.get_state(gq.STATE_CHI)
            chi = o.get_state(oracle_mod.CHI)[0]
            assert vec_err(gpsi[sb], o.get_state(oracle_mod.PSI)[0]) <= TOL
            assert vec_err(gchi[sb], chi) <= TOL
            npsi = np.sqrt(np.sum(gpsi * gpsi, axis=(1, 2)))
            assert np.max(np.abs(npsi - np.sqrt(model.N))) <= 1e-9 * np.sqrt(model.N)
            chi2 = np.sum(gchi * gchi, axis=(1, 2))                       # <chi|chi> per vector
            del gpsi, gchi
            msd = g.msd(nm)
            assert np.max(np.abs(msd[:, 0] - chi2) / chi2) <= TOL         # C_0^MSD = <chi|chi>
            assert np.max(np.abs(msd) / chi2[:, None]) <= 1 + 1e-9
            assert np.max(np.abs(msd[sb, :P] - o.msd(P)[0])) / norm(chi) ** 2 <= TOL
        again = g.msd(nm)                                                 # fixed-order reductions
        assert again.tobytes() == msd.tobytes()
    g.close()
    o.close()
