"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (default
options, the config's own batch B, N_m and N_p).

The oracle cannot run a whole config in seconds, so it follows the parity schedule of SURVEY.md
8(d): ONE sampled random vector (slot SLOT[key] of the batch, an inner slot, so the [N][B] interleave
is exercised) at full N through the config's OWN number of time steps; the oracle runs the evolutions
of the schedule and the evolved state vectors of the sample are compared element by element; the
sample's moments are compared over the WHOLE N_m at the first and at the last measured time step and
on the prefix n < 64 at every step in between (C_n does not depend on N_m [A19]).  Before that, EVERY
slot of the batch goes through one time step against the oracle (states element by element, prefix
moments), so no slot is left to properties alone.  c1-c4 run all their time steps (10, 20, 50, 40).
c5 (1.6e7 orbitals, complex hoppings, N_m = 3000, 30 steps) runs its first 2 steps with prefix moments
by default; GPUQT_PARITY_ALL_STEPS=1 runs all 30, GPUQT_PARITY_C5_FULL=1 adds the full N_m = 3000 VAC
comparison at full N at the first measured step (minutes of host time each: run once per round under
gpurun, log in profiles/r3_parity_full_schedule.txt); its full depth is also covered on a reduced
lattice of the same family in every run (test_c5_family_full_depth).  Properties that hold at any
size cover the other B - 1 vectors beyond the first step: C_0 = <phi|phi> = N, norm conservation of U,
|C_n| <= ||phi_L|| ||phi_R||, run-to-run bit identity.

Tolerances as in test_gpu_parity.py (north_star: 1e-10 in the norms of A22; tables bit-exact).
"""
import os

import numpy as np
import pytest

from workloads import configs
from workloads import lattices as L

pytestmark = pytest.mark.gpu

TOL = 1e-10
PREFIX = 64
ALL_STEPS = os.environ.get("GPUQT_PARITY_ALL_STEPS", "0") == "1"
C5_FULL = os.environ.get("GPUQT_PARITY_C5_FULL", "0") == "1"
STEPS = {"c1": 10, "c2": 20, "c3": 50, "c4": 40, "c5": 2}      # time steps run here (c1-c4: all of them)
SLOT = {"c4": 2, "c5": 5}                                      # the vector of the batch the oracle follows (default 0)


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


def every_slot_one_step(gq, oracle_mod, w, model, g, o, phi):
    """One time step of EVERY vector of the batch against the oracle (one vector at a time on the host): evolved
    states element by element, the first PREFIX moments in the A22 norms."""
    B, P = w.batch, min(PREFIX, w.n_moments)
    g.set_state(phi)
    g.evolve(w.dt, w.order)
    if w.path == "vac":
        got = {gq.STATE_VAC_A: g.get_state(gq.STATE_VAC_A), gq.STATE_VAC_B: g.get_state(gq.STATE_VAC_B)}
        names = {gq.STATE_VAC_A: oracle_mod.VAC_A, gq.STATE_VAC_B: oracle_mod.VAC_B}
        mom = g.vac(P)
    else:
        got = {gq.STATE_PSI: g.get_state(gq.STATE_PSI), gq.STATE_CHI: g.get_state(gq.STATE_CHI)}
        names = {gq.STATE_PSI: oracle_mod.PSI, gq.STATE_CHI: oracle_mod.CHI}
        mom = g.msd(P)
    worst = 0.0
    for b in range(B):
        o.set_state(phi[b:b + 1])
        o.evolve(w.dt, w.order)
        for which, ow in names.items():
            err = vec_err(got[which][b], o.get_state(ow)[0])
            assert err <= TOL, (b, which, err)
        if w.path == "vac":
            scale = norm(o.apply_v(o.get_state(oracle_mod.VAC_A)[0])) * norm(o.get_state(oracle_mod.VAC_B)[0])
            err = np.max(np.abs(mom[b] - o.vac(P)[0])) / scale
        else:
            err = np.max(np.abs(mom[b] - o.msd(P)[0])) / norm(o.get_state(oracle_mod.CHI)[0]) ** 2
        worst = max(worst, err)
        assert err <= TOL, (b, err)
    print(f"{w.key}: every slot of B={B} through one step: worst moment error {worst:.2e}")


def run_schedule(gq, oracle_mod, w, model, n_steps, full_depth, vector_checks, full_at=None, dos_full=None, sb=0):
    """The schedule of the module docstring for one workload; `full_depth`: compare all N_m moments at the measured
    steps `full_at` (default: the first and the last; else the prefix there as well) and, with `dos_full` (default:
    full_depth), of the DOS; `vector_checks`: the steps (0-based) after whose evolution the state vectors are compared;
    `sb`: the slot of the batch the oracle follows."""
    order = w.order
    B, nm = w.batch, w.n_moments
    full_at = {0, n_steps - 1} if full_at is None else full_at
    dos_full = full_depth if dos_full is None else dos_full
    phi = w.phases(model)
    modes_g = gq.MODE_MSD if w.path == "msd" else gq.MODE_VAC
    modes_o = oracle_mod.MODE_MSD if w.path == "msd" else oracle_mod.MODE_VAC
    g = gq.GpuQT(model, batch=B, modes=modes_g)
    o = oracle_mod.Oracle(model, batch=1, modes=modes_o)

    # a1: the device table decodes to the oracle's padded ELL, bit for bit (col, re, im, dx)
    for a, b in zip(g.get_table(), o.get_table()):
        assert a.tobytes() == b.tobytes()

    if B > 1:
        every_slot_one_step(gq, oracle_mod, w, model, g, o, phi)

    g.set_state(phi)
    o.set_state(phi[sb:sb + 1])

    def depth(k):                                     # moments the oracle computes at measured step k
        return nm if (full_depth and k in full_at) else min(PREFIX, nm)

    # a6 (DOS): full N_m on the GPU
    dos = g.dos_moments(nm)
    assert dos.shape == (B, nm)
    assert np.max(np.abs(dos[:, 0] - model.N)) <= TOL * model.N            # C_0 = <phi|phi> = N  [A7]
    assert np.max(np.abs(dos)) <= model.N * (1 + 1e-9)                     # |T_n| <= 1 on the spectrum
    P = nm if dos_full else min(PREFIX, nm)
    assert np.max(np.abs(dos[sb, :P] - o.dos_moments(P)[0])) / model.N <= TOL

    worst = 0.0
    if w.path == "vac":
        for k in range(n_steps):                                          # measure, evolve, measure ... [A4]
            vac = g.vac(nm)
            va, vb = o.get_state(oracle_mod.VAC_A)[0], o.get_state(oracle_mod.VAC_B)[0]
            scale = norm(o.apply_v(va)) * norm(vb)
            P = depth(k)
            err = np.max(np.abs(vac[sb, :P] - o.vac(P)[0])) / scale
            worst = max(worst, err)
            assert err <= TOL, (k, P, err)
            if k == n_steps - 1:
                break
            g.evolve(w.dt, order)
            o.evolve(w.dt, order)
            if k in vector_checks:
                ga, gb = g.get_state(gq.STATE_VAC_A), g.get_state(gq.STATE_VAC_B)
                assert vec_err(ga[sb], o.get_state(oracle_mod.VAC_A)[0]) <= TOL
                assert vec_err(gb[sb], o.get_state(oracle_mod.VAC_B)[0]) <= TOL
                na = np.sqrt(np.sum(ga * ga, axis=(1, 2)))                # U(-dt) is unitary: every vector
                assert np.max(np.abs(na - np.sqrt(model.N))) <= 1e-9 * np.sqrt(model.N)
                del ga, gb
        again = g.vac(nm)
        assert again.tobytes() == vac.tobytes()                           # fixed-order reductions
    else:
        for k in range(n_steps):                                          # evolve, measure ... [A4]
            g.evolve(w.dt, order)
            o.evolve(w.dt, order)
            chi = o.get_state(oracle_mod.CHI)[0]
            if k in vector_checks:
                gpsi, gchi = g.get_state(gq.STATE_PSI), g.get_state(gq.STATE_CHI)
                assert vec_err(gpsi[sb], o.get_state(oracle_mod.PSI)[0]) <= TOL
                assert vec_err(gchi[sb], chi) <= TOL
                npsi = np.sqrt(np.sum(gpsi * gpsi, axis=(1, 2)))
                assert np.max(np.abs(npsi - np.sqrt(model.N))) <= 1e-9 * np.sqrt(model.N)
                chi2 = np.sum(gchi * gchi, axis=(1, 2))                   # <chi|chi> per vector
                del gpsi, gchi
            msd = g.msd(nm)
            if k in vector_checks:
                assert np.max(np.abs(msd[:, 0] - chi2) / chi2) <= TOL     # C_0^MSD = <chi|chi>
                assert np.max(np.abs(msd) / chi2[:, None]) <= 1 + 1e-9
            P = depth(k)
            err = np.max(np.abs(msd[sb, :P] - o.msd(P)[0])) / norm(chi) ** 2
            worst = max(worst, err)
            assert err <= TOL, (k, P, err)
        again = g.msd(nm)                                                 # fixed-order reductions
        assert again.tobytes() == msd.tobytes()
    deep = sorted(k for k in full_at if 0 <= k < n_steps) if full_depth else []
    print(f"{w.key}: N={model.N} B={B} slot={sb} N_m={nm} steps={n_steps} (all N_m at steps {deep}, n < {PREFIX} elsewhere): "
          f"worst moment error {worst:.2e} (A22 norm), states at steps {sorted(k for k in vector_checks if 0 <= k < n_steps)} <= {TOL:g}")
    g.close()
    o.close()


@pytest.mark.parametrize("key", ["c1", "c2", "c3", "c4", "c5"])
def test_full_size_config(gq, oracle_mod, key):
    w = configs.WORKLOADS[key]
    model = w.build()
    n_steps = w.n_steps if ALL_STEPS else min(STEPS[key], w.n_steps)
    checks = {0, 1, n_steps // 2, n_steps - 2, n_steps - 1}
    if key == "c5":           # full N_m = 3000 of the VAC at the first measured step only, and only on request
        run_schedule(gq, oracle_mod, w, model, n_steps, full_depth=C5_FULL, vector_checks=checks, full_at={0}, dos_full=False,
                     sb=SLOT[key])
    else:
        run_schedule(gq, oracle_mod, w, model, n_steps, full_depth=True, vector_checks=checks, sb=SLOT.get(key, 0))


def test_c5_family_full_depth(gq, oracle_mod):
    """c5's family (Peierls phases, Gaussian-correlated potential, complex hoppings, B = 8, VAC) at
    700 x 350 four-atom cells = 980 000 orbitals: all N_m = 3000 moments of the sampled vector at the
    first and the last of 3 measured steps."""
    w = configs.WORKLOADS["c5"]
    model = L.graphene_peierls_correlated(700, 350, config=5)
    run_schedule(gq, oracle_mod, w, model, 3, full_depth=True, vector_checks={0, 1})
