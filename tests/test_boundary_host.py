"""Host-side logic of the C-ABI library, no GPU: the library loads, exports every symbol that
include/gpuqt.h declares, validates inputs with the documented status codes, and its Bessel table
(Miller recurrence) agrees with identities, textbook values and the oracle's libm-based table."""
import ctypes
import os
import re

import numpy as np
import pytest

from workloads import lattices as L

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def gq():
    from paper_1705_01387_b200 import build
    build.build()
    import paper_1705_01387_b200 as g
    g.load()
    return g


def test_every_declared_symbol_is_exported(gq):
    header = open(os.path.join(ROOT, "include", "gpuqt.h")).read()
    declared = set(re.findall(r"\b(gpuqt_[a-z_]+)\s*\(", header))
    declared -= {"gpuqt_status"}
    assert {"gpuqt_create", "gpuqt_dos_moments", "gpuqt_evolve", "gpuqt_vac", "gpuqt_msd", "gpuqt_destroy"} <= declared
    lib = ctypes.CDLL(os.path.join(ROOT, "paper_1705_01387_b200", "libgpuqt.so"))
    for name in sorted(declared):
        assert hasattr(lib, name), f"{name} declared in gpuqt.h but not exported"
    from paper_1705_01387_b200 import binding
    assert declared == set(binding._SIGNATURES), "binding and header must list the same entry points"


def test_validate_status_codes(gq):
    m = L.square(6, 5, W=2.0, seed=1)
    assert gq.validate(m) == 0
    bad = L.square(6, 5, W=2.0, seed=1)
    bad.nbr_index = bad.nbr_index.copy()
    bad.nbr_index[7] = bad.N
    assert gq.validate(bad) == -2                      # GPUQT_ERR_INDEX
    bad = L.square(6, 5, W=2.0, seed=1)
    bad.nbr_count = bad.nbr_count.copy()
    bad.nbr_count[3] = 5
    assert gq.validate(bad) == -2
    bad = L.square_peierls(6, 5, flux_quanta=1)
    bad.hop_im = bad.hop_im.copy()
    bad.hop_im[0] = -bad.hop_im[0] + 0.25              # break conjugate symmetry
    assert gq.validate(bad) == -3                      # GPUQT_ERR_NOT_HERMITIAN
    bad = L.square(6, 5, W=2.0, seed=1)
    bad.nbr_count = bad.nbr_count.copy()
    bad.nbr_count[0] = 3                               # one directed bond missing
    assert gq.validate(bad) == -3
    bad = L.square(6, 5, W=2.0, seed=1, energy_scale=4.5)
    assert gq.validate(bad) == -4                      # GPUQT_ERR_SCALE (Gershgorin 4 + |U| > 4.5 somewhere)
    bad = L.chain(4)
    bad.x = np.array([0.0, 2.0, 1.0, 3.0])             # |X_n - X_m| = L/2 on a bond
    assert gq.validate(bad) == -9                      # GPUQT_ERR_POSITION
    bad = L.chain(8)
    bad.energy_scale = -1.0
    assert gq.validate(bad) == -1
    # every generator output used by the benchmarks validates
    for m in (L.cubic(6, W=16.5, seed=1, energy_scale=16.0), L.graphene(5, 4, W=1.0, seed=2),
              L.graphene(6, 5, vacancy_fraction=0.05, vacancy_seed=3), L.square_peierls(7, 6, 2)):
        assert gq.validate(m) == 0


def test_workspace_bytes(gq):
    lib = gq.load()
    a = lib.gpuqt_workspace_bytes(4096000, 6, 0, 4, 2)
    assert 2.5e9 < a < 4e9                             # ~10 vector sets of 262 MB + 360 MB matrix
    assert lib.gpuqt_workspace_bytes(1000, 4, 0, 3, 0) == 0    # unsupported batch
    assert lib.gpuqt_workspace_bytes(0, 4, 0, 1, 0) == 0
    assert lib.gpuqt_workspace_bytes(1000, 4, 1, 1, 3) > lib.gpuqt_workspace_bytes(1000, 4, 0, 1, 3)


def test_bessel_table(gq, oracle_mod):
    gold = np.loadtxt(os.path.join(ROOT, "tests", "golden", "bessel_j_at_1.txt"))
    c = gq.bessel_coeffs(1.0, 1.0, 4)
    J = np.array([c[0].real, -c[1].imag / 2, -c[2].real / 2, c[3].imag / 2])
    assert np.allclose(J, gold, rtol=0, atol=5e-11)
    for dE, dt in ((16.0, 1.0), (10.0, 1.0), (5.1, 2.0), (6.1, 0.2), (4.1, 100.0), (4.1, -0.1), (10.0, -2.0)):
        n = int(dE * abs(dt)) + 70
        c = gq.bessel_coeffs(dE, dt, n)
        ref = oracle_mod.bessel_coeffs(dE, dt, n)       # libm jn(): an independent routine
        assert np.max(np.abs(c - ref)) < 4e-15
        Jm = np.abs(c) / np.where(np.arange(n) == 0, 1.0, 2.0)
        assert abs(Jm[0] ** 2 + 2 * np.sum(Jm[1:] ** 2) - 1.0) < 1e-13
    # tail rule used to choose N_p [A5]: smallest N_p with |J_m| < 1e-15 for m >= N_p
    for x, expect in ((10.0, 34), (16.0, 44), (20.0, 50)):
        Jm = np.abs(gq.bessel_coeffs(x, 1.0, 120)) / 2
        n_p = int(np.max(np.nonzero(Jm >= 1e-15)[0])) + 1
        assert n_p == expect
    assert gq.bessel_coeffs(3.0, 0.0, 3).tolist() == [1.0, 0.0, 0.0]


def test_no_gpu_fails_loudly(gq):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        gq.GpuQT(L.chain(8), batch=1)


def _csr(sets):
    ptr = np.zeros(len(sets) + 1, np.int32)
    ptr[1:] = np.cumsum([len(x) for x in sets])
    return ptr, np.array([v for x in sets for v in sorted(x)], np.int32)


def _check_schedule(sets, run, grid, reverse, slack):
    """Invariants the fused kernel relies on (kernels.cuh, cheb_step_kernel): `sets[s]` = slices that
    slice s gathers from."""
    from paper_1705_01387_b200 import binding
    n = len(sets)
    ptr, lst = _csr(sets)
    items, dep_ptr, dep_list = binding.fused_schedule(ptr, lst, run, grid, reverse, slack)
    NO = (1 << 30) - 1
    n_runs = (n + run - 1) // run
    runs, steps = items[:, 0] & NO, (items[:, 0] >> 30) & 1
    real = runs != NO
    # every run exactly once per step; first-step items in sweep order
    assert list(runs[real & (steps == 0)]) == list(range(n_runs))
    assert sorted(runs[real & (steps == 1)]) == list(range(n_runs))
    assert np.all(steps[~real] == 0)
    pos1 = {int(r): t for t, r in enumerate(runs) if r != NO and steps[t] == 0}
    virt = (lambda s_: n - 1 - s_) if reverse else (lambda s_: s_)
    for R in range(n_runs):
        need = set()
        for vs in range(R * run, min(n, (R + 1) * run)):
            need |= {virt(d) // run for d in sets[virt(vs)]}
        assert R in need
        assert sorted(need) == list(dep_list[dep_ptr[R]:dep_ptr[R + 1]])     # exactly the runs gathered from
    for t in np.nonzero(real & (steps == 1))[0]:
        deps = dep_list[dep_ptr[runs[t]]:dep_ptr[runs[t] + 1]]
        # a second-step item depends only on EARLIER items (no deadlock), at least `slack` back
        assert max(pos1[int(r)] for r in deps) + slack <= t
    return items


def test_fused_schedule_invariants():
    rng_ = np.random.default_rng(5)
    # periodic cubic 12^3 in slices of 32 rows: neighbours +-1, +-12, +-144 rows with wrap-around
    L3 = 12
    N = L3 ** 3
    n = (N + 31) // 32
    sets = [{s_} for s_ in range(n)]
    for m in range(N):
        x, y, z = m % L3, (m // L3) % L3, m // (L3 * L3)
        for c in (((x - 1) % L3, y, z), ((x + 1) % L3, y, z), (x, (y - 1) % L3, z), (x, (y + 1) % L3, z),
                  (x, y, (z - 1) % L3), (x, y, (z + 1) % L3)):
            sets[m >> 5].add((c[0] + L3 * (c[1] + L3 * c[2])) >> 5)
    for run, grid, reverse, slack in ((8, 3, 0, 3), (8, 3, 1, 1), (16, 2, 0, 2), (8, 7, 1, 10), (8, 100, 0, 100)):
        _check_schedule(sets, run, grid, reverse, slack)
    # banded open chain: the second sweep follows the first at a constant distance, few no-ops
    n = 4000
    sets = [{max(s_ - 1, 0), s_, min(s_ + 1, n - 1)} for s_ in range(n)]
    items = _check_schedule(sets, 8, 16, 0, 16)
    assert len(items) <= 2 * 500 + 3 * 16
    # both kinds of work reach every CTA: within any two consecutive rounds a CTA sees both steps
    steps = (items[:, 0] >> 30) & 1
    for c in range(16):
        mine = steps[c::16][2:-3]
        assert 0 < mine.mean() < 1
    # arbitrary sparsity: still valid (the second step simply follows the whole first sweep)
    n = 300
    sets = [{s_, int(rng_.integers(0, n)), int(rng_.integers(0, n))} for s_ in range(n)]
    _check_schedule(sets, 8, 5, 0, 5)
    _check_schedule(sets, 8, 5, 1, 5)
