"""Host-side logic of the C-ABI library, no GPU: the library loads, exports every symbol that
include/gpuqt.h declares, validates inputs with the documented status codes, and its Bessel table
(Miller recurrence) agrees with identities, textbook values and the oracle's libm-based table, the
tuning options have the documented defaults and create-time failures report through
gpuqt_last_error(NULL)."""
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


def test_options_and_create_errors(gq):
    """gpuqt_default_options documents the defaults; a failing gpuqt_create leaves its reason in
    gpuqt_last_error(NULL) instead of printing (checks that need no GPU run before any CUDA call)."""
    from paper_1705_01387_b200 import binding
    o = binding.default_options()
    assert o.struct_bytes == ctypes.sizeof(binding.Options)
    assert (o.stages, o.blocks_per_sm, o.run, o.alternate, o.hop_const, o.idx16, o.small, o.persistent) == \
        (0, 0, 0, 1, 1, 1, 1, -1)
    with pytest.raises(KeyError):
        binding.default_options(no_such_option=1)
    lib = gq.load()
    m = L.square(6, 5, W=2.0, seed=1)
    h = ctypes.c_void_p()
    dummy = ctypes.c_void_p(256)                      # never dereferenced: the calls below fail before any CUDA work

    def create(model, batch=1, options=None, volume=None):
        return lib.gpuqt_create_with_options(ctypes.byref(h), *binding._model_tuple(model),
                                             ctypes.c_double(model.volume if volume is None else volume),
                                             ctypes.c_double(model.energy_scale), ctypes.c_int32(batch), ctypes.c_int(0),
                                             dummy, ctypes.c_size_t(1 << 30), None,
                                             None if options is None else ctypes.byref(options))
    assert create(m, batch=3) == -1 and b"batch" in lib.gpuqt_last_error(None)
    assert create(m, volume=0.0) == -1
    bad = binding.default_options()
    bad.struct_bytes = 4096
    assert create(m, options=bad) == -1 and b"struct_bytes" in lib.gpuqt_last_error(None)
    assert create(m, options=binding.default_options(stages=9)) == -1
    broken = L.square(6, 5, W=2.0, seed=1)
    broken.nbr_index = broken.nbr_index.copy()
    broken.nbr_index[7] = broken.N
    assert create(broken) == -2 and b"out of range" in lib.gpuqt_last_error(None)
    assert h.value is None


def test_storage_plan_regular_lattices_need_no_index_array(gq):
    """gpuqt_plan_storage (host only): regular periodic lattices with one hopping value (the paper's default,
    PAPER.md:248, and its examples) are stored as an implicit stencil -- on-site energies
    plus a small dictionary of per-slice column patterns; vacancies, bond disorder and complex hoppings fall
    back to the explicit tables."""
    REAL, CPLX, CONST32, CONST16, CONST16P, STENCIL = range(6)
    MB = 1 << 20              # pretend L2 size: the stencil is only taken when a step's working set exceeds the L2
    # cubic 64^3: x-lines are two slices long -> patterns = {first, second half of a line} x {y = 0, mid, 63} x {z = 0, mid, 63}
    m = L.cubic(64, W=16.5, seed=1, energy_scale=16.0)
    hop, nbytes, pats = gq.plan_storage(m, batch=4, l2_bytes=MB, options={"reorder": 0})
    assert hop == STENCIL and pats == 2 * 3 * 3               # N is a multiple of 128 rows: no all-padding tail records
    # by default a recognised cubic lattice beyond the L2 is stored in bricks of 4 x 4 x 2 sites: one pattern per
    # (first, middle, last) brick position in each direction, same bytes
    hop_b, nbytes_b, pats_b = gq.plan_storage(m, batch=4, l2_bytes=MB)
    assert hop_b == STENCIL and pats_b == 3 * 3 * 3 and abs(nbytes_b - nbytes) <= 27 * 6 * 32 * 4
    assert nbytes < 8.2 * m.N + 8 * (m.N + 1)                  # 8 B on-site + 0.125 B pattern id per row (+ x)
    hop16, nbytes16, _ = gq.plan_storage(m, batch=4, l2_bytes=MB, options={"stencil": 0, "reorder": 0})
    assert hop16 == CONST16 and nbytes16 > nbytes + 12 * m.N   # 16-bit columns: 21 B per row at K = 6
    hop32, nbytes32, _ = gq.plan_storage(m, batch=4, l2_bytes=MB, options={"stencil": 0, "idx16": 0, "reorder": 0})
    assert hop32 == CONST32 and nbytes32 == (m.N // 32) * (256 + 128 * 6) + 8 * (m.N + 1)
    # square 1000 x 96 (lines not aligned with slices): a dozen patterns
    m = L.square(1000, 96, W=2.0, seed=2)
    hop, nbytes, pats = gq.plan_storage(m, batch=4, l2_bytes=MB)
    assert hop == STENCIL and 5 <= pats <= 40                   # where the line end falls in the slice x (first, middle, last line)
    # chain: K = 2
    assert gq.plan_storage(L.chain(100000, W=1.0, seed=3), batch=8, l2_bytes=MB)[0] == STENCIL
    # graphene (4-atom cell, period 4 in the row index)
    assert gq.plan_storage(L.graphene(256, 64, W=1.0, seed=4), batch=4, l2_bytes=MB)[0] == STENCIL
    # one or two vectors: a tile streams too few bytes to pay for the stencil's extra copies (the paper's example 5.1: 1.57 s
    # with explicit columns, 2.07 s with the stencil) -- explicit columns unless forced
    m1 = L.square(1000, 96, W=2.0, seed=2)
    assert gq.plan_storage(m1, batch=1, l2_bytes=MB)[0] != STENCIL and gq.plan_storage(m1, batch=2, l2_bytes=MB)[0] != STENCIL
    assert gq.plan_storage(m1, batch=1, l2_bytes=MB, options={"stencil": 2})[0] == STENCIL
    # fall-backs: vacancies (every slice its own pattern), bond disorder (per-entry hoppings), Peierls phases
    assert gq.plan_storage(L.graphene(256, 64, vacancy_fraction=0.01, vacancy_seed=5), l2_bytes=MB)[0] in (CONST32, CONST16, CONST16P)
    assert gq.plan_storage(L.with_bond_disorder(L.square(256, 64, W=1.0, seed=6), 0.3, 7), l2_bytes=MB)[0] == REAL
    assert gq.plan_storage(L.square_peierls(128, 64, flux_quanta=2), l2_bytes=MB)[0] == CPLX
    # small lattices: the dictionary would not pay; forced (option 2) it is still exact
    m = L.cubic(12, W=1.0, seed=8, energy_scale=8.0)
    assert gq.plan_storage(m, l2_bytes=MB)[0] != STENCIL and gq.plan_storage(m, l2_bytes=MB, options={"stencil": 2})[0] == STENCIL
    # on the real L2 (126 MB) a 64^3 lattice with 4 vectors (59 MB per step) keeps its explicit 16-bit columns:
    # the index array is re-read from L2 there, and the stencil's extra copies would only cost time
    m = L.cubic(64, W=16.5, seed=1, energy_scale=16.0)
    assert gq.plan_storage(m, batch=4)[0] == CONST16 and gq.plan_storage(m, batch=4, l2_bytes=32 * MB)[0] == STENCIL
    bad = L.square(8, 8)
    bad.nbr_index = bad.nbr_index.copy()
    bad.nbr_index[5] = bad.N
    with pytest.raises(gq.GpuqtError) as ei:
        gq.plan_storage(bad)
    assert ei.value.status == -2
