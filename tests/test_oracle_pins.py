"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Every test compares oracle/ with something that is NOT the oracle: dense exact diagonalisation
(tests/dense_ref.py), closed forms, textbook values, or identities.  SURVEY.md 8(c) "Pins".
"""
import os

import numpy as np
import pytest

from tests import dense_ref as D
from workloads import lattices as L
from workloads import rng

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def rand_vec(N, seed):
    u = rng.uniform01(seed, 2 * N)
    return np.stack([u[:N] - 0.5, u[N:] - 0.5], axis=1)


def models():
    return [
        L.square(6, 5, W=2.0, seed=11),                       # periodic, disorder, default hops
        L.square(5, 4, W=1.0, seed=12, periodic=False),       # open boundary, ragged counts
        L.square_peierls(6, 5, flux_quanta=2, W=1.5, seed=13),  # complex hoppings
        L.graphene(3, 3, W=1.0, seed=14),                     # explicit real hoppings -2.7
        L.graphene(4, 3, vacancy_fraction=0.1, vacancy_seed=5),  # rows with 0-3 neighbours
        L.chain(9, W=0.5, seed=15),
        L.random_graph(40, 5, 16, complex_hops=True, degree_fill=0.8),    # random bonds, rows of 0..5 neighbours in random order
        L.random_graph(37, 3, 17, complex_hops=False, degree_fill=0.9, locality=6, open_x=False),
    ]


# --------------------------------------------------------------------- operators vs dense
@pytest.mark.parametrize("model", models(), ids=lambda m: m.name)
def test_operators_match_dense(oracle_mod, model):
    o = oracle_mod.Oracle(model)
    H = D.dense_H(model)
    assert np.allclose(H, H.conj().T, atol=0), "generator must give a Hermitian H"
    V = D.dense_V(model, H)
    assert np.allclose(V, V.conj().T, atol=1e-15), "V is Hermitian"
    X = np.diag(model.x)
    v = rand_vec(model.N, 77)
    z = D.to_c(v)
    assert np.allclose(D.to_c(o.apply_h(v)), (H @ z) / model.energy_scale, rtol=0, atol=1e-14)
    assert np.allclose(D.to_c(o.apply_v(v)), V @ z, rtol=0, atol=1e-13)
    # [X, H~] = i V / dE  (from V = i[H, X] = i(HX - XH)); on open lattices also the literal XH - HX
    assert np.allclose(D.to_c(o.apply_xh(v)), (1j * V @ z) / model.energy_scale, rtol=0, atol=1e-13)
    if model.box_length <= 0:
        assert np.allclose(D.to_c(o.apply_xh(v)), ((X @ H - H @ X) @ z) / model.energy_scale, atol=1e-13)


def test_table_padding_and_defaults(oracle_mod):
    model = L.graphene(4, 3, vacancy_fraction=0.1, vacancy_seed=5)
    o = oracle_mod.Oracle(model)
    col, re, im, dx = o.get_table()
    K = model.K
    for m in range(model.N):
        c = model.nbr_count[m]
        assert np.array_equal(col[m * K:m * K + c], model.nbr_index[m * K:m * K + c])
        assert np.all(col[m * K + c:(m + 1) * K] == m)          # padding = own row
        assert np.all(re[m * K + c:(m + 1) * K] == 0.0)
    sq = L.square(4, 4)
    _, re, im, dx = oracle_mod.Oracle(sq).get_table()
    assert np.all(re == -1.0) and np.all(im == 0.0)             # PAPER.md:248 default -1
    # minimum image: neighbours [-x,+x,-y,+y] -> dx = -1, +1, 0, 0 everywhere incl. the seam
    assert np.array_equal(dx.reshape(-1, 4), np.tile([-1.0, 1.0, 0.0, 0.0], (16, 1)))


# --------------------------------------------------------------------- Bessel coefficients
def test_bessel_textbook_values_and_identities(oracle_mod):
    # J_0..J_3(1): Abramowitz & Stegun Table 9.1 (tests/golden/bessel_j_at_1.txt)
    gold = np.loadtxt(os.path.join(GOLD, "bessel_j_at_1.txt"))
    c = oracle_mod.bessel_coeffs(1.0, 1.0, 4)
    J = np.array([c[0].real, -c[1].imag / 2, -c[2].real / 2, c[3].imag / 2])
    assert np.allclose(J, gold, rtol=0, atol=5e-11)
    for x in (0.41, 1.22, 10.0, 16.0, 20.4):
        n = int(x) + 60
        c = oracle_mod.bessel_coeffs(2.0, x / 2.0, n)
        J = np.abs(c) / np.where(np.arange(n) == 0, 1.0, 2.0)
        # J_0^2 + 2 sum J_m^2 = 1
        assert abs(J[0] ** 2 + 2 * np.sum(J[1:] ** 2) - 1.0) < 1e-14
        # phases (-i)^m for +dt, (+i)^m for -dt   (Eq. 17)
        cm = oracle_mod.bessel_coeffs(2.0, -x / 2.0, n)
        assert np.allclose(cm, np.conj(c), atol=0)
        m = np.arange(n)
        Jsigned = (c / ((-1j) ** m) / np.where(m == 0, 1.0, 2.0)).real
        # J_0 + 2 sum_k J_2k = 1 ; generating function at theta=0
        assert abs(Jsigned[0] + 2 * np.sum(Jsigned[2::2]) - 1.0) < 1e-13


# --------------------------------------------------------------------- U(dt) vs dense exp(-iHt)
@pytest.mark.parametrize("model", models()[:4], ids=lambda m: m.name)
@pytest.mark.parametrize("dt", [0.7, -1.3])
def test_evolve_matches_dense_expm(oracle_mod, model, dt):
    o = oracle_mod.Oracle(model)
    H = D.dense_H(model)
    v = rand_vec(model.N, 3)
    ref = D.dense_U(H, dt) @ D.to_c(v)
    got = D.to_c(o.evolve_vec(v, dt, 60))
    assert np.max(np.abs(got - ref)) < 2e-14            # "machine precision"
    # norm preservation and reversibility
    assert abs(np.linalg.norm(got) - np.linalg.norm(D.to_c(v))) < 1e-13
    back = D.to_c(o.evolve_vec(D.from_c(got), -dt, 60))
    assert np.max(np.abs(back - D.to_c(v))) < 5e-14


def test_evolve_truncation_matters(oracle_mod):
    """A dropped Chebyshev term or wrong tail must be visible: too few terms gives a large error."""
    model = L.square(6, 5, W=2.0, seed=11)
    o = oracle_mod.Oracle(model)
    v = rand_vec(model.N, 3)
    ref = D.dense_U(D.dense_H(model), 2.0) @ D.to_c(v)
    err_small = np.max(np.abs(D.to_c(o.evolve_vec(v, 2.0, 8)) - ref))
    err_full = np.max(np.abs(D.to_c(o.evolve_vec(v, 2.0, 45)) - ref))
    assert err_small > 1e-3 and err_full < 2e-14


# --------------------------------------------------------------------- [X,U] vs dense XU - UX
def test_commutator_single_and_multi_step_open_boundary(oracle_mod):
    model = L.square(5, 4, W=1.0, seed=12, periodic=False)
    o = oracle_mod.Oracle(model, batch=1)
    H = D.dense_H(model)
    X = np.diag(model.x)
    v = rand_vec(model.N, 9)
    z = D.to_c(v)
    U = D.dense_U(H, 0.6)
    got = D.to_c(o.commutator_vec(v, 0.6, 50))
    assert np.max(np.abs(got - (X @ U - U @ X) @ z)) < 5e-14
    # multi-step with non-uniform steps: chi(t) = [X, U(t)] phi by the product rule [A3]
    o.set_state(v[None])
    t = 0.0
    for dt in (0.3, 0.9, 0.5, 1.1, 0.2):
        o.evolve(dt, 55)
        t += dt
    Ut = D.dense_U(H, t)
    assert np.max(np.abs(D.to_c(o.get_state(oracle_mod.CHI)[0]) - (X @ Ut - Ut @ X) @ z)) < 2e-13
    assert np.max(np.abs(D.to_c(o.get_state(oracle_mod.PSI)[0]) - Ut @ z)) < 1e-13
    # VAC branches step with U(-dt)  [A1]
    V = D.dense_V(model, H)
    assert np.max(np.abs(D.to_c(o.get_state(oracle_mod.VAC_A)[0]) - Ut.conj().T @ z)) < 1e-13
    assert np.max(np.abs(D.to_c(o.get_state(oracle_mod.VAC_B)[0]) - Ut.conj().T @ (V @ z))) < 2e-13


# --------------------------------------------------------------------- plane-wave closed forms
def test_plane_wave_closed_forms_hand_example(oracle_mod):
    """4-site ring, gamma = 1, k = pi/2: eps = 0, v = 2 =>
    C_n^DOS = 4 cos(n pi/2), C_n^VAC = 16 cos(n pi/2), C_n^MSD(t) = 16 t^2 cos(n pi/2).
    (tests/golden/ring4_plane_wave.txt; derivation in DESIGN.md 'Pins')"""
    gold = np.loadtxt(os.path.join(GOLD, "ring4_plane_wave.txt"))   # columns: n, DOS, VAC, MSD/t^2
    model = L.chain(4, energy_scale=2.5)
    o = oracle_mod.Oracle(model)
    k = np.pi / 2
    phi = np.exp(1j * k * model.x)
    o.set_state(D.from_c(phi)[None])
    n = gold.shape[0]
    assert np.allclose(o.dos_moments(n)[0], gold[:, 1], atol=1e-13)
    assert np.allclose(o.vac(n)[0], gold[:, 2], atol=1e-12)
    t = 0.0
    for dt in (0.4, 0.8):
        o.evolve(dt, 30)
        t += dt
        assert np.allclose(o.msd(n)[0], gold[:, 3] * t * t, atol=1e-11)
        assert np.allclose(o.vac(n)[0], gold[:, 2], atol=1e-11)       # time independent


@pytest.mark.parametrize("kq", [1, 3, 5])
def test_plane_wave_general_k(oracle_mod, kq):
    """Clean ring of 12 sites: H~phi = (eps_k/dE) phi, V phi = v_k phi, v_k = 2 sin k,
    [X,U(t)]phi = t v_k e^{-i eps_k t} phi, C_n^MSD = N t^2 v_k^2 T_n(eps_k/dE)."""
    Ls, dE, t = 12, 2.3, 0.9
    model = L.chain(Ls, energy_scale=dE)
    o = oracle_mod.Oracle(model)
    k = 2 * np.pi * kq / Ls
    eps, vk = -2 * np.cos(k), 2 * np.sin(k)
    phi = np.exp(1j * k * model.x)
    v = D.from_c(phi)
    assert np.allclose(D.to_c(o.apply_h(v)), eps / dE * phi, atol=5e-15)
    assert np.allclose(D.to_c(o.apply_v(v)), vk * phi, atol=1e-14)
    assert np.allclose(D.to_c(o.evolve_vec(v, t, 40)), np.exp(-1j * eps * t) * phi, atol=1e-14)
    assert np.allclose(D.to_c(o.commutator_vec(v, t, 40)), t * vk * np.exp(-1j * eps * t) * phi, atol=1e-13)
    o.set_state(v[None])
    o.evolve(t, 40)
    n = np.arange(20)
    Tn = np.cos(n * np.arccos(eps / dE))
    assert np.allclose(o.msd(20)[0], Ls * t * t * vk * vk * Tn, atol=1e-11)   # ballistic ~ t^2
    assert np.allclose(o.vac(20)[0], Ls * vk * vk * Tn, atol=1e-11)
    assert np.allclose(o.dos_moments(20)[0], Ls * Tn, atol=1e-11)


# --------------------------------------------------------------------- moments vs exact trace
def test_moments_sum_over_basis_is_exact_trace(oracle_mod):
    model = L.square_peierls(5, 4, flux_quanta=1, W=2.0, seed=21)
    o = oracle_mod.Oracle(model)
    H = D.dense_H(model)
    w = np.linalg.eigvalsh(H / model.energy_scale)
    nm = 24
    exact = np.array([np.sum(np.cos(n * np.arccos(w))) for n in range(nm)])
    acc = np.zeros(nm, dtype=complex)
    for i in range(model.N):
        e = np.zeros((model.N, 2))
        e[i, 0] = 1.0
        acc += o.moments_vec(e, e, nm)
    assert np.allclose(acc.real, exact, atol=1e-12) and np.max(np.abs(acc.imag)) < 1e-13
    # low moments: Tr H~ = sum U / dE ; mu_2 = 2 Tr H~^2 - N
    assert abs(exact[1] - np.sum(model.onsite) / model.energy_scale) < 1e-12
    trh2 = (np.sum(model.onsite ** 2) + np.sum(model.hop_re ** 2 + model.hop_im ** 2)) / model.energy_scale ** 2
    assert abs(acc.real[2] - (2 * trh2 - model.N)) < 1e-12


def test_clean_ring_trace_special_case(oracle_mod):
    """Clean ring, H_mn = -gamma, dE = 2 gamma: eigenvalues -cos(2 pi j/N), T_n(-cos k) =
    (-1)^n cos(n k), so Tr T_n = (-1)^n N if n = 0 mod N else 0."""
    Ls = 7
    model = L.chain(Ls, energy_scale=2.0)
    o = oracle_mod.Oracle(model)
    acc = np.zeros(2 * Ls + 1, dtype=complex)
    for i in range(Ls):
        e = np.zeros((Ls, 2))
        e[i, 0] = 1.0
        acc += o.moments_vec(e, e, 2 * Ls + 1)
    n = np.arange(2 * Ls + 1)
    expect = np.where(n % Ls == 0, Ls * (-1.0) ** n, 0.0)
    assert np.allclose(acc.real, expect, atol=1e-12)


def test_random_phase_estimate_converges(oracle_mod):
    """Tr[A] ~ <phi|A|phi> with error ~ 1/sqrt(R N): averaging 64 vectors on a
    400-site lattice must agree with the exact trace to a few 1/sqrt(R N) and beat a single one."""
    model = L.square(20, 20, W=2.0, seed=31)
    o = oracle_mod.Oracle(model)
    w = np.linalg.eigvalsh(D.dense_H(model) / model.energy_scale)
    nm = 12
    exact = np.array([np.sum(np.cos(n * np.arccos(w))) for n in range(nm)]) / model.N
    R = 64
    phis = L.random_phase_vectors(model.N, R, config=99)
    est = np.array([o.moments_vec(phis[r], phis[r], nm).real for r in range(R)]) / model.N
    assert np.allclose(est[:, 0], 1.0, atol=1e-13)                 # <phi|phi> = N
    err_avg = np.max(np.abs(est.mean(axis=0) - exact))
    err_one = np.mean(np.max(np.abs(est - exact), axis=1))
    assert err_avg < 4.0 / np.sqrt(R * model.N)
    assert err_avg < 0.5 * err_one


def test_low_moments_identities(oracle_mod):
    model = L.graphene(3, 3, W=1.0, seed=14)
    o = oracle_mod.Oracle(model)
    H = D.dense_H(model) / model.energy_scale
    l, r = rand_vec(model.N, 1), rand_vec(model.N, 2)
    c = o.moments_vec(l, r, 4)
    zl, zr = D.to_c(l), D.to_c(r)
    assert abs(c[0] - np.vdot(zl, zr)) < 1e-14                    # conj on the LEFT vector
    assert abs(c[1] - np.vdot(zl, H @ zr)) < 1e-14
    assert abs(c[2] - np.vdot(zl, (2 * H @ H - np.eye(model.N)) @ zr)) < 1e-14
    assert abs(c[3] - np.vdot(zl, (4 * H @ H @ H - 3 * H) @ zr)) < 1e-14


# --------------------------------------------------------------------- VAC / MSD vs dense
def test_vac_and_msd_match_dense(oracle_mod):
    model = L.square_peierls(6, 5, flux_quanta=2, W=1.5, seed=13)
    B = 2
    o = oracle_mod.Oracle(model, batch=B)
    H = D.dense_H(model)
    V = D.dense_V(model, H)
    phis = L.random_phase_vectors(model.N, B, config=98)
    o.set_state(phis)
    nm = 10
    Tn = [D.dense_Tn(H, model.energy_scale, n) for n in range(nm)]
    t = 0.0
    for step, dt in enumerate((0.5, 0.7, 0.4)):
        U = D.dense_U(H, t)
        vac = o.vac(nm)                                  # measure, then evolve [A4]
        for b in range(B):
            z = D.to_c(phis[b])
            ref = [np.real(np.vdot(z, U @ V @ Tn[n] @ U.conj().T @ V @ z)) for n in range(nm)]
            assert np.allclose(vac[b], ref, atol=2e-11)
        o.evolve(dt, 50)
        t += dt
    # trace of Re-part is invariant under t -> -t, a single vector is not  [A1]
    U = D.dense_U(H, t)
    tr_p = sum(np.trace(U @ V @ Tn[n] @ U.conj().T @ V) for n in (3,))
    tr_m = sum(np.trace(U.conj().T @ V @ Tn[n] @ U @ V) for n in (3,))
    assert abs(tr_p.real - tr_m.real) < 1e-10


def test_msd_dense_open_boundary_and_short_time_link(oracle_mod):
    model = L.square(5, 4, W=1.0, seed=12, periodic=False)
    o = oracle_mod.Oracle(model)
    H = D.dense_H(model)
    X = np.diag(model.x)
    V = D.dense_V(model, H)
    phi = L.random_phase_vectors(model.N, 1, config=97)
    z = D.to_c(phi[0])
    nm = 8
    Tn = [D.dense_Tn(H, model.energy_scale, n) for n in range(nm)]
    o.set_state(phi)
    vac0 = o.vac(nm)[0]
    ref0 = [np.real(np.vdot(V @ z, Tn[n] @ V @ z)) for n in range(nm)]
    assert np.allclose(vac0, ref0, atol=1e-12)
    o.evolve(1e-3, 12)
    # C^MSD(t)/t^2 -> C^VAC(0) as t -> 0
    assert np.allclose(o.msd(nm)[0] / 1e-6, vac0, rtol=0, atol=2e-3 * np.max(np.abs(vac0)))
    o.evolve(0.8, 50)
    U = D.dense_U(H, 0.801)
    chi = (X @ U - U @ X) @ z
    ref = [np.real(np.vdot(chi, Tn[n] @ chi)) for n in range(nm)]
    assert np.allclose(o.msd(nm)[0], ref, atol=1e-11)


# --------------------------------------------------------------------- Jackson + transform
def test_jackson_values(oracle_mod):
    # Eq. 31 evaluated by hand for N_m = 4 (tests/golden/jackson_nm4.txt): 1, cos(pi/5), 1/sqrt5, ...
    gold = np.loadtxt(os.path.join(GOLD, "jackson_nm4.txt"))
    assert np.allclose(oracle_mod.jackson(4), gold, atol=5e-9)
    g = oracle_mod.jackson(4)
    assert abs(g[1] - np.cos(np.pi / 5)) < 1e-15 and abs(g[2] - 1 / np.sqrt(5)) < 1e-15
    g = oracle_mod.jackson(1000)
    assert g[0] == 1.0 and np.all(np.diff(g) < 0) and g[-1] > 0
    # equivalent standard form [A14]
    n = np.arange(1000)
    std = ((1000 - n + 1) * np.cos(np.pi * n / 1001) + np.sin(np.pi * n / 1001) / np.tan(np.pi / 1001)) / 1001
    assert np.allclose(g, std, atol=1e-14)


def test_transform_integral_and_chain_dos(oracle_mod):
    # integral of rho over the band = 2 C_0 / Omega, exact by Chebyshev-Gauss quadrature
    Ls, dE, nm = 4000, 2.2, 200
    model = L.chain(Ls, energy_scale=dE)
    o = oracle_mod.Oracle(model)
    phi = L.random_phase_vectors(Ls, 1, config=96)
    o.set_state(phi)
    C = o.dos_moments(nm)
    Kq = 256
    nodes = np.cos(np.pi * (np.arange(Kq) + 0.5) / Kq)
    rho = o.kpm_transform(C, nodes * dE)[0]
    integral = np.sum(rho * np.sqrt(1 - nodes ** 2)) * np.pi / Kq * dE
    assert abs(integral - 2 * C[0, 0] / model.volume) < 1e-12
    # clean chain DOS = (2/Omega) N / (pi sqrt(4 gamma^2 - E^2)) away from the band edges (spin
    # factor 2).  phi = sqrt(N) e_0 gives the exact trace on a translation-invariant ring
    # (<0|T_n|0> = Tr T_n / N), so only the Jackson broadening (~ pi dE / N_m) remains.
    e0 = np.zeros((1, Ls, 2))
    e0[0, 0, 0] = np.sqrt(Ls)
    o.set_state(e0)
    C0 = o.dos_moments(nm)
    E = np.linspace(-1.2, 1.2, 25)
    rho = o.kpm_transform(C0, E)[0]
    ref = 2.0 / (np.pi * np.sqrt(4 - E ** 2))
    assert np.max(np.abs(rho - ref) / ref) < 2e-3
    # a single moment set: transform of C = delta_{n,0} is the n=0 term alone
    one = np.zeros((1, 5))
    one[0, 0] = 3.0
    out = o.kpm_transform(one, np.array([0.3]))[0, 0]
    e = 0.3 / dE
    assert abs(out - 2 * 3.0 / (np.pi * model.volume * dE * np.sqrt(1 - e * e))) < 1e-15
    # and of C = delta_{n,2}: g_2 * 2 * T_2(e)
    one[:] = 0
    one[0, 2] = 1.0
    out = o.kpm_transform(one, np.array([0.3]))[0, 0]
    g = oracle_mod.jackson(5)
    assert abs(out - 2 / (np.pi * model.volume * dE * np.sqrt(1 - e * e)) * g[2] * 2 * (2 * e * e - 1)) < 1e-15


def test_other_damping_kernels(oracle_mod):
    """Lorentz and undamped kernels (the paper's ref. [33]) pinned by what they DO, not by
    their formula: (i) any kernel's damped moment g_k C_k is recovered exactly by the Chebyshev-Gauss
    projection of the transformed density, which ties the transform to oracle_damping term by term and
    fixes g_0 = 1 (norm conservation); (ii) the undamped series reproduces a polynomial density exactly;
    (iii) the Lorentz kernel turns a single level delta(x - a) into the Lorentzian
    (1/pi) eps / ((x - a)^2 + eps^2) with eps = lambda / N_m -- its defining property."""
    model = L.chain(16, energy_scale=1.0)             # dE = 1 and Omega = 16: out = 2 / (16 pi sqrt(1 - x^2)) sum ...
    o = oracle_mod.Oracle(model)
    rng_ = np.random.default_rng(11)
    nm, Kq = 40, 128
    nodes = np.cos(np.pi * (np.arange(Kq) + 0.5) / Kq)
    C = rng_.standard_normal((1, nm))
    for kind, lam in ((0, 0.0), (1, 3.5), (2, 0.0)):
        g = oracle_mod.damping(kind, lam, nm)
        rho = o.kpm_transform(C, nodes, damping=kind, lam=lam)[0]
        for k in (0, 1, 7, nm - 1):
            proj = np.sum(rho * np.cos(k * np.arccos(nodes)) * np.sqrt(1 - nodes ** 2)) * np.pi / Kq
            assert abs(proj - 2.0 / model.volume * g[k] * C[0, k]) < 1e-13        # int rho T_k dE = (2 / Omega) g_k C_k
        assert g[0] == 1.0 and np.all(g <= 1.0) and np.all(g >= 0.0)
    assert np.all(oracle_mod.damping(2, 0.0, nm) == 1.0)
    assert np.array_equal(oracle_mod.damping(0, 0.0, nm), oracle_mod.jackson(nm))
    gl = oracle_mod.damping(1, 4.0, 1000)
    assert np.all(np.diff(gl) < 0) and abs(gl[500] - np.sinh(2.0) / np.sinh(4.0)) < 1e-15
    with pytest.raises(RuntimeError):
        oracle_mod.damping(1, 0.0, 8)
    # (ii) density (1 + x) / (pi sqrt(1 - x^2)): moments mu_0 = 1, mu_1 = 1/2, the rest 0
    mu = np.zeros((1, 12))
    mu[0, 0], mu[0, 1] = 1.0, 0.5
    x = np.linspace(-0.9, 0.9, 7)
    rho = o.kpm_transform(mu, x, damping=2)[0] * model.volume / 2.0
    assert np.allclose(rho, (1 + x) / (np.pi * np.sqrt(1 - x ** 2)), rtol=1e-14)
    # (iii) one level at a: mu_n = T_n(a); Lorentz kernel -> half width eps = lambda / N_m in arccos x, i.e.
    # eps sqrt(1 - a^2) in x; the kernel is exp(-lambda n / N_m) up to O(exp(-lambda)) corrections
    a_, nm = 0.3, 4000
    mu = np.cos(np.arange(nm) * np.arccos(a_))[None]
    for lam, tol in ((4.0, 0.05), (6.0, 0.01)):
        eps = lam / nm
        w = eps * np.sqrt(1 - a_ ** 2)
        x = a_ + w * np.array([-3.0, -1.0, -0.3, 0.0, 0.5, 2.0])
        rho = o.kpm_transform(mu, x, damping=1, lam=lam)[0] * model.volume / 2.0
        lorentz = w / (np.pi * ((x - a_) ** 2 + w ** 2))
        assert np.max(np.abs(rho - lorentz) / lorentz) < tol
    # while Jackson gives a Gaussian-like peak of width pi / N_m: much lower tails at 3 eps
    jack = o.kpm_transform(mu, x, damping=0)[0] * model.volume / 2.0
    assert jack[0] < 0.2 * rho[0]


def test_transform_rejects_energy_outside_band(oracle_mod):
    model = L.chain(8)
    o = oracle_mod.Oracle(model)
    with pytest.raises(RuntimeError):
        o.kpm_transform(np.ones((1, 4)), np.array([model.energy_scale * 1.01]))


# ------------------------------------------------------------------ running conductivity (Eq. 2, 5, 7-11)
def test_running_conductivity_closed_forms(oracle_mod):
    """oracle_running_conductivity against closed forms: ballistic (plane wave: rho C_vv = c constant,
    rho dX^2 = c t^2, PAPER.md 8(c) of SURVEY) and the diffusive regime of the paper's own Eq. 7-10
    (C_vv = v^2 exp(-t/tau))."""
    dt = np.array([0.1, 0.2, 0.3, 0.5, 1.0, 1.0, 2.0])                    # non-uniform steps [A18]
    t = np.concatenate([[0.0], np.cumsum(dt)])
    c = np.array([3.0, 0.25])
    # ballistic VAC: the trapezoid rule is exact for a constant: sigma(t_k) = c t_k
    sig, _ = oracle_mod.running_conductivity("vac", np.tile(c, (t.size, 1)), None, dt)
    assert np.allclose(sig, np.outer(t, c), rtol=0, atol=1e-14)
    # ballistic MSD: (c t_k^2 - c t_{k-1}^2) / (2 dt_k) = c (t_k + t_{k-1}) / 2: the value at mid-step
    dos = np.array([0.5, 2.0])
    msd = np.outer(t[1:] ** 2, c)
    sig, length = oracle_mod.running_conductivity("msd", msd, dos, dt)
    assert np.allclose(sig, np.outer(0.5 * (t[1:] + t[:-1]), c), rtol=1e-14, atol=0)
    assert np.allclose(length, 2.0 * np.outer(t[1:], np.sqrt(c / dos)), rtol=1e-14)     # Eq. 11
    # diffusive regime (Eq. 7): rho C_vv = rho v^2 exp(-t/tau)
    rho, v2, tau = 0.7, 4.0, 1.5
    dtf = np.full(600, 0.02)
    tf = np.concatenate([[0.0], np.cumsum(dtf)])
    sig, _ = oracle_mod.running_conductivity("vac", (rho * v2 * np.exp(-tf / tau))[:, None], None, dtf)
    exact = rho * v2 * tau * (1.0 - np.exp(-tf / tau))
    assert np.max(np.abs(sig[:, 0] - exact)) <= 2e-5 * exact[-1]         # trapezoid error ~ dt^2 / (12 tau^2)
    assert abs(sig[-1, 0] / (rho * v2 * tau) - 1.0) < 1e-3               # -> sigma_sc = rho v^2 tau   (Eq. 8)
    # the same physics through the MSD: rho dX^2 = 2 rho v^2 tau (t - tau (1 - exp(-t/tau)))  (d/2dt = sigma)
    x2 = 2.0 * rho * v2 * tau * (tf[1:] - tau * (1.0 - np.exp(-tf[1:] / tau)))
    sig_m, length = oracle_mod.running_conductivity("msd", x2[:, None], np.array([rho]), dtf)
    mid = 0.5 * (tf[1:] + tf[:-1])
    assert np.max(np.abs(sig_m[:, 0] - rho * v2 * tau * (1.0 - np.exp(-mid / tau)))) <= 2e-5 * exact[-1]
    assert abs(x2[-1] / rho / (2.0 * tf[-1]) / (v2 * tau) - 1.0) < 0.15  # Einstein relation (Eq. 10), t = 8 tau
    assert np.allclose(length[:, 0], 2.0 * np.sqrt(x2 / rho))
    # sigma^VAC and sigma^MSD are the same function of time: compare at the mid-steps
    sig_v_mid = 0.5 * (sig[1:, 0] + sig[:-1, 0])
    assert np.max(np.abs(sig_v_mid - sig_m[:, 0])) <= 1e-4 * exact[-1]


def test_localization_length_pins(oracle_mod):
    """oracle_localization_length (Eq. 12, reading A27) against hand values, an exact plateau and a saturating series."""
    # hand values: L_last = (2 pi, 8 pi), L_prev = (2 pi, 4 pi)  ->  xi = (1, 4), growth = (0, 1/2)
    xi, gr = oracle_mod.localization_length(np.array([[2 * np.pi, 4 * np.pi], [2 * np.pi, 8 * np.pi]]))
    assert np.allclose(xi, [1.0, 4.0], rtol=1e-15) and np.array_equal(gr, [0.0, 0.5])
    # an exact plateau gives xi exactly and zero growth, whatever came before it
    L0 = np.array([0.3, 17.0, 1e-9])
    series = np.vstack([np.linspace(0, 1, 9)[:, None] * L0[None, :], L0[None, :], L0[None, :]])
    xi, gr = oracle_mod.localization_length(series)
    assert np.array_equal(xi, L0 / (2.0 * np.pi)) and np.array_equal(gr, np.zeros(3))
    # a saturating length L(t) = Linf (1 - exp(-t/tau)): xi -> Linf / 2 pi from below, growth -> 0 as exp(-t/tau) dt/tau
    t = np.arange(1, 41) * 0.5
    Linf, tau = 12.0, 2.0
    xi, gr = oracle_mod.localization_length((Linf * (1.0 - np.exp(-t / tau)))[:, None])
    assert 0.0 < Linf / (2 * np.pi) - xi[0] < 1e-4 * Linf
    assert 0.0 < gr[0] < 1.5e-5
    # a length that still grows linearly (ballistic) is flagged by its growth = dt / t_last
    xi, gr = oracle_mod.localization_length((2.0 * t)[:, None])
    assert np.isclose(gr[0], 0.5 / t[-1], rtol=1e-12) and np.isclose(xi[0], 2.0 * t[-1] / (2 * np.pi), rtol=1e-15)
    # degenerate rows: a single time (nothing known about saturation), a vanishing length
    xi, gr = oracle_mod.localization_length(np.array([[5.0, 0.0]]))
    assert np.allclose(xi, [5.0 / (2 * np.pi), 0.0]) and np.array_equal(gr, [1.0, 0.0])


def test_running_conductivity_on_a_lattice(oracle_mod):
    """The two routes to sigma(E, t) agree on a clean periodic chain with a plane-wave state, where both
    correlation functions are known exactly: rho C_vv = rho v_k^2, rho dX^2 = rho v_k^2 t^2."""
    Lc, kq = 64, 5
    model = L.chain(Lc, energy_scale=2.5)
    k = 2 * np.pi * kq / Lc
    phi = np.stack([np.cos(k * model.x), np.sin(k * model.x)], axis=1)[None]
    o = oracle_mod.Oracle(model, batch=1, modes=oracle_mod.MODE_VAC | oracle_mod.MODE_MSD)
    o.set_state(phi)
    nm, dts = 64, [0.5, 0.5, 1.0]
    E = np.array([-2.0 * np.cos(k)])                                      # eps_k for hopping -1
    dos = o.kpm_transform(o.dos_moments(nm), E)[0]
    vac_rows, msd_rows = [], []
    for dt in dts:
        vac_rows.append(o.kpm_transform(o.vac(nm), E)[0])
        o.evolve(dt, 40)
        msd_rows.append(o.kpm_transform(o.msd(nm), E)[0])
    vac_rows.append(o.kpm_transform(o.vac(nm), E)[0])
    sv, _ = oracle_mod.running_conductivity("vac", np.array(vac_rows), dos, np.array(dts))
    sm, length = oracle_mod.running_conductivity("msd", np.array(msd_rows), dos, np.array(dts))
    vk2 = (2.0 * np.sin(k)) ** 2
    t = np.concatenate([[0.0], np.cumsum(dts)])
    assert np.allclose(sv[:, 0], dos[0] * vk2 * t, rtol=1e-9)
    assert np.allclose(sm[:, 0], dos[0] * vk2 * 0.5 * (t[1:] + t[:-1]), rtol=1e-9)
    assert np.allclose(length[:, 0], 2.0 * np.sqrt(vk2) * t[1:], rtol=1e-9)
