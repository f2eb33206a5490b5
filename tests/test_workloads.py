"""Invariants of the seeded input generators."""
import numpy as np

from tests import dense_ref as D
from workloads import lattices as L
from workloads import rng


def test_splitmix64_reference_values():
    # splitmix64 with state0 = 0: first outputs of the published reference implementation
    z = rng.splitmix64(0, 3)
    assert [int(v) for v in z] == [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]
    u = rng.uniform01(12345, 1000)
    assert 0.0 <= u.min() and u.max() < 1.0 and abs(u.mean() - 0.5) < 0.05
    assert np.array_equal(rng.splitmix64(7, 10)[4:], rng.splitmix64(7, 6, offset=4))


def test_graphene_geometry():
    idx, xy, Lx, Ly = L.graphene_geometry(6, 4)
    N = idx.shape[0]
    d = xy[idx] - xy[:, None, :]
    d[..., 0] -= Lx * np.round(d[..., 0] / Lx)
    d[..., 1] -= Ly * np.round(d[..., 1] / Ly)
    assert np.allclose(np.hypot(d[..., 0], d[..., 1]), L.A_CC, atol=1e-12)      # all bonds = a_cc
    A = np.zeros((N, N), int)
    for m in range(N):
        A[m, idx[m]] += 1
    assert np.array_equal(A, A.T) and A.max() == 1


def test_vacancies():
    m0 = L.graphene(10, 8)
    m = L.graphene(10, 8, vacancy_fraction=0.05, vacancy_seed=3)
    assert m.N == m0.N - int(np.floor(0.05 * m0.N))
    H = D.dense_H(m)
    assert np.array_equal(H, H.T)
    assert np.all(np.diff(m.x.reshape(-1)) > -1e9)
    hist = np.bincount(m.nbr_count, minlength=4)
    assert hist[3] > hist[2] > 0


def test_peierls_hermitian_and_flux():
    """H_nm = conj(H_mn) bit-exactly, and the phase around EVERY plaquette (seam included) is
    2 pi phi mod 2 pi."""
    Lx, Ly, q = 7, 6, 2
    m = L.square_peierls(Lx, Ly, flux_quanta=q)
    H = D.dense_H(m)
    assert np.array_equal(H, H.conj().T)
    phi = q / (Lx * Ly)
    for x in range(Lx):
        for y in range(Ly):
            a = x + Lx * y
            b = (x + 1) % Lx + Lx * y
            c = (x + 1) % Lx + Lx * ((y + 1) % Ly)
            d = x + Lx * ((y + 1) % Ly)
            # counter-clockwise loop a -> b -> c -> d -> a; hop n -> m is H[m, n]
            loop = H[b, a] * H[c, b] * H[d, c] * H[a, d]
            ang = np.angle(loop) / (2 * np.pi)
            assert abs(((ang - phi + 0.5) % 1.0) - 0.5) < 1e-12 or abs(((ang + phi + 0.5) % 1.0) - 0.5) < 1e-12
    # all plaquettes carry the SAME flux sign
    signs = []
    for x in range(Lx):
        for y in range(Ly):
            a, b = x + Lx * y, (x + 1) % Lx + Lx * y
            c, d = (x + 1) % Lx + Lx * ((y + 1) % Ly), x + Lx * ((y + 1) % Ly)
            signs.append(np.sign(np.angle(H[b, a] * H[c, b] * H[d, c] * H[a, d])))
    assert len(set(signs)) == 1


def test_graphene_peierls_hexagon_flux_and_potential():
    ncx, ncy = 13, 8          # >= 3 cell-list bins of 5 xi = 10 A per side
    m = L.graphene_peierls_correlated(ncx, ncy, flux_per_hexagon=0.02, centre_density=0.05)
    H = D.dense_H(m)
    assert np.array_equal(H - np.diag(np.diag(H)), (H - np.diag(np.diag(H))).conj().T)
    phi = m.meta["phi"]

    def site(cx, cy, s):
        return 4 * ((cx % ncx) + ncx * (cy % ncy)) + s
    angs = []
    for cx in range(ncx):
        for cy in range(ncy):
            hexes = [
                [site(cx + 1, cy, 0), site(cx + 1, cy, 1), site(cx + 1, cy, 2), site(cx + 1, cy, 3),
                 site(cx, cy, 2), site(cx, cy, 1)],
                [site(cx, cy, 2), site(cx + 1, cy, 3), site(cx + 1, cy + 1, 0), site(cx, cy + 1, 1),
                 site(cx, cy + 1, 0), site(cx, cy, 3)],
            ]
            for hx in hexes:
                loop = 1.0 + 0j
                for i in range(6):
                    n_, m_ = hx[i], hx[(i + 1) % 6]
                    assert H[m_, n_] != 0
                    loop *= H[m_, n_] / 2.7
                angs.append(np.angle(loop) / (2 * np.pi))
    angs = np.array(angs)
    assert np.allclose(np.abs(angs), phi, atol=1e-10) and len(set(np.sign(angs))) == 1
    # potential: brute-force Gaussian sum on this small sheet
    xy = m.meta["xy"]
    Lx, Ly = m.box_length, m.meta["Ly"]
    n_c = m.meta["n_centres"]
    u = rng.uniform01(rng.stream_seed(5, 2, 0), n_c)
    perm = np.arange(m.N)
    for j in range(n_c):
        r = j + int(u[j] * (m.N - j))
        perm[j], perm[r] = perm[r], perm[j]
    eps = 2 * rng.uniform01(rng.stream_seed(5, 2, 1), n_c) - 1
    U = np.zeros(m.N)
    for k in range(n_c):
        d = xy - xy[perm[k]]
        d[:, 0] -= Lx * np.round(d[:, 0] / Lx)
        d[:, 1] -= Ly * np.round(d[:, 1] / Ly)
        r2 = np.sum(d * d, axis=1)
        U += np.where(r2 <= 100.0, eps[k] * np.exp(-r2 / 8.0), 0.0)
    assert np.allclose(m.onsite, U, atol=1e-13)


def test_random_phase_vectors():
    v = L.random_phase_vectors(1000, 3, config=4)
    assert np.allclose(np.sum(v * v, axis=2), 1.0, atol=1e-15)
    assert not np.array_equal(v[0], v[1])
    assert np.array_equal(v[1], L.random_phase_vectors(1000, 1, config=4, first_vector=1)[0])


def test_bond_disorder_is_hermitian_and_not_constant():
    from paper_1705_01387_b200 import binding
    base = L.graphene(7, 5, vacancy_fraction=0.1, vacancy_seed=2)
    m = L.with_bond_disorder(base, 0.4, 7)
    assert binding.validate(m) == 0                                   # bit-exact Hermiticity, Gershgorin
    h = m.hop_re.reshape(m.N, m.K)
    valid = np.arange(m.K)[None, :] < m.nbr_count[:, None]
    assert np.unique(h[valid]).size > 10
    assert np.all(np.abs(h[valid] / -2.7 - 1.0) <= 0.2 + 1e-12)
    assert np.all(h[~valid] == 0.0)


def test_random_graph_generator_is_hermitian_and_reproducible():
    """workloads.random_graph (fuzz input of tests/test_gpu_fuzz.py): degrees within K, no self or double bonds,
    H_nm = conj(H_mn) bit for bit, the stated Gershgorin margin, same seed -> same arrays."""
    for cplx in (False, True):
        m = L.random_graph(300, 6, 41, complex_hops=cplx, degree_fill=0.8, locality=20)
        again = L.random_graph(300, 6, 41, complex_hops=cplx, degree_fill=0.8, locality=20)
        assert m.nbr_index.tobytes() == again.nbr_index.tobytes() and m.hop_re.tobytes() == again.hop_re.tobytes()
        idx = m.nbr_index.reshape(m.N, m.K)
        assert m.nbr_count.max() <= m.K and m.nbr_count.min() >= 0
        g = np.zeros(m.N)
        for i in range(m.N):
            row = idx[i, :m.nbr_count[i]]
            assert len(set(row)) == len(row) and i not in row and np.all(idx[i, m.nbr_count[i]:] == -1)
            for k, j in enumerate(row):
                back = list(idx[j, :m.nbr_count[j]]).index(i)
                assert m.hop_re[i * m.K + k] == m.hop_re[j * m.K + back]
                if cplx:
                    assert m.hop_im[i * m.K + k] == -m.hop_im[j * m.K + back]
                g[i] += np.hypot(m.hop_re[i * m.K + k], m.hop_im[i * m.K + k] if cplx else 0.0)
        assert np.max(g + np.abs(m.onsite)) < m.energy_scale
        assert (m.hop_im is not None) == cplx
