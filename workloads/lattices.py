"""Seeded synthetic tight-binding inputs shaped like the paper's workloads.

Everything here is *input generation* (neighbour lists, hoppings, on-site
potentials, positions, random phases) in the form of the paper's four data sets
(PAPER.md:240 and §4.2.1-4.2.4).  No arithmetic of the method (SpMV, Chebyshev,
KPM) lives here; the CUDA library and the oracle both receive these arrays.

Site / neighbour ordering is the bit-exact contract of SURVEY.md §8(d).
"""
from dataclasses import dataclass, field
from typing import Optional

import numpy as np

from . import rng

A_CC = 1.42  # graphene C-C distance, Angstrom


@dataclass
class TBModel:
    """The paper's four input data sets as flat arrays."""
    name: str
    N: int
    K: int                               # K_max, line 1 of neighbor.in
    nbr_count: np.ndarray                # int32 [N]
    nbr_index: np.ndarray                # int32 [N*K] row-major, 0-based; unused slots = -1
    hop_re: Optional[np.ndarray]         # float64 [N*K] or None => all -1
    hop_im: Optional[np.ndarray]         # float64 [N*K] or None => real
    onsite: Optional[np.ndarray]         # float64 [N] or None => 0
    x: np.ndarray                        # float64 [N] transport-direction coordinate
    box_length: float                    # <= 0 => open boundary in x
    volume: float
    energy_scale: float                  # Delta E
    meta: dict = field(default_factory=dict)


def _pack(name, count, index, hop_re, hop_im, onsite, x, box, vol, dE, meta=None):
    N, K = index.shape
    return TBModel(name=name, N=int(N), K=int(K),
                   nbr_count=np.ascontiguousarray(count, dtype=np.int32),
                   nbr_index=np.ascontiguousarray(index.reshape(-1), dtype=np.int32),
                   hop_re=None if hop_re is None else np.ascontiguousarray(hop_re.reshape(-1), dtype=np.float64),
                   hop_im=None if hop_im is None else np.ascontiguousarray(hop_im.reshape(-1), dtype=np.float64),
                   onsite=None if onsite is None else np.ascontiguousarray(onsite, dtype=np.float64),
                   x=np.ascontiguousarray(x, dtype=np.float64),
                   box_length=float(box), volume=float(vol), energy_scale=float(dE),
                   meta=meta or {})


def anderson_onsite(N: int, W: float, seed: int) -> np.ndarray:
    """U_m uniform in [-W/2, W/2] (Eq. 35)."""
    return (rng.uniform01(seed, N) - 0.5) * W


def random_phase_vectors(N: int, batch: int, config: int, first_vector: int = 0) -> np.ndarray:
    """phi_i = exp(i theta_i), theta ~ U[0, 2 pi)  ->  float64 [batch][N][2] (re, im).

    <phi|phi> = N.  Stream 3 of the config, one sub-stream per vector.
    """
    out = np.empty((batch, N, 2), dtype=np.float64)
    for b in range(batch):
        theta = 2.0 * np.pi * rng.uniform01(rng.stream_seed(config, 3, first_vector + b), N)
        out[b, :, 0] = np.cos(theta)
        out[b, :, 1] = np.sin(theta)
    return out


def with_bond_disorder(model: TBModel, delta: float, seed: int) -> TBModel:
    """Real, bond-dependent hoppings h_mn = h0 * (1 + delta * (u_mn - 1/2)), u_mn = u_nm a counter-based
    uniform of the unordered pair (min, max) -- symmetric bit for bit, so H stays Hermitian.  Exercises
    the per-entry real-hopping storage (the paper's hopping.in with distinct values)."""
    assert model.hop_im is None
    N, K = model.N, model.K
    idx = model.nbr_index.reshape(N, K).astype(np.int64)
    rows = np.repeat(np.arange(N, dtype=np.int64)[:, None], K, axis=1)
    valid = np.arange(K)[None, :] < model.nbr_count[:, None]
    lo, hi = np.minimum(rows, idx), np.maximum(rows, idx)
    pair = np.where(valid, lo * N + hi, 0).reshape(-1)
    with np.errstate(over="ignore"):
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + rng._GAMMA * (pair.astype(np.uint64) + np.uint64(1))
        z = (z ^ (z >> np.uint64(30))) * rng._M1
        z = (z ^ (z >> np.uint64(27))) * rng._M2
        z = z ^ (z >> np.uint64(31))
    u = (z >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)
    h0 = model.hop_re if model.hop_re is not None else np.full(N * K, -1.0)
    hre = np.where(valid.reshape(-1), h0 * (1.0 + delta * (u - 0.5)), 0.0)
    return TBModel(name=model.name + "_bonddis", N=N, K=K, nbr_count=model.nbr_count, nbr_index=model.nbr_index,
                   hop_re=np.ascontiguousarray(hre), hop_im=None, onsite=model.onsite, x=model.x,
                   box_length=model.box_length, volume=model.volume,
                   energy_scale=model.energy_scale * (1.0 + abs(delta) / 2.0), meta=dict(model.meta))


# --------------------------------------------------------------------------- hypercubic lattices
def chain(L: int, W: float = 0.0, seed: int = 0, periodic: bool = True, hop: float = -1.0,
          energy_scale: Optional[float] = None, explicit_hop: bool = False) -> TBModel:
    """1-D chain, neighbours [-x, +x] (paper example E2)."""
    i = np.arange(L, dtype=np.int64)
    if periodic:
        idx = np.stack([(i - 1) % L, (i + 1) % L], axis=1)
        cnt = np.full(L, 2, dtype=np.int32)
    else:
        idx = np.full((L, 2), -1, dtype=np.int64)
        cnt = np.zeros(L, dtype=np.int32)
        left = i > 0
        right = i < L - 1
        # compact the present neighbours to the front, order [-x, +x]
        idx[left, 0] = i[left] - 1
        cnt[left] += 1
        pos = cnt.copy()
        idx[right, pos[right]] = i[right] + 1
        cnt[right] += 1
    hre = None
    if hop != -1.0 or explicit_hop:
        hre = np.where(idx >= 0, hop, 0.0)
    onsite = anderson_onsite(L, W, seed) if W > 0 else None
    dE = energy_scale if energy_scale is not None else 2 * abs(hop) + W / 2 + 0.1
    return _pack(f"chain{L}", cnt, idx, hre, None, onsite, i.astype(np.float64),
                 L if periodic else 0.0, float(L), dE)


def square(Lx: int, Ly: int, W: float = 0.0, seed: int = 0, periodic: bool = True,
           energy_scale: Optional[float] = None) -> TBModel:
    """2-D square lattice, i = x + Lx*y, neighbours [-x, +x, -y, +y], hoppings -1 (default)."""
    i = np.arange(Lx * Ly, dtype=np.int64)
    xx, yy = i % Lx, i // Lx
    if periodic:
        idx = np.stack([(xx - 1) % Lx + Lx * yy, (xx + 1) % Lx + Lx * yy,
                        xx + Lx * ((yy - 1) % Ly), xx + Lx * ((yy + 1) % Ly)], axis=1)
        cnt = np.full(Lx * Ly, 4, dtype=np.int32)
        hre = None
    else:
        cand = [(xx - 1, yy), (xx + 1, yy), (xx, yy - 1), (xx, yy + 1)]
        idx = np.full((Lx * Ly, 4), -1, dtype=np.int64)
        cnt = np.zeros(Lx * Ly, dtype=np.int32)
        for cx, cy in cand:
            ok = (cx >= 0) & (cx < Lx) & (cy >= 0) & (cy < Ly)
            idx[i[ok], cnt[ok]] = (cx + Lx * cy)[ok]
            cnt[ok] += 1
        hre = None
    onsite = anderson_onsite(Lx * Ly, W, seed) if W > 0 else None
    dE = energy_scale if energy_scale is not None else 4 + W / 2 + 0.1
    return _pack(f"square{Lx}x{Ly}", cnt, idx, hre, None, onsite, xx.astype(np.float64),
                 Lx if periodic else 0.0, float(Lx * Ly), dE)


def cubic(L: int, W: float = 0.0, seed: int = 0, energy_scale: Optional[float] = None) -> TBModel:
    """3-D simple cubic, periodic, i = x + L*(y + L*z), neighbours [-x,+x,-y,+y,-z,+z]."""
    i = np.arange(L ** 3, dtype=np.int64)
    xx, yy, zz = i % L, (i // L) % L, i // (L * L)

    def at(a, b, c):
        return a + L * (b + L * c)
    idx = np.stack([at((xx - 1) % L, yy, zz), at((xx + 1) % L, yy, zz),
                    at(xx, (yy - 1) % L, zz), at(xx, (yy + 1) % L, zz),
                    at(xx, yy, (zz - 1) % L), at(xx, yy, (zz + 1) % L)], axis=1)
    cnt = np.full(L ** 3, 6, dtype=np.int32)
    onsite = anderson_onsite(L ** 3, W, seed) if W > 0 else None
    dE = energy_scale if energy_scale is not None else 6 + W / 2 + 0.1
    return _pack(f"cubic{L}", cnt, idx, None, None, onsite, xx.astype(np.float64),
                 float(L), float(L ** 3), dE)


# --------------------------------------------------------------------------- graphene
_BASIS = np.array([[0.0, 0.0], [np.sqrt(3.0) / 2, 0.5], [np.sqrt(3.0) / 2, 1.5], [0.0, 2.0]])  # units of a_cc
# (neighbour sublattice, cell offset dx, cell offset dy) in the contract order of SURVEY.md 8(d)
_GNBR = {
    0: [(1, 0, 0), (1, -1, 0), (3, 0, -1)],
    1: [(0, 0, 0), (0, 1, 0), (2, 0, 0)],
    2: [(1, 0, 0), (3, 0, 0), (3, 1, 0)],
    3: [(2, 0, 0), (2, -1, 0), (0, 0, 1)],
}


def graphene_geometry(ncx: int, ncy: int):
    """Returns (idx [N,3] int64, xy [N,2] Angstrom, Lx, Ly) of the periodic 4-atom-cell sheet."""
    N = 4 * ncx * ncy
    i = np.arange(N, dtype=np.int64)
    s = i % 4
    c = i // 4
    cx, cy = c % ncx, c // ncx
    idx = np.empty((N, 3), dtype=np.int64)
    for sub in range(4):
        m = s == sub
        for k, (ns, ox, oy) in enumerate(_GNBR[sub]):
            idx[m, k] = 4 * (((cx[m] + ox) % ncx) + ncx * ((cy[m] + oy) % ncy)) + ns
    ax, ay = np.sqrt(3.0) * A_CC, 3.0 * A_CC
    xy = np.empty((N, 2), dtype=np.float64)
    xy[:, 0] = cx * ax + _BASIS[s, 0] * A_CC
    xy[:, 1] = cy * ay + _BASIS[s, 1] * A_CC
    return idx, xy, ncx * ax, ncy * ay


def graphene(ncx: int, ncy: int, hop: float = -2.7, W: float = 0.0, seed: int = 0,
             vacancy_fraction: float = 0.0, vacancy_seed: int = 0,
             energy_scale: float = 10.0) -> TBModel:
    """Periodic graphene sheet (rectangular 4-atom cells), real hopping, optional Anderson
    disorder U[-W/2, W/2] and optional vacancies (sites removed uniformly at random by a partial
    Fisher-Yates shuffle, indices compacted preserving order, neighbour lists rebuilt)."""
    idx, xy, Lx, Ly = graphene_geometry(ncx, ncy)
    N0 = idx.shape[0]
    cnt = np.full(N0, 3, dtype=np.int32)
    meta = {"ncx": ncx, "ncy": ncy, "Ly": Ly}
    if vacancy_fraction > 0:
        nrem = int(np.floor(vacancy_fraction * N0))
        u = rng.uniform01(vacancy_seed, nrem)
        perm = np.arange(N0, dtype=np.int64)
        for j in range(nrem):                      # partial Fisher-Yates
            r = j + int(u[j] * (N0 - j))
            perm[j], perm[r] = perm[r], perm[j]
        removed = np.zeros(N0, dtype=bool)
        removed[perm[:nrem]] = True
        newid = np.cumsum(~removed) - 1
        keep = ~removed
        idx_k = idx[keep]
        alive = ~removed[idx_k]
        mapped = np.where(alive, newid[idx_k], -1)
        # compact alive neighbours to the front, preserving their order
        order = np.argsort(~alive, axis=1, kind="stable")
        mapped = np.take_along_axis(mapped, order, axis=1)
        cnt = alive.sum(axis=1).astype(np.int32)
        idx = mapped
        xy = xy[keep]
        meta["removed"] = nrem
    N = idx.shape[0]
    hre = np.where(idx >= 0, hop, 0.0)
    onsite = anderson_onsite(N, W, seed) if W > 0 else None
    return _pack(f"graphene{ncx}x{ncy}", cnt, idx, hre, None, onsite, xy[:, 0], Lx,
                 Lx * Ly, energy_scale, meta)


def peierls_hoppings(idx, xy, Lx, Ly, beta, hop_abs):
    """Complex hoppings H_mn = -hop_abs * exp(i theta_mn) for a uniform perpendicular field in the
    Landau gauge A = (-B y, 0); beta = flux quanta per unit area.  For the hop n -> m (stored in
    row m, column n = idx[m, k]) with (dx, dy) the minimum-image components of r_m - r_n and
    wrap = round(((y_m - y_n) - dy) / Ly):
        theta_mn = -2 pi beta [dx (y_n + dy/2) + Ly wrap x_m]
    (midpoint-rule line integral + magnetic-translation phase on bonds crossing the y seam;
    consistent when beta Lx Ly is an integer).  theta is evaluated once per bond, from its
    lower-index end, and negated for the reverse direction, so H_nm = conj(H_mn) bit-exactly
    (cos is even and sin is odd bit-exactly).  SURVEY.md 8(d) "Config 5 details"."""
    N = idx.shape[0]
    d = xy[idx] - xy[:, None, :]                        # r_n - r_m
    dx = -(d[..., 0] - Lx * np.round(d[..., 0] / Lx))   # min-image of r_m - r_n
    dy = -(d[..., 1] - Ly * np.round(d[..., 1] / Ly))
    y_n = xy[idx][..., 1]
    y_m = xy[:, None, 1]
    x_m = xy[:, None, 0]
    wrap = np.round(((y_m - y_n) - dy) / Ly)
    theta = -2.0 * np.pi * beta * (dx * (y_n + dy / 2.0) + Ly * wrap * x_m)
    m_idx = np.arange(N, dtype=np.int64)[:, None]
    lower = m_idx < idx
    back = np.argmax(idx[idx] == m_idx[:, :, None], axis=2)   # position of m in row n's list
    theta = np.where(lower, theta, -theta[idx, back])
    return -hop_abs * np.cos(theta), -hop_abs * np.sin(theta)


def square_peierls(Lx: int, Ly: int, flux_quanta: int = 1, W: float = 0.0, seed: int = 0,
                   energy_scale=None) -> TBModel:
    """Periodic square lattice with complex Peierls hoppings (|h| = 1), total flux = flux_quanta."""
    base = square(Lx, Ly, W=W, seed=seed, energy_scale=energy_scale)
    idx = base.nbr_index.reshape(-1, 4).astype(np.int64)
    i = np.arange(Lx * Ly)
    xy = np.stack([(i % Lx).astype(np.float64), (i // Lx).astype(np.float64)], axis=1)
    hre, him = peierls_hoppings(idx, xy, float(Lx), float(Ly), flux_quanta / (Lx * Ly), 1.0)
    base.hop_re = np.ascontiguousarray(hre.reshape(-1))
    base.hop_im = np.ascontiguousarray(him.reshape(-1))
    base.name = f"square_peierls{Lx}x{Ly}"
    base.meta = {"xy": xy, "flux_quanta": flux_quanta}
    return base


def graphene_peierls_correlated(ncx: int, ncy: int, config: int = 5, hop_abs: float = 2.7,
                                flux_per_hexagon: float = 1e-4, centre_density: float = 0.02,
                                xi: float = 2.0, energy_scale: Optional[float] = None) -> TBModel:
    """Config-5 style sheet: complex Peierls-phase hoppings for a uniform perpendicular field
    (Landau gauge A = (-B y, 0), flux rounded so the total flux is an integer number of quanta)
    plus a Gaussian-correlated on-site potential
        U_m = sum_k eps_k exp(-|r_m - R_k|^2 / (2 xi^2)),  eps_k ~ U[-1, 1] eV,
    centres at distinct random sites, minimum-image distances, cut off at 5 xi.
    Recipe: SURVEY.md 8(d) "Config 5 details"."""
    idx, xy, Lx, Ly = graphene_geometry(ncx, ncy)
    N = idx.shape[0]
    n_hex = N // 2
    quanta = max(1, int(round(flux_per_hexagon * n_hex)))
    phi = quanta / n_hex
    s_hex = 1.5 * np.sqrt(3.0) * A_CC ** 2
    beta = phi / s_hex
    hre, him = peierls_hoppings(idx, xy, Lx, Ly, beta, hop_abs)
    # correlated potential
    n_c = int(round(centre_density * N))
    u = rng.uniform01(rng.stream_seed(config, 2, 0), n_c)
    perm = np.arange(N, dtype=np.int64)
    for j in range(n_c):
        r = j + int(u[j] * (N - j))
        perm[j], perm[r] = perm[r], perm[j]
    centres = perm[:n_c]
    eps = 2.0 * rng.uniform01(rng.stream_seed(config, 2, 1), n_c) - 1.0
    onsite = _gaussian_potential(xy, Lx, Ly, centres, eps, xi)
    cnt = np.full(N, 3, dtype=np.int32)
    if energy_scale is None:
        G = float(np.max(np.abs(onsite)) + 3 * hop_abs)
        energy_scale = max(10.0, np.ceil(10.2 * G) / 10.0)
    return _pack(f"graphene_peierls{ncx}x{ncy}", cnt, idx, hre, him, onsite, xy[:, 0], Lx,
                 Lx * Ly, energy_scale,
                 {"ncx": ncx, "ncy": ncy, "Ly": Ly, "flux_quanta": quanta, "phi": phi,
                  "xy": xy, "n_centres": n_c})


def _gaussian_potential(xy, Lx, Ly, centres, eps, xi):
    """Cell-list accumulation of the Gaussian bumps, cut off at 5 xi, minimum image."""
    N = xy.shape[0]
    rc = 5.0 * xi
    nbx = max(1, int(np.floor(Lx / rc)))
    nby = max(1, int(np.floor(Ly / rc)))
    bx, by = Lx / nbx, Ly / nby
    if nbx < 3 or nby < 3:          # the 3x3 stencil would alias: small sheet, all pairs directly
        U = np.zeros(N, dtype=np.float64)
        for k in range(len(centres)):
            dxy = xy - xy[centres[k]]
            dxy[:, 0] -= Lx * np.round(dxy[:, 0] / Lx)
            dxy[:, 1] -= Ly * np.round(dxy[:, 1] / Ly)
            r2 = dxy[:, 0] ** 2 + dxy[:, 1] ** 2
            U += np.where(r2 <= rc * rc, eps[k] * np.exp(-r2 / (2.0 * xi * xi)), 0.0)
        return U
    cell = (np.minimum((xy[:, 0] / bx).astype(np.int64), nbx - 1)
            + nbx * np.minimum((xy[:, 1] / by).astype(np.int64), nby - 1))
    order = np.argsort(cell, kind="stable")
    start = np.searchsorted(cell[order], np.arange(nbx * nby + 1))
    U = np.zeros(N, dtype=np.float64)
    cxy = xy[centres]
    ccx = np.minimum((cxy[:, 0] / bx).astype(np.int64), nbx - 1)
    ccy = np.minimum((cxy[:, 1] / by).astype(np.int64), nby - 1)
    for ox, oy in [(a, b) for a in (-1, 0, 1) for b in (-1, 0, 1)]:
        tx = (ccx + ox) % nbx
        ty = (ccy + oy) % nby
        tc = tx + nbx * ty
        lo, hi = start[tc], start[tc + 1]
        nmax = int((hi - lo).max()) if len(lo) else 0
        for j in range(nmax):
            valid = (lo + j) < hi
            site = order[np.where(valid, lo + j, 0)]
            dxy = xy[site] - cxy
            dxy[:, 0] -= Lx * np.round(dxy[:, 0] / Lx)
            dxy[:, 1] -= Ly * np.round(dxy[:, 1] / Ly)
            r2 = dxy[:, 0] ** 2 + dxy[:, 1] ** 2
            ok = valid & (r2 <= rc * rc)
            np.add.at(U, site[ok], eps[ok] * np.exp(-r2[ok] / (2.0 * xi * xi)))
    return U


# --------------------------------------------------------------------------- random sparse Hermitian graphs
def random_graph(N: int, K: int, seed: int, complex_hops: bool = False, degree_fill: float = 0.7,
                 locality: int = 0, open_x: bool = True, hop_value: Optional[float] = None) -> TBModel:
    """A random sparse Hermitian tight-binding model for fuzzing the storage paths: every site proposes bonds to
    random partners (anywhere, or within `locality` rows), a bond is kept while both ends have fewer than K
    neighbours, hoppings are random (real, or complex with conj symmetry bit for bit), on-site energies random,
    positions random in a box (open boundary by default, so every X_n - X_m is unambiguous).  Rows with 0 .. K
    neighbours in random order; not a lattice the paper discusses, only an input the library must handle
    (PAPER.md:256 'the inputs are made as general as possible')."""
    u = rng.uniform01(seed, 4 * N * K + 4 * N + 8)
    nbrs = [[] for _ in range(N)]
    hops = {}
    pos = 0
    for m in range(N):
        for _ in range(K):
            r0, r1, r2, r3 = u[pos:pos + 4]
            pos += 4
            if r0 > degree_fill:
                continue
            n = int(r1 * N) if locality <= 0 else (m + 1 + int(r1 * locality)) % N
            if n == m or n in nbrs[m] or len(nbrs[m]) >= K or len(nbrs[n]) >= K:
                continue
            h = complex(-0.5 - r2, (r3 - 0.5) if complex_hops else 0.0)
            if hop_value is not None:              # one hopping value everywhere: the constant-hopping record variants
                h = complex(hop_value, 0.0)
            nbrs[m].append(n)
            nbrs[n].append(m)
            hops[(m, n)] = h
            hops[(n, m)] = h.conjugate()
    count = np.array([len(v) for v in nbrs], dtype=np.int32)
    index = np.full((N, K), -1, dtype=np.int32)
    hre = np.zeros((N, K))
    him = np.zeros((N, K))
    for m in range(N):
        for k, n in enumerate(nbrs[m]):
            index[m, k] = n
            hre[m, k] = hops[(m, n)].real
            him[m, k] = hops[(m, n)].imag
    tail = u[4 * N * K:]
    onsite = tail[:N] - 0.5
    x = np.cumsum(0.25 + tail[N:2 * N]) if locality > 0 else 100.0 * tail[N:2 * N]
    dE = 1.05 * float(np.max(np.abs(onsite) + np.sum(np.hypot(hre, him), axis=1))) + 0.1
    box = 0.0 if open_x else 4.0 * float(np.max(x) - np.min(x)) + 4.0     # a box so wide that no image is closer
    return _pack(f"random_N{N}_K{K}_s{seed}{'_c' if complex_hops else ''}", count, index,
                 None if hop_value == -1.0 else hre,                       # None = the paper's default, every hopping -1
                 him if (complex_hops and hop_value is None) else None, onsite, x, box, float(N), dE)
