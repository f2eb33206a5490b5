"""Dense exact-diagonalisation reference used to PIN the oracle (tiny lattices only).

Built directly from the TBModel input arrays with numpy complex128 — it shares nothing with
oracle/ or the CUDA library.  Definitions: PAPER.md Eq. 32 (H), Eq. 33 (X), Eq. 34 (V),
U(t) = exp(-iHt) (hbar = 1), T_n by cos(n arccos(lambda)) on the eigenvalues.
"""
import numpy as np


def to_c(v):
    """[..., 2] float64 (re, im) -> complex128"""
    return v[..., 0] + 1j * v[..., 1]


def from_c(z):
    return np.stack([z.real, z.imag], axis=-1)


def dense_H(model):
    N, K = model.N, model.K
    H = np.zeros((N, N), dtype=np.complex128)
    idx = model.nbr_index.reshape(N, K)
    for m in range(N):
        for k in range(model.nbr_count[m]):
            h = -1.0 if model.hop_re is None else model.hop_re[m * K + k]
            if model.hop_im is not None:
                h = h + 1j * model.hop_im[m * K + k]
            H[m, idx[m, k]] += h
        if model.onsite is not None:
            H[m, m] += model.onsite[m]
    return H


def dense_V(model, H=None):
    """V_mn = i (X_n - X_m) H_mn with the minimum-image difference (Eq. 34)."""
    H = dense_H(model) if H is None else H
    x = model.x
    d = x[None, :] - x[:, None]                 # d[m, n] = X_n - X_m
    if model.box_length > 0:
        d = d - model.box_length * np.round(d / model.box_length)
    return 1j * d * H


def dense_U(H, t):
    w, Q = np.linalg.eigh(H)
    return (Q * np.exp(-1j * w * t)) @ Q.conj().T


def dense_Tn(H, dE, n):
    w, Q = np.linalg.eigh(H / dE)
    assert np.max(np.abs(w)) < 1.0
    return (Q * np.cos(n * np.arccos(w))) @ Q.conj().T
