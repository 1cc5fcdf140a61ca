"""Dense-matrix helpers for the oracle pins (numpy only; independent of oracle/ and of the CUDA path).

H of Eq. (1) is assembled from Kronecker products of cyclic shift matrices and
Pauli matrices -- a different construction from the oracle's neighbour loops."""
import numpy as np

SIGMA = np.array([[[0, 1], [1, 0]], [[0, -1j], [1j, 0]], [[1, 0], [0, -1]]], dtype=np.complex128)


def dense_H(L, t, JH, S):
    P = np.roll(np.eye(L), 1, axis=0)          # cyclic shift
    A1 = P + P.T                               # ring adjacency (L = 2 gives weight 2: counted twice)
    I = np.eye(L)
    A = np.kron(np.kron(I, I), A1) + np.kron(np.kron(I, A1), I) + np.kron(np.kron(A1, I), I)
    H = -t * np.kron(A, np.eye(2)).astype(np.complex128)
    N = L ** 3
    for i in range(N):
        H[2 * i:2 * i + 2, 2 * i:2 * i + 2] += JH * np.einsum("c,cab->ab", S[i], SIGMA)
    return H


def cheb_T(n, x):
    """T_n(x) for real x in [-1,1] (array) by the defining cosine formula, Eq. (23) PAPER.md:155."""
    return np.cos(n * np.arccos(np.clip(x, -1.0, 1.0)))


def spinors(S):
    """chi_i = (cos(th/2) e^{-i ph/2}, sin(th/2) e^{+i ph/2}): the spin-1/2 state along S_i in the gauge in which
    chi_i^dagger chi_j reproduces Eq. (3) -- half-angle algebra, not the oracle's cos/sin formula."""
    S = np.asarray(S, dtype=np.float64)
    ph = np.arctan2(S[:, 1], S[:, 0])
    c = np.sqrt(np.clip((1.0 + S[:, 2]) / 2.0, 0.0, 1.0))
    s = np.sqrt(np.clip((1.0 - S[:, 2]) / 2.0, 0.0, 1.0))
    return np.stack([c * np.exp(-0.5j * ph), s * np.exp(0.5j * ph)], axis=1)


def dense_H_dex(L, t, S):
    """Eq. (2)-(3): <i|H|j> = -t chi_i^dagger chi_j on nearest-neighbour bonds of the periodic cubic
    lattice (adjacency from Kronecker products of cyclic shifts)."""
    P = np.roll(np.eye(L), 1, axis=0)
    A1 = P + P.T
    I = np.eye(L)
    A = np.kron(np.kron(I, I), A1) + np.kron(np.kron(I, A1), I) + np.kron(np.kron(A1, I), I)
    chi = spinors(S)
    return -t * A * (chi.conj() @ chi.T)
