"""Brute-force pin P1: exact dense H psi / psi over all 2^N basis states (N <= 12).

Independent of oracle/ by construction: the Hamiltonian is assembled from Kronecker products
of the 2x2 Pauli matrices (no flip / matrix-element rules), and psi is evaluated as
exp(sum a_i s_i) * prod_j cosh(theta_j) (no logarithm).  Conventions it fixes:
  * site 0 is the leftmost Kronecker factor; basis index k <-> s_i = +1 iff bit (N-1-i) of
    k is 0; +1 == "up" == first basis vector (1,0)^T  (readings Q2, Q3 of DESIGN.md);
  * E_loc(s) = sum_s' <s|H|s'> psi(s') / psi(s) = (H psi)[s] / psi[s]   (Eq. 4).
"""
from __future__ import annotations

import numpy as np

PAULI = {
    0: np.array([[1, 0], [0, 1]], dtype=np.complex128),
    1: np.array([[0, 1], [1, 0]], dtype=np.complex128),
    2: np.array([[0, -1j], [1j, 0]], dtype=np.complex128),
    3: np.array([[1, 0], [0, -1]], dtype=np.complex128),
}


def dense_hamiltonian(N: int, sites, paulis, coeffs) -> np.ndarray:
    assert N <= 12
    dim = 1 << N
    H = np.zeros((dim, dim), dtype=np.complex128)
    for srow, prow, c in zip(np.asarray(sites), np.asarray(paulis), np.asarray(coeffs)):  # [T,K]: K slots per term
        factors = [PAULI[0]] * N
        for site, p in zip((int(v) for v in srow), (int(v) for v in prow)):
            if site >= 0:
                assert factors[site] is PAULI[0], "two operators on one site"
                factors[site] = PAULI[p]
        term = np.array([[1.0 + 0j]])
        for f in factors:
            term = np.kron(term, f)
        H += complex(c) * term
    return H


def all_states(N: int) -> np.ndarray:
    k = np.arange(1 << N)[:, None]
    bits = (k >> (N - 1 - np.arange(N))[None, :]) & 1
    return (1 - 2 * bits).astype(np.float64)


def psi_all(N: int, a, b, W) -> np.ndarray:
    """psi(s) for every basis state, as a plain product (no log): Eq. 38 exponentiated."""
    s = all_states(N)
    a = np.asarray(a, dtype=np.complex128)
    b = np.asarray(b, dtype=np.complex128)
    W = np.asarray(W, dtype=np.complex128)
    theta = s @ W.T + b[None, :]
    return np.exp(s @ a) * np.prod(np.cosh(theta), axis=1)


def local_energy_all(N: int, a, b, W, sites, paulis, coeffs):
    H = dense_hamiltonian(N, sites, paulis, coeffs)
    psi = psi_all(N, a, b, W)
    return (H @ psi) / psi, psi, H
