"""Pins of oracle.fisher (the quantum Fisher matrix S, Eq. 10-11; CPU only).

PS1 dense-basis identity.  With exact weights p(s) = |psi(s)|^2 / <psi|psi> over the full basis,
        S_kk' = <d_k psi|d_k' psi>/<psi|psi> - <d_k psi|psi><psi|d_k' psi>/<psi|psi>^2
    where d_k psi comes from central finite differences of the INDEPENDENT dense psi (dense_reference.psi_all,
    a plain product with no logarithm and no derivative formula inside).  A conjugate on the wrong factor, a
    missing disconnected term, a transposed index or a wrong parameter order fails it.
PS2 S is Hermitian and positive semi-definite; its diagonal holds the variances of O_k (numpy.var).
PS3 library special case: with uniform weights S is numpy.cov of the log-derivatives (bias=True), transposed.
PS4 the connected correlation does not see a constant added to O, is quadratic under O -> c O, and uniform
    weights equal no weights.
"""
import numpy as np
import pytest

import workloads as wl
from dense_reference import all_states, psi_all


def _unpack(theta, N, M):
    return theta[:N], theta[N:N + M], theta[N + M:].reshape(M, N)


def _pack(a, b, W):
    return np.concatenate([np.asarray(a).ravel(), np.asarray(b).ravel(), np.asarray(W).ravel()]).astype(np.complex128)


@pytest.mark.parametrize("N,M,sigma,seed", [(3, 2, 0.4, 71), (4, 3, 0.3, 72), (5, 2, 0.25, 73)])
def test_ps1_dense_basis_identity(oracle, N, M, sigma, seed):
    w = wl.make_random(N, M, 1 << N, 4, sigma, seed)
    assert np.array_equal(w.spins.astype(np.float64), all_states(N))
    theta = _pack(w.a, w.b, w.W)
    K = theta.size
    psi = psi_all(N, w.a, w.b, w.W)
    Z = np.vdot(psi, psi).real
    h = 1e-6
    dpsi = np.empty((K, 1 << N), np.complex128)
    for k in range(K):
        tp, tm = theta.copy(), theta.copy()
        tp[k] += h
        tm[k] -= h
        dpsi[k] = (psi_all(N, *_unpack(tp, N, M)) - psi_all(N, *_unpack(tm, N, M))) / (2 * h)
    S_dense = dpsi.conj() @ dpsi.T / Z - np.outer((dpsi.conj() @ psi) / Z, (psi.conj() @ dpsi.T) / Z)
    S, Obar = oracle.fisher(w.spins, w.a, w.b, w.W, weights=np.abs(psi) ** 2)
    assert S.shape == (K, K)
    assert np.max(np.abs(S - S_dense)) < 1e-8 * max(1.0, np.abs(S_dense).max())
    assert np.max(np.abs(Obar - (psi.conj() @ dpsi.T) / Z)) < 1e-8


def test_ps2_hermitian_psd_diagonal(oracle):
    w = wl.make_random(7, 5, 300, 4, 0.3, 74)
    rng = np.random.default_rng(75)
    wts = rng.random(w.B)
    S, Obar = oracle.fisher(w.spins, w.a, w.b, w.W, weights=wts)
    assert np.max(np.abs(S - S.conj().T)) < 1e-14
    ev = np.linalg.eigvalsh(0.5 * (S + S.conj().T))
    assert ev.min() > -1e-12 * max(1.0, ev.max())
    O = oracle.log_derivatives(w.spins, w.a, w.b, w.W)
    p = wts / wts.sum()
    var = (p[:, None] * np.abs(O - (p[:, None] * O).sum(0)) ** 2).sum(0)
    assert np.allclose(np.diag(S).real, var, atol=1e-13) and np.max(np.abs(np.diag(S).imag)) < 1e-15


def test_ps3_numpy_cov(oracle):
    w = wl.make_random(6, 4, 200, 4, 0.3, 76)
    S, Obar = oracle.fisher(w.spins, w.a, w.b, w.W)
    O = oracle.log_derivatives(w.spins, w.a, w.b, w.W)
    cov = np.cov(O.T, bias=True)  # cov[i, j] = E[(x_i - m_i) conj(x_j - m_j)]
    assert np.max(np.abs(S - cov.T)) < 1e-13
    assert np.max(np.abs(Obar - O.mean(0))) < 1e-15


def test_ps4_invariances(oracle):
    rng = np.random.default_rng(77)
    O = rng.standard_normal((50, 9)) + 1j * rng.standard_normal((50, 9))
    wts = rng.random(50)
    S, Obar = oracle.fisher_from_derivatives(O, wts)
    shift = rng.standard_normal(9) + 1j * rng.standard_normal(9)
    S2, Obar2 = oracle.fisher_from_derivatives(O + shift[None, :], wts)
    assert np.max(np.abs(S - S2)) < 1e-12 and np.max(np.abs(Obar2 - Obar - shift)) < 1e-13
    c = 0.7 - 1.3j
    S3, _ = oracle.fisher_from_derivatives(c * O, wts)
    assert np.max(np.abs(S3 - abs(c) ** 2 * S)) < 1e-12
    S4, _ = oracle.fisher_from_derivatives(O, np.full(50, 3.7))
    S5, _ = oracle.fisher_from_derivatives(O, None)
    assert np.max(np.abs(S4 - S5)) < 1e-13
