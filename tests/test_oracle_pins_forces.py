"""Pins of the oracle's SURVEY.md 8(f) functions (CPU only): batch statistics, logarithmic
derivatives and the force vector.

PF1 O_k = d log psi / d theta_k against central finite differences of the independent
    dense_reference.psi_all (plain product, no logarithm inside)          Eq. 8
PF2 with exact weights p(s) over the full basis, 2 Re F_k / 2 Im F_k are the derivatives of
    E(theta) = <psi|H|psi>/<psi|psi> along Re / Im theta_k; E from the dense Kronecker H
                                                                          Eq. 6-7, :77-89; Eq. 16
PF3 mean / variance against numpy.average, and Eq. 3: sum_s p(s) E_loc(s) = <H>   :56-61, :70-73
PF4 eigenstate => variance 0 and F = 0 (E_loc constant, connected correlation vanishes)  :604
PF5 invariances of the connected correlation: E_loc -> E_loc + const leaves F unchanged;
    F is linear in E_loc; uniform weights == no weights
"""
import numpy as np
import pytest

import workloads as wl
from dense_reference import all_states, dense_hamiltonian, psi_all


def _hermitian_workload(N, M, sigma, seed):
    """Random RBM + a Hermitian H (real coefficients on Pauli strings are Hermitian)."""
    w = wl.make_random(N, M, 1 << N, 3 * N, sigma, seed)
    coeffs = w.ham.coeffs.real.astype(np.complex64)
    return w, coeffs


def _unpack(theta, N, M):
    return theta[:N], theta[N:N + M], theta[N + M:].reshape(M, N)


def _pack(a, b, W):
    return np.concatenate([np.asarray(a).ravel(), np.asarray(b).ravel(), np.asarray(W).ravel()]).astype(np.complex128)


# ----------------------------------------------------------------------------- PF1
@pytest.mark.parametrize("N,M,sigma,seed", [(4, 3, 0.3, 21), (5, 6, 0.2, 22)])
def test_pf1_log_derivatives_vs_finite_differences(oracle, N, M, sigma, seed):
    w = wl.make_random(N, M, 1 << N, 4, sigma, seed)
    O = oracle.log_derivatives(w.spins, w.a, w.b, w.W)
    theta = _pack(w.a, w.b, w.W)
    K = theta.size
    assert O.shape == (1 << N, K)
    assert np.array_equal(w.spins.astype(np.float64), all_states(N))
    h = 1e-6
    for k in range(K):
        for direction in (1.0, 1j):  # holomorphic: the derivative is the same along Re and Im
            tp, tm = theta.copy(), theta.copy()
            tp[k] += h * direction
            tm[k] -= h * direction
            fd = (np.log(psi_all(N, *_unpack(tp, N, M))) - np.log(psi_all(N, *_unpack(tm, N, M)))) / (2 * h * direction)
            assert np.max(np.abs(fd - O[:, k])) < 1e-8, (k, direction)


# ----------------------------------------------------------------------------- PF2
@pytest.mark.parametrize("N,M,sigma,seed", [(4, 3, 0.3, 31), (6, 4, 0.2, 32)])
def test_pf2_forces_are_the_energy_gradient(oracle, N, M, sigma, seed):
    w, coeffs = _hermitian_workload(N, M, sigma, seed)
    H = dense_hamiltonian(N, w.ham.sites, w.ham.paulis, coeffs)
    assert np.allclose(H, H.conj().T)

    def energy(theta):
        psi = psi_all(N, *_unpack(theta, N, M))
        return (psi.conj() @ H @ psi).real / (psi.conj() @ psi).real

    theta = _pack(w.a, w.b, w.W)
    psi = psi_all(N, w.a, w.b, w.W)
    p = np.abs(psi) ** 2
    e_loc, _ = oracle.local_energy_definition(w.spins, w.a, w.b, w.W, w.ham.sites, w.ham.paulis, coeffs)
    F = oracle.forces(w.spins, w.a, w.b, w.W, e_loc, weights=p)
    h = 1e-6
    for k in range(theta.size):
        for direction, part in ((1.0, F[k].real), (1j, F[k].imag)):
            tp, tm = theta.copy(), theta.copy()
            tp[k] += h * direction
            tm[k] -= h * direction
            fd = (energy(tp) - energy(tm)) / (2 * h)
            assert abs(fd - 2 * part) < 2e-7 * max(1.0, abs(fd)), (k, direction, fd, 2 * part)


# ----------------------------------------------------------------------------- PF3
def test_pf3_mean_variance_vs_numpy_and_eq3(oracle):
    rng = np.random.default_rng(41)
    x = rng.normal(size=1000) + 1j * rng.normal(size=1000)
    wgt = rng.random(1000)
    m, v, sw = oracle.mean_variance(x)
    assert abs(m - x.mean()) < 1e-13 and abs(v - np.var(x)) < 1e-13 and sw == 1000
    m, v, sw = oracle.mean_variance(x, wgt)
    mu = np.average(x, weights=wgt)
    assert abs(m - mu) < 1e-13 and abs(v - np.average(np.abs(x - mu) ** 2, weights=wgt)) < 1e-13
    assert abs(sw - wgt.sum()) < 1e-10
    # Eq. 3: the p-weighted mean of E_loc over the full basis is <H>; its variance is <H^2> - <H>^2
    N, M = 6, 5
    w, coeffs = _hermitian_workload(N, M, 0.25, 42)
    H = dense_hamiltonian(N, w.ham.sites, w.ham.paulis, coeffs)
    psi = psi_all(N, w.a, w.b, w.W)
    e_loc, _ = oracle.local_energy_fast(w.spins, w.a, w.b, w.W, w.ham.sites, w.ham.paulis, coeffs)
    m, v, _ = oracle.mean_variance(e_loc, np.abs(psi) ** 2)
    nrm = (psi.conj() @ psi).real
    eh = (psi.conj() @ H @ psi) / nrm
    eh2 = (psi.conj() @ H @ H @ psi).real / nrm
    assert abs(m - eh) < 1e-11 and abs(v - (eh2 - abs(eh) ** 2)) < 1e-10


# ----------------------------------------------------------------------------- PF4
def test_pf4_eigenstate_has_zero_variance_and_zero_force(oracle):
    """W = b = 0, a_i in {0, i pi/2}: a product of |+> / |-> states, eigenstate of -h sum X."""
    N, M = 6, 3
    a = np.array([0, 0.5j * np.pi, 0, 0, 0.5j * np.pi, 0.5j * np.pi], dtype=np.complex64)
    b = np.zeros(M, dtype=np.complex64)
    W = np.zeros((M, N), dtype=np.complex64)
    sites = np.array([[i, -1] for i in range(N)], dtype=np.int32)
    paulis = np.array([[1, 0]] * N, dtype=np.uint8)
    coeffs = np.full(N, -0.7, dtype=np.complex64)
    spins = all_states(N).astype(np.int8)
    e_loc, _ = oracle.local_energy_definition(spins, a, b, W, sites, paulis, coeffs)
    m, v, _ = oracle.mean_variance(e_loc)
    assert v < 1e-12 and abs(m - 0.7 * (3 - 3)) < 1e-6  # float32 pi/2: cos is 4e-8, not 0
    F = oracle.forces(spins, a, b, W, e_loc)
    assert np.max(np.abs(F)) < 1e-6


# ----------------------------------------------------------------------------- PF5
def test_pf5_connected_correlation_invariances(oracle):
    w = wl.make_random(9, 5, 300, 10, 0.3, 51)
    rng = np.random.default_rng(52)
    e1 = rng.normal(size=300) + 1j * rng.normal(size=300)
    e2 = rng.normal(size=300) + 1j * rng.normal(size=300)
    F1 = oracle.forces(w.spins, w.a, w.b, w.W, e1)
    F2 = oracle.forces(w.spins, w.a, w.b, w.W, e2)
    assert np.max(np.abs(oracle.forces(w.spins, w.a, w.b, w.W, e1 + (3.0 - 2.0j)) - F1)) < 1e-12
    assert np.max(np.abs(oracle.forces(w.spins, w.a, w.b, w.W, 2 * e1 - 1j * e2) - (2 * F1 - 1j * F2))) < 1e-12
    assert np.max(np.abs(oracle.forces(w.spins, w.a, w.b, w.W, e1, weights=np.full(300, 0.37)) - F1)) < 1e-12
    # the a-part is a plain covariance with the spins: F_{a_i} = <<s_i E>> - <<s_i>><<E>>
    s = w.spins.astype(np.float64)
    cov = (s * e1[:, None]).mean(0) - s.mean(0) * e1.mean()
    assert np.max(np.abs(F1[:9] - cov)) < 1e-12
