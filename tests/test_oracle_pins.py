"""Pins of the float64 oracle against what the paper and the mathematics fix (CPU only).

P1  brute force: dense H (Kronecker products) psi / psi, N <= 10        Eq. 4
P2  sum_s p(s) E_loc(s) = <psi|H|psi>/<psi|psi>                          Eq. 2-3, :56-61
P3  zero parameters => psi == 1 => E_loc = diagonal + sum of elements   closed form
P4  product eigenstate => E_loc constant (variance 0)                   :604
P5  singlet dimer: E_loc = -3 for XX+YY+ZZ                              textbook
P6  global spin-flip symmetry at a = b = 0                              BASELINE.json north_star
P7  1-D TFIM ring ground energy (Pfeuty) pins the dense-H builder       :588, ref [66]
P8  definition mode <-> fast mode
P9  log cosh: real-argument library routine, exp(F1) = cosh, F1 = definition mod 2 pi i
P11 Eq. 39 data (connected configurations + elements) against the dense matrix rows
"""
import json
import os

import numpy as np
import pytest

import workloads as wl
from dense_reference import all_states, dense_hamiltonian, local_energy_all, psi_all

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _wrap(d):
    return (d + np.pi) % (2 * np.pi) - np.pi


def _assert_close(x, ref, rtol, what):
    err = np.abs(np.asarray(x) - np.asarray(ref))
    tol = rtol * np.maximum(1.0, np.abs(ref))
    assert np.all(err <= tol), f"{what}: max err {err.max():.3e} (tol {tol.min():.3e})"


def _assert_logpsi(lp, psi_ref, rtol, what):
    """exp(log psi) must be psi; equivalently log psi agrees mod 2 pi i."""
    ref = np.log(psi_ref)
    assert np.all(np.abs(lp.real - ref.real) <= rtol * np.maximum(1, np.abs(ref))), what
    assert np.all(np.abs(_wrap(lp.imag - ref.imag)) <= rtol * np.maximum(1, np.abs(ref))), what


# ----------------------------------------------------------------------------- P1
@pytest.mark.parametrize("N,M,T,sigma,seed", [(4, 3, 12, 0.4, 11), (6, 9, 30, 0.3, 12), (8, 5, 40, 0.25, 13),
                                               (10, 12, 60, 0.15, 14)])
def test_p1_bruteforce_random_terms(oracle, N, M, T, sigma, seed):
    w = wl.make_random(N, M, 1 << N, T, sigma, seed)
    assert w.spins.shape == (1 << N, N)
    e_ref, psi, _ = local_energy_all(N, w.a, w.b, w.W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    for fn in (oracle.local_energy_definition, oracle.local_energy_fast):
        e, lp = fn(w.spins, w.a, w.b, w.W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
        _assert_close(e, e_ref, 1e-10, f"E_loc {fn.__name__}")
        _assert_logpsi(lp, psi, 1e-11, f"log psi {fn.__name__}")


@pytest.mark.parametrize("N,M,T,K,sigma,seed,max_flips", [
    (5, 4, 30, 3, 0.3, 15, 4), (7, 6, 40, 4, 0.25, 16, 4), (8, 5, 50, 6, 0.2, 17, 4), (9, 7, 25, 8, 0.15, 18, 4),
    # flip sets of up to K sites: beyond what the CUDA path accepts (four), so that the oracle is already pinned there
    (8, 5, 50, 6, 0.2, 17, 6), (9, 7, 40, 8, 0.15, 18, 8), (8, 4, 60, 8, 0.2, 21, 8)])
def test_p1_bruteforce_k_site_pauli_strings(oracle, N, M, T, K, sigma, seed, max_flips):
    """k-site Pauli strings ("tensor products of branch-free operators"): term
    arrays [T,K] with up to K operators per term, up to `max_flips` of them flipping, against the dense Kronecker-product
    H (which knows no flip / sign rule).  Several Y factors in one string pin the (-i)^n phase; strings with the same
    flip set pin the grouping of fast mode.  The generator's limit on flipping factors is lifted to K in the last
    cases (a shared generator must not be shaped by the kernel's limits)."""
    w = wl.make_random(N, M, 1 << N, 4, sigma, seed)
    ham = wl.random_strings(N, T, K, np.random.default_rng([seed, 3]), max_flips=max_flips)
    assert ham.sites.shape == (T, K)
    n_flips = ((ham.paulis == 1) | (ham.paulis == 2)).sum(axis=1)
    assert n_flips.max() <= max_flips and (max_flips <= 4 or n_flips.max() > 4), n_flips.max()
    e_ref, psi, H = local_energy_all(N, w.a, w.b, w.W, ham.sites, ham.paulis, ham.coeffs)
    assert np.abs(H).max() > 0
    for fn in (oracle.local_energy_definition, oracle.local_energy_fast):
        e, lp = fn(w.spins, w.a, w.b, w.W, ham.sites, ham.paulis, ham.coeffs)
        _assert_close(e, e_ref, 1e-10, f"E_loc {fn.__name__} K={K}")
        _assert_logpsi(lp, psi, 1e-11, f"log psi {fn.__name__} K={K}")
    # Eq. 39 as data: every term's (s', element) is an entry of the dense matrix row
    sp, mel = oracle.connected(w.spins[:8], ham.sites, ham.paulis, ham.coeffs)
    states = all_states(N)
    index = {tuple(row): k for k, row in enumerate(states)}
    for bidx in range(8):
        row = np.zeros(1 << N, np.complex128)
        for t in range(T):
            row[index[tuple(sp[bidx, t].astype(np.float64))]] += mel[bidx, t]
        assert np.allclose(row, H[index[tuple(w.spins[bidx].astype(np.float64))]], atol=1e-12)


def test_p1_three_and_four_site_strings_by_hand(oracle):
    """XXX, YYY, XYZ, ZZZZ and XZZX on a 5-site chain with fixed coefficients: a term list a reader can check."""
    N, M = 5, 3
    w = wl.make_random(N, M, 1 << N, 1, 0.3, 19)
    X, Y, Z = 1, 2, 3
    sites = np.array([[0, 1, 2, -1], [1, 2, 3, -1], [0, 2, 4, -1], [0, 1, 2, 3], [1, 2, 3, 4]], np.int32)
    paulis = np.array([[X, X, X, 0], [Y, Y, Y, 0], [X, Y, Z, 0], [Z, Z, Z, Z], [X, Z, Z, X]], np.uint8)
    coeffs = np.array([0.5, -0.25 + 0.5j, 1.5, -1.0, 0.75j], np.complex64)
    e_ref, _, _ = local_energy_all(N, w.a, w.b, w.W, sites, paulis, coeffs)
    for fn in (oracle.local_energy_definition, oracle.local_energy_fast):
        e, _ = fn(w.spins, w.a, w.b, w.W, sites, paulis, coeffs)
        _assert_close(e, e_ref, 1e-11, fn.__name__)


@pytest.mark.parametrize("pauli", [1, 2, 3])
def test_p1_single_pauli_terms(oracle, pauli):
    """One single-site Pauli with a complex coefficient: a column-convention or sigma^y sign
    mistake changes the sign of exactly these."""
    N, M = 5, 4
    w = wl.make_random(N, M, 1 << N, 1, 0.3, 21)
    sites = np.array([[2, -1]], np.int32)
    paulis = np.array([[pauli, 0]], np.uint8)
    coeffs = np.array([0.7 - 0.2j], np.complex64)
    e_ref, _, _ = local_energy_all(N, w.a, w.b, w.W, sites, paulis, coeffs)
    e, _ = oracle.local_energy_definition(w.spins, w.a, w.b, w.W, sites, paulis, coeffs)
    _assert_close(e, e_ref, 1e-11, "single Pauli")


def test_p1_config1_against_dense(oracle):
    w = wl.make_config(1)
    e_ref, psi, _ = local_energy_all(w.N, w.a, w.b, w.W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    e, lp = oracle.local_energy_definition(w.spins, w.a, w.b, w.W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    _assert_close(e, e_ref, 1e-12, "c1 E_loc")
    _assert_logpsi(lp, psi, 1e-12, "c1 log psi")
    _assert_logpsi(oracle.log_psi(w.spins, w.a, w.b, w.W, stable=True), psi, 1e-12, "c1 log psi F1")


def test_basis_state_order_matches_dense():
    N = 5
    assert np.array_equal(wl.basis_states(N).astype(np.float64), all_states(N))


# ----------------------------------------------------------------------------- P2
def test_p2_weighted_average_is_rayleigh_quotient(oracle):
    w = wl.make_config(1)
    H = dense_hamiltonian(w.N, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    assert np.allclose(H, H.conj().T)
    psi = psi_all(w.N, w.a, w.b, w.W)
    rayleigh = (psi.conj() @ H @ psi) / (psi.conj() @ psi)
    e, lp = oracle.local_energy_fast(w.spins, w.a, w.b, w.W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    p = np.exp(2 * lp.real)
    avg = np.sum(p * e) / np.sum(p)
    assert abs(avg - rayleigh) < 1e-12 * abs(rayleigh)
    assert abs(avg.imag) < 1e-12  # Hermitian H: real expectation value


# ----------------------------------------------------------------------------- P3
@pytest.mark.parametrize("k", [2, 5])
def test_p3_zero_parameters_closed_form(oracle, k):
    w = wl.make_config(k, B=8)
    a0, b0, W0 = np.zeros_like(w.a), np.zeros_like(w.b), np.zeros_like(w.W)
    spec = wl.config_spec(k)
    bonds = wl.chain_bonds(w.N) if spec["lattice"] == "chain" else wl.square_bonds(spec["L"])
    s = w.spins.astype(np.float64)
    zz = sum(s[:, i] * s[:, j] for i, j in bonds)
    expect = -spec["J"] * zz - spec["h"] * w.N
    for fn in (oracle.local_energy_definition, oracle.local_energy_fast):
        e, lp = fn(w.spins, a0, b0, W0, w.ham.sites, w.ham.paulis, w.ham.coeffs)
        assert np.allclose(e, expect, rtol=0, atol=1e-12)
        assert np.allclose(lp, 0, atol=1e-15)


def test_p3_heisenberg_zero_parameters(oracle):
    w = wl.make_config(4, B=16)
    a0, b0, W0 = np.zeros_like(w.a), np.zeros_like(w.b), np.zeros_like(w.W)
    s = w.spins.astype(np.float64)
    bonds = wl.square_bonds(10)
    # diag sum s_i s_k, off-diagonal element 1 - s_i s_k (reading Q9)
    expect = sum(s[:, i] * s[:, j] + (1 - s[:, i] * s[:, j]) for i, j in bonds)
    e, _ = oracle.local_energy_fast(w.spins, a0, b0, W0, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    assert np.allclose(e, expect, atol=1e-12)
    assert np.all(w.spins.sum(axis=1) == 0)  # zero magnetisation


# ----------------------------------------------------------------------------- P4
def test_p4_product_eigenstate_constant_local_energy(oracle):
    """W = b = 0, a_i in {0, i pi/2}: psi(s) = prod_i (1 or i^{s_i}) is a product of |+> / |->
    states; H = -h sum X has eigenvalue h (n_minus - n_plus) and E_loc is that for every s."""
    N, M, h = 7, 3, 1.3
    rng = np.random.default_rng(4)
    minus = rng.integers(0, 2, N).astype(bool)
    a = np.where(minus, 0.5j * np.pi, 0).astype(np.complex128)  # float64 on purpose: exact pi/2
    sites = np.array([[i, -1] for i in range(N)], np.int32)
    paulis = np.array([[1, 0]] * N, np.uint8)
    coeffs = np.full(N, -h, np.complex64)
    spins = wl.basis_states(N)
    # complex64 parameter bytes round pi/2: tolerance reflects that rounding only
    e, _ = oracle.local_energy_definition(spins, a.astype(np.complex64), np.zeros(M, np.complex64),
                                          np.zeros((M, N), np.complex64), sites, paulis, coeffs)
    expect = float(np.float32(h)) * (minus.sum() - (~minus).sum())
    assert np.allclose(e, expect, atol=2e-6)
    assert np.std(e) < 2e-6


# ----------------------------------------------------------------------------- P5
def test_p5_singlet(oracle):
    q = 0.25j * np.pi
    a = np.array([q, -q], np.complex64)
    b = np.zeros(1, np.complex64)
    W = np.array([[q, q]], np.complex64)
    ham = wl.heisenberg([(0, 1)])
    spins = np.array([[1, -1], [-1, 1], [1, 1]], np.int8)
    psi = psi_all(2, a, b, W)  # order: ++, +-, -+, --
    assert abs(psi[1] - 1j) < 1e-6 and abs(psi[2] + 1j) < 1e-6 and abs(psi[0]) < 1e-6 and abs(psi[3]) < 1e-6
    for fn in (oracle.local_energy_definition, oracle.local_energy_fast):
        e, _ = fn(spins, a, b, W, ham.sites, ham.paulis, ham.coeffs)
        assert np.allclose(e[:2], -3.0, atol=1e-6)
        assert np.allclose(e[2], 1.0, atol=1e-6)  # triplet component: XX and YY elements cancel


# ----------------------------------------------------------------------------- P6
def test_p6_spin_flip_symmetry(oracle):
    w = wl.make_config(2, B=64, sigma=0.2)
    a0, b0 = np.zeros_like(w.a), np.zeros_like(w.b)
    args = (a0, b0, w.W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    e1, l1 = oracle.local_energy_fast(w.spins, *args)
    e2, l2 = oracle.local_energy_fast(-w.spins, *args)
    assert np.allclose(e1, e2, rtol=0, atol=1e-12)
    assert np.allclose(l1, l2, rtol=0, atol=1e-13)
    # and the symmetry is genuinely broken by a visible bias (the test has teeth)
    e3, _ = oracle.local_energy_fast(-w.spins, w.a, b0, w.W, *args[3:])
    e4, _ = oracle.local_energy_fast(w.spins, w.a, b0, w.W, *args[3:])
    assert not np.allclose(e3, e4, atol=1e-6)


# ----------------------------------------------------------------------------- P7
def test_p7_pfeuty_ground_energy_pins_dense_builder():
    with open(os.path.join(GOLDEN, "tfim_ring_ground_energy.json")) as f:
        gold = json.load(f)
    for case in gold["cases"]:
        N, h = case["N"], case["h"]
        ham = wl.tfim(wl.chain_bonds(N), N, 1.0, h)
        H = dense_hamiltonian(N, ham.sites, ham.paulis, ham.coeffs)
        e0 = np.linalg.eigvalsh(H)[0]
        m = np.arange(N)
        closed = -np.sum(np.sqrt(1 + h * h - 2 * h * np.cos((2 * m + 1) * np.pi / N)))
        assert abs(e0 - closed) < 1e-10
        assert abs(e0 - case["E0"]) < 1e-9


# ----------------------------------------------------------------------------- P8
@pytest.mark.parametrize("k,nsub", [(1, None), (2, 2048), (3, 48), (4, 48), (5, 12)])
def test_p8_definition_vs_fast(oracle, k, nsub):
    w = wl.make_config(k, B=nsub) if k != 1 else wl.make_config(1)
    args = (w.spins, w.a, w.b, w.W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    e_d, l_d = oracle.local_energy_definition(*args)
    e_f, l_f = oracle.local_energy_fast(*args)
    _assert_close(e_f, e_d, 1e-10, f"c{k} E_loc fast vs definition")
    assert np.all(np.abs(l_f.real - l_d.real) <= 1e-12 * np.maximum(1, np.abs(l_d)))
    assert np.all(np.abs(_wrap(l_f.imag - l_d.imag)) <= 1e-12 * np.maximum(1, np.abs(l_d)))


def test_p8_definition_vs_fast_large_parameters(oracle):
    """sigma = 0.3 at config-3 shapes: |theta| up to ~12, |Im theta| passes pi/2 (branch Q6)."""
    w = wl.make_robustness(0.3, B=16)
    args = (w.spins, w.a, w.b, w.W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    e_d, l_d = oracle.local_energy_definition(*args)
    e_f, l_f = oracle.local_energy_fast(*args)
    _assert_close(e_f, e_d, 1e-9, "P10 shapes")
    assert np.all(np.abs(l_f.real - l_d.real) <= 1e-11 * np.maximum(1, np.abs(l_d)))
    assert np.all(np.abs(_wrap(l_f.imag - l_d.imag)) <= 1e-9)


# ----------------------------------------------------------------------------- P9
def test_p9_lncosh_real_argument_is_logaddexp(oracle):
    x = np.concatenate([np.linspace(-30, 30, 601), [0.0, 1e-9, -1e-9, 700.0, -700.0]])
    ref = np.logaddexp(x, -x) - np.log(2.0)
    for stable in (False, True):
        if not stable:
            xs, rs = x[np.abs(x) < 600], ref[np.abs(x) < 600]  # cosh overflows in the definition
        else:
            xs, rs = x, ref
        got = oracle.lncosh(xs.astype(np.complex128), stable)
        assert np.allclose(got.real, rs, rtol=1e-14, atol=1e-16)
        assert np.allclose(got.imag, 0, atol=1e-16)


def test_p9_lncosh_complex(oracle):
    rng = np.random.default_rng(9)
    z = rng.standard_normal(4000) * 3 + 1j * rng.standard_normal(4000) * 3
    f1 = oracle.lncosh(z, True)
    d = oracle.lncosh(z, False)
    assert np.allclose(np.exp(f1), np.cosh(z), rtol=1e-13)
    assert np.allclose(f1.real, d.real, rtol=1e-12, atol=1e-13)
    assert np.allclose(_wrap(f1.imag - d.imag), 0, atol=1e-12)
    small = np.abs(z.imag) < np.pi / 2
    assert np.allclose(f1.imag[small], d.imag[small], atol=1e-12)  # principal value there (Q6)
    # Taylor: log cosh z = z^2/2 - z^4/12 + z^6/45 - ...  for small |z|
    zs = (rng.standard_normal(100) + 1j * rng.standard_normal(100)) * 0.01
    series = zs**2 / 2 - zs**4 / 12 + zs**6 / 45 - 17 * zs**8 / 2520
    for stable in (True, False):  # absolute error of either form is a few ulp of ln 2
        assert np.allclose(oracle.lncosh(zs, stable), series, rtol=0, atol=5e-16)


# ----------------------------------------------------------------------------- P11
def test_p11_connected_data_against_dense_rows(oracle):
    N = 6
    w = wl.make_random(N, 4, 1 << N, 25, 0.2, 31)
    sp, mel = oracle.connected(w.spins, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    weights = 1 << (N - 1 - np.arange(N))
    for t in range(w.ham.T):
        Ht = dense_hamiltonian(N, w.ham.sites[t:t + 1], w.ham.paulis[t:t + 1], w.ham.coeffs[t:t + 1])
        kprime = ((1 - sp[:, t, :].astype(np.int64)) // 2) @ weights
        rows = np.arange(1 << N)
        assert np.allclose(Ht[rows, kprime], mel[:, t], atol=1e-12)
        # branch-free: that is the only non-zero of the row
        Hz = Ht.copy()
        Hz[rows, kprime] = 0
        assert np.allclose(Hz, 0)
