"""small_eloc_kernel (csrc/nqs_small.cuh; SURVEY.md 7.1 "Small G"): steps a1 .. a6 in ONE launch for problems below the
size threshold of the tensor-core series path.  Parity against the float64 oracle through the C ABI: configs 1 and 2 at
full size, random term lists of every Pauli type, k-site strings, ragged batches (B not a multiple of any SB), the
robustness set's large parameters on a small shape (exponent renormalisation), the multi-launch path on the same inputs
(the two must agree within the tolerance of each against the oracle), and the rule that selects the kernel."""
import numpy as np
import pytest

import workloads as wl
from test_gpu_parity import check_eloc, check_logpsi, gpu_eloc, oracle_on, to_dev

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def nqs():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests need a B200")
    import paper_2108_03409_b200 as m

    m.load_library()
    yield m
    m.set_option("small_path", 0)
    m.set_option("a5_path", 0)


@pytest.fixture(scope="module")
def oracle():
    import oracle as o

    o.build()
    return o


def run(nqs, w, small=True):
    nqs.set_option("small_path", 0 if small else 1)
    try:
        e, l = gpu_eloc(nqs, w)
        took = nqs.debug_last_a5()
    finally:
        nqs.set_option("small_path", 0)
    return e, l, took


def test_config1_and_config2_take_the_single_launch(nqs, oracle):
    for k, mode in ((1, "definition"), (2, "fast")):
        w = wl.make_config(k)
        n0 = nqs.launch_count()
        e, l, took = run(nqs, w)
        assert took["path"] == "small", took
        assert nqs.launch_count() - n0 == 1, "one kernel for the whole call"
        e_ref, l_ref = oracle_on(oracle, w, slice(None), mode)
        check_eloc(e, e_ref, f"c{k} small")
        check_logpsi(l, l_ref, f"c{k} small")
        e2, l2, took2 = run(nqs, w, small=False)
        assert took2["path"] == "product", took2
        check_eloc(e2, e_ref, f"c{k} multi-launch")
    w = wl.make_config(2)
    idx = np.arange(0, w.B, 41)
    e, l, _ = run(nqs, w)
    e_def, l_def = oracle_on(oracle, w, idx, "definition")
    check_eloc(e[idx], e_def, "c2 small, definition mode")
    check_logpsi(l[idx], l_def, "c2 small, definition mode")


@pytest.mark.parametrize("B", [1, 3, 17, 129, 1000, 2111])
def test_ragged_batches(nqs, oracle, B):
    w = wl.make_config(2, B=B)
    e, l, took = run(nqs, w)
    assert took["path"] == "small"
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "fast")
    check_eloc(e, e_ref, f"c2 B={B}")
    check_logpsi(l, l_ref, f"c2 B={B}")


def test_random_terms_of_every_pauli_type(nqs, oracle):
    """Random 1- and 2-site terms (X, Y, Z, identity slots, complex coefficients, several terms per flip set, pair
    flips with both relative signs) against DEFINITION mode."""
    rng = np.random.default_rng(77)
    seen_small = 0
    for case in range(16):
        N = int(rng.integers(2, 40))
        M = int(rng.integers(1, 48))
        B = int(rng.integers(1, 400))
        T = int(rng.integers(1, 4 * N))
        sigma = float(rng.choice([0.02, 0.1, 0.25]))
        w = wl.make_random(N, M, B, T, sigma, 5000 + case)
        e, l, took = run(nqs, w)
        seen_small += took["path"] == "small"
        e_ref, l_ref = oracle_on(oracle, w, slice(None), "definition")
        what = f"case {case}: N={N} M={M} B={w.B} T={T} sigma={sigma} path={took['path']}"
        check_eloc(e, e_ref, what)
        check_logpsi(l, l_ref, what)
    assert seen_small >= 12


def test_large_parameters_exponent_renormalisation(nqs, oracle):
    """sigma = 0.5 on a shape with M = 120 hidden units: single factors of the product reach e^{+-4}, the running
    product leaves the float32 range without the renormalisation.  Relative tolerance 1e-3 as for the robustness set
    P10 at these parameters; finite output required."""
    N, M, B = 24, 120, 300
    a, b, W = wl.rbm_parameters(N, M, 0.5, [93, 0])
    ham = wl.tfim(wl.chain_bonds(N), N, 1.0, 0.7)
    w = wl.Workload("chain_N24_sigma0.5", N, M, B, wl.iid_spins(B, N, [93, 1]), a, b, W, ham)
    e, l, took = run(nqs, w)
    assert took["path"] == "small"
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "fast")
    check_eloc(e, e_ref, "sigma 0.5", rtol=1e-3)
    check_logpsi(l, l_ref, "sigma 0.5", rtol=1e-4)


def test_hidden_unit_rows_of_vanishing_weight(nqs, oracle):
    """the two-level split of W scales each row by 2^(11 - e), e the exponent of max|W_j|; for a row
    with 0 < max|W_j| < ~2^-116 that scale overflowed to inf and inf * 0 made theta NaN.  Rows at 1e-36, in the
    subnormal range and exactly zero, beside ordinary rows; the multi-launch path handles the same inputs."""
    N, M, B = 16, 32, 200
    a, b, W = wl.rbm_parameters(N, M, 0.05, [94, 0])
    W = W.copy()
    W[3] *= np.float32(1e-35)   # ~5e-37: normal float32, far below 2^-116
    W[7] *= np.float32(1e-36)
    W[7] *= np.float32(1e-6)    # ~5e-44: subnormal
    W[11] = 0
    assert 0 < np.abs(W[3]).max() < 2.0 ** -116 and 0 < np.abs(W[7]).max() < 1.2e-38
    ham = wl.tfim(wl.chain_bonds(N), N, 1.0, 0.7)
    w = wl.Workload("chain_N16_tiny_rows", N, M, B, wl.iid_spins(B, N, [94, 1]), a, b, W, ham)
    e, l, took = run(nqs, w)
    assert took["path"] == "small"
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "definition")
    check_eloc(e, e_ref, "tiny rows")
    check_logpsi(l, l_ref, "tiny rows")
    e2, l2, took2 = run(nqs, w, small=False)
    assert took2["path"] == "product"
    check_eloc(e2, e_ref, "tiny rows, multi-launch")


def test_selection_rule(nqs):
    """Tables that do not fit in shared memory (config-3 shapes: 100 x 400 x 16 bytes) and calls that keep tanh(theta)
    for the force vector take the multi-launch path; NQS_OPT_A5_PATH = 1 still means eloc_kernel."""
    w = wl.make_config(3, B=500)
    _, _, took = run(nqs, w)
    assert took["path"] == "product", took
    w = wl.make_config(2, B=500)
    nqs.set_option("a5_path", nqs.A5_PATHS["product"])
    try:
        _, _, took = run(nqs, w)
    finally:
        nqs.set_option("a5_path", 0)
    assert took["path"] == "product", took
    import torch

    spins, a, b, W = to_dev(w)
    ham = nqs.Hamiltonian(w.N, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    ham.local_energy_forces(spins, a, b, W)
    torch.cuda.synchronize()
    assert nqs.debug_last_a5()["path"] == "product"
    e1, _ = ham.local_energy(spins, a, b, W)
    e2, _ = ham.local_energy(spins, a, b, W)
    torch.cuda.synchronize()
    assert nqs.debug_last_a5()["path"] == "small" and torch.equal(e1, e2)  # run-to-run deterministic
    ham.close()


@pytest.mark.parametrize("N,M,B,T,K,sigma,seed", [
    (5, 4, 32, 30, 3, 0.3, 601),
    (7, 6, 128, 40, 4, 0.25, 602),
    (12, 9, 300, 80, 6, 0.2, 603),
    (20, 17, 517, 150, 8, 0.1, 604),
])
def test_k_site_strings(nqs, oracle, N, M, B, T, K, sigma, seed):
    """k-site Pauli strings (flip sets of up to four sites with all their relative-sign columns, Z riders beyond the
    first two) through the single-launch kernel, against definition mode."""
    w = wl.make_random(N, M, B, 4, sigma, seed)
    w.ham = wl.random_strings(N, T, K, np.random.default_rng([seed, 3]))
    e, l, took = run(nqs, w)
    assert took["path"] == "small", took
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "definition")
    check_eloc(e, e_ref, f"strings K={K} small")
    check_logpsi(l, l_ref, f"strings K={K} small")
