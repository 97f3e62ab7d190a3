"""Parity of nqs_fisher / nqs_vmc_step_h (the quantum Fisher matrix
S = <<O* O>>_c, Eq. 10-11) against the float64 oracle, element by element.

Tolerance.  An entry S_kk' is a sum over the samples of terms bounded by the Cauchy-Schwarz
scale sqrt(S_kk S_k'k').  The GPU forms each term from a float32 tanh (<= 1.2e-7 relative) split into two FP16 parts
(2^-22) and accumulates B / 16 tensor-core steps in FP32 (error modelled as a random walk: sqrt(B/16 * 12) * 2^-24
~ 7e-6 at B = 16384).  Hence  |dS_kk'| <= 2e-5 sqrt(S_kk S_k'k') + 1e-7 max_k S_kk  per real / imaginary part
(about 3 x the model).  <O_k> comes from the exact int8 contraction of nqs_forces, so it carries only the float32
error of tanh theta itself: 2e-6 max(1, max_bj |tanh theta_bj|), the tolerance of tests/test_gpu_forces.py.
"""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu

S_RTOL = 2e-5


@pytest.fixture(scope="module")
def nqs():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests need a B200")
    import paper_2108_03409_b200 as m

    m.load_library()
    return m


def gpu_fisher(nqs, w, weights=None):
    import torch

    d = torch.device("cuda:0")
    t = lambda x: torch.from_numpy(np.ascontiguousarray(x)).to(d)  # noqa: E731
    S, Obar = nqs.fisher(t(w.spins), t(w.a), t(w.b), t(w.W), t(weights) if weights is not None else None)
    torch.cuda.synchronize()
    assert torch.equal(S, S.conj().transpose(0, 1).contiguous()), "S is not exactly Hermitian"
    return S.cpu().numpy().astype(np.complex128), Obar.cpu().numpy().astype(np.complex128)


def tanh_scale(w):
    theta = w.spins.astype(np.float64) @ w.W.astype(np.complex128).T + w.b.astype(np.complex128)[None, :]
    return max(1.0, float(np.abs(np.tanh(theta)).max()))


def check(S, Obar, S_ref, Obar_ref, what, tscale=1.0):
    d = np.sqrt(np.maximum(np.diag(S_ref).real, 0.0))
    tol = S_RTOL * np.outer(d, d) + 1e-7 * d.max() ** 2
    err = np.maximum(np.abs(S.real - S_ref.real), np.abs(S.imag - S_ref.imag))
    worst = (err / tol).max()
    assert np.all(np.isfinite(S.view(np.float64))), what
    assert worst <= 1.0, f"{what}: S error {worst:.3f} x tolerance at {np.unravel_index((err / tol).argmax(), err.shape)}"
    assert np.abs(Obar - Obar_ref).max() <= 2e-6 * tscale, what
    return worst


def test_fisher_config1_full_basis_with_born_weights(nqs, oracle):
    """Config 1: all 256 basis states weighted with p(s) ~ |psi(s)|^2 -- the exact S of the state (K = 80)."""
    w = wl.make_config(1)
    lp = oracle.log_psi(w.spins, w.a, w.b, w.W)
    wts = np.exp(2.0 * (lp.real - lp.real.max())).astype(np.float32)
    S, Obar = gpu_fisher(nqs, w, wts)
    S_ref, Obar_ref = oracle.fisher(w.spins, w.a, w.b, w.W, weights=wts)
    assert S.shape == (80, 80)
    check(S, Obar, S_ref, Obar_ref, "config 1")


def test_fisher_config2_full_batch(nqs, oracle):
    """Config 2 at full size: K = 3320 parameters, B = 16384 samples, every one of the 11 million entries."""
    w = wl.make_config(2)
    S, Obar = gpu_fisher(nqs, w)
    S_ref, Obar_ref = oracle.fisher(w.spins, w.a, w.b, w.W)
    assert S.shape == (3320, 3320)
    check(S, Obar, S_ref, Obar_ref, "config 2")


@pytest.mark.parametrize("N,M,B,sigma,seed,weighted", [
    (7, 5, 300, 0.3, 401, True),      # K = 47: one ragged tile, ragged batch
    (13, 9, 1000, 0.2, 402, False),   # K = 139: two tiles, the second with 11 live rows
    (20, 18, 777, 0.25, 403, True),   # K = 398: four tiles -> ten tile pairs incl. mirrored ones
    (3, 2, 5, 0.4, 404, False),       # tiny: B = 5 samples
])
def test_fisher_ragged_shapes(nqs, oracle, N, M, B, sigma, seed, weighted):
    w = wl.make_random(N, M, B, 4, sigma, seed)
    wts = np.random.default_rng(seed).random(w.B).astype(np.float32) if weighted else None
    S, Obar = gpu_fisher(nqs, w, wts)
    S_ref, Obar_ref = oracle.fisher(w.spins, w.a, w.b, w.W, weights=wts)
    check(S, Obar, S_ref, Obar_ref, f"N={N} M={M} B={w.B}", tanh_scale(w))


def test_fisher_properties(nqs):
    import torch

    w = wl.make_random(9, 6, 400, 4, 0.3, 405)
    S1, O1 = gpu_fisher(nqs, w)
    S2, O2 = gpu_fisher(nqs, w)
    assert np.array_equal(S1, S2) and np.array_equal(O1, O2)  # deterministic
    ev = np.linalg.eigvalsh(S1)
    assert ev.min() > -1e-5 * ev.max()  # positive semi-definite up to rounding
    # the a-block of S is the plain covariance matrix of the spins
    s = w.spins.astype(np.float64)
    cov = np.cov(s.T, bias=True)
    assert np.abs(S1[:w.N, :w.N] - cov).max() <= S_RTOL
    # uniform weights equal no weights
    S3, _ = gpu_fisher(nqs, w, np.full(w.B, 2.5, np.float32))
    assert np.abs(S3 - S1).max() <= 1e-6
    d = torch.device("cuda:0")
    lib = nqs.load_library()
    assert lib.nqs_fisher(None, 0, 9, 6, None, None, None, None, None, None, None) == 0   # B == 0: no-op
    assert lib.nqs_fisher(None, 4, 9, 6, None, None, None, None, None, None, None) == -1  # NULL pointers
    big = wl.make_config(3, B=256)  # K = 40500 > 8192
    t = lambda x: torch.from_numpy(np.ascontiguousarray(x)).to(d)  # noqa: E731
    with pytest.raises(nqs.NqsError) as ei:
        nqs.fisher(t(big.spins), t(big.a), t(big.b), t(big.W))
    assert ei.value.code == -4


def test_vmc_step_equals_the_separate_calls(nqs, oracle):
    import torch

    d = torch.device("cuda:0")
    w = wl.make_config(2, B=3000)
    t = lambda x: torch.from_numpy(np.ascontiguousarray(x)).to(d)  # noqa: E731
    spins, a, b, W = t(w.spins), t(w.a), t(w.b), t(w.W)
    ham = nqs.Hamiltonian(w.N, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    e1, l1, F1, st1 = ham.local_energy_forces(spins, a, b, W)
    S1, O1 = nqs.fisher(spins, a, b, W)
    e2, l2, F2, S2, O2, st2 = ham.vmc_step(spins, a, b, W)
    torch.cuda.synchronize()
    assert torch.equal(e1, e2) and torch.equal(l1, l2) and torch.equal(F1, F2) and torch.equal(st1, st2)
    assert torch.equal(S1, S2) and torch.equal(O1, O2)
    # and against the oracle on this batch (Algorithm 1 lines 6-9 in one call)
    S_ref, Obar_ref = oracle.fisher(w.spins, w.a, w.b, w.W)
    check(S2.cpu().numpy().astype(np.complex128), O2.cpu().numpy().astype(np.complex128), S_ref, Obar_ref, "vmc_step")
