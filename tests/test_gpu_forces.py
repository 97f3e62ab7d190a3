"""Parity of nqs_energy_stats / nqs_forces against the float64 oracle.

Tolerance: every term w_b conj(t_bj) (E_b - mean) of the sum is formed in float32
from a float32 tanh (<= ~8 ulp = 5e-7 relative per term) and then summed EXACTLY (integer GEMM), so
    |dF_k| <= 2e-6 * S,   S = <<|E - mean|>> * max(1, max |tanh theta|),
for the real and imaginary parts separately (4x margin over the per-term bound).
The statistics are float64 sums of the float32 inputs: 1e-12 relative.
"""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu

F_TOL = 2e-6


@pytest.fixture(scope="module")
def nqs():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests need a B200")
    import paper_2108_03409_b200 as m

    m.load_library()
    return m


def synthetic_eloc(B, seed, centre=-50.0, spread=3.0):
    """Stand-in local energies (complex64): the force vector is linear in them, any values do."""
    rng = np.random.default_rng([seed, 7])
    return (centre + spread * rng.standard_normal(B) + 1j * spread * 0.3 * rng.standard_normal(B)).astype(np.complex64)


def gpu_forces(nqs, w, eloc, weights=None):
    import torch

    d = torch.device("cuda:0")
    t = lambda x: torch.from_numpy(np.ascontiguousarray(x)).to(d)  # noqa: E731
    F, st = nqs.forces(t(w.spins), t(w.a), t(w.b), t(w.W), t(eloc), None if weights is None else t(weights),
                       want_stats=True)
    torch.cuda.synchronize()
    return F.cpu().numpy().astype(np.complex128), st.cpu().numpy()


def scale_S(w, eloc, weights=None):
    e = eloc.astype(np.complex128)
    wt = np.ones(len(e)) if weights is None else weights.astype(np.float64)
    mean = (wt * e).sum() / wt.sum()
    theta = w.spins.astype(np.float64) @ w.W.astype(np.complex128).T + w.b.astype(np.complex128)[None, :]
    return (wt * np.abs(e - mean)).sum() / wt.sum() * max(1.0, np.abs(np.tanh(theta)).max())


def check_forces(F, F_ref, S, what):
    err = max(np.abs(F.real - F_ref.real).max(), np.abs(F.imag - F_ref.imag).max())
    assert np.all(np.isfinite(F.view(np.float64))), what
    assert err <= F_TOL * S, f"{what}: max |dF| = {err:.3e} = {err / (F_TOL * S):.2f} x tolerance"


@pytest.mark.parametrize("N,M,B,sigma,seed,weighted", [
    (8, 8, 256, 0.05, 1, False),        # config-1 shapes, one tile
    (37, 45, 1000, 0.2, 2, True),       # ragged everything, weights
    (130, 70, 777, 0.1, 3, False),      # two site tiles (N + 1 > 128), three hidden tiles
    (127, 31, 300, 0.3, 4, True),       # N + 1 = 128 and M + 1 = 32 exactly fill a tile
    (40, 80, 16384, 0.02, 5, False),    # config-2 shapes
])
def test_forces_vs_oracle_small(nqs, oracle, N, M, B, sigma, seed, weighted):
    w = wl.make_random(N, M, B, 4, sigma, 100 + seed)
    eloc = synthetic_eloc(w.B, seed)
    weights = np.random.default_rng([seed, 8]).random(w.B).astype(np.float32) if weighted else None
    F, st = gpu_forces(nqs, w, eloc, weights)
    F_ref = oracle.forces(w.spins, w.a, w.b, w.W, eloc, None if weights is None else weights.astype(np.float64))
    check_forces(F, F_ref, scale_S(w, eloc, weights), f"N={N} M={M} B={w.B}")
    m, v, sw = oracle.mean_variance(eloc, None if weights is None else weights.astype(np.float64))
    assert abs(complex(st[0], st[1]) - m) <= 1e-12 * abs(m) and abs(st[2] - v) <= 1e-9 * v and abs(st[3] - sw) <= 1e-12 * sw


def test_forces_with_real_local_energies_config1(nqs, oracle):
    """End to end on config 1: E_loc from the oracle (cast to complex64, the ABI's type) -> forces."""
    w = wl.make_config(1)
    e, _ = oracle.local_energy_definition(w.spins, w.a, w.b, w.W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    eloc = e.astype(np.complex64)
    F, _ = gpu_forces(nqs, w, eloc)
    check_forces(F, oracle.forces(w.spins, w.a, w.b, w.W, eloc), scale_S(w, eloc), "config 1")


def test_forces_config3_full_batch(nqs, oracle):
    w = wl.make_config(3)
    eloc = synthetic_eloc(w.B, 33, centre=-300.0)
    F, _ = gpu_forces(nqs, w, eloc)
    check_forces(F, oracle.forces(w.spins, w.a, w.b, w.W, eloc), scale_S(w, eloc), "config 3 full batch")


def test_forces_config5_full_size_sampled_outputs(nqs, oracle):
    """Config 5 at full size (the launch configuration bench.py times).  An RBM restricted to a subset
    of hidden units has the same O_{b_j}, O_{W_ji} for those units and the same O_{a_i}, so the oracle
    computes the a-part, and the b- and W-parts of 12 sampled hidden units, one by one."""
    w = wl.make_config(5)
    eloc = synthetic_eloc(w.B, 55, centre=-1200.0)
    F, st = gpu_forces(nqs, w, eloc)
    # 12 random hidden units plus the tile boundaries of force_mma_kernel (32 hidden units per CTA column):
    # first / last unit and both sides of a boundary near each end.  All N sites are compared for every
    # sampled unit, so the site-tile boundaries i = 127|128, 255|256, 383|384 are covered by construction
    # (asserted below).
    forced = [0, 31, 32, 1567, 1568, w.M - 1]
    rnd = np.random.default_rng(56).choice(w.M, size=12, replace=False)
    jsel = np.unique(np.concatenate([rnd, forced]))
    assert {31, 32, 1567, 1568} <= set(jsel.tolist()) and w.N > 384
    F_ref = oracle.forces(w.spins, w.a, w.b[jsel], w.W[jsel], eloc)
    N, M = w.N, w.M
    S = scale_S(wl.Workload("sub", N, len(jsel), w.B, w.spins, w.a, w.b[jsel], w.W[jsel], w.ham), eloc)
    check_forces(F[:N], F_ref[:N], S, "config 5 a-part")
    check_forces(F[N:N + M][jsel], F_ref[N:N + len(jsel)], S, "config 5 b-part (sampled)")
    check_forces(F[N + M:].reshape(M, N)[jsel], F_ref[N + len(jsel):].reshape(len(jsel), N), S, "config 5 W-part (sampled)")
    m, v, _ = oracle.mean_variance(eloc)
    assert abs(complex(st[0], st[1]) - m) <= 1e-12 * abs(m) and abs(st[2] - v) <= 1e-9 * v


def test_forces_properties_and_determinism(nqs):
    import torch

    w = wl.make_config(3, B=5000)
    const = np.full(w.B, -7.0 + 2.0j, dtype=np.complex64)
    F0, st = gpu_forces(nqs, w, const)
    assert np.all(F0 == 0) and st[2] == 0.0  # constant E_loc: connected correlation vanishes exactly
    eloc = synthetic_eloc(w.B, 9)
    F1, _ = gpu_forces(nqs, w, eloc)
    F2, _ = gpu_forces(nqs, w, eloc)
    assert np.array_equal(F1, F2)  # integer accumulation: run-to-run identical
    # the a-part is a plain covariance with the spins
    s = w.spins.astype(np.float64)
    e = eloc.astype(np.complex128)
    cov = (s * e[:, None]).mean(0) - s.mean(0) * e.mean()
    assert np.abs(F1[:w.N] - cov).max() <= F_TOL * np.abs(e - e.mean()).mean()
    d = torch.device("cuda:0")
    x = torch.from_numpy(eloc).to(d)
    st2 = nqs.energy_stats(x).cpu().numpy()
    assert abs(complex(st2[0], st2[1]) - e.mean()) <= 1e-12 * abs(e.mean()) and abs(st2[2] - e.var()) <= 1e-9 * e.var()


def test_forces_error_codes(nqs):
    import torch

    d = torch.device("cuda:0")
    w = wl.make_config(1)
    t = lambda x: torch.from_numpy(x).to(d)  # noqa: E731
    with pytest.raises(ValueError):
        nqs.forces(t(w.spins), t(w.a), t(w.b), t(w.W), t(synthetic_eloc(w.B + 1, 1)))
    lib = nqs.load_library()
    assert lib.nqs_forces(None, 4, 8, 8, None, None, None, None, None, None, None, None) == -1
    assert lib.nqs_energy_stats(None, None, -1, None, None) == -1
    assert lib.nqs_energy_stats(None, None, 0, None, None) == 0  # B == 0 is a no-op for every entry point
    assert lib.nqs_forces(None, 0, 8, 8, None, None, None, None, None, None, None, None) == 0


def test_fused_local_energy_forces_equals_the_two_calls(nqs):
    import torch

    d = torch.device("cuda:0")
    for k, B in ((2, 3000), (4, 1111)):
        w = wl.make_config(k, B=B)
        t = lambda x: torch.from_numpy(np.ascontiguousarray(x)).to(d)  # noqa: E731
        spins, a, b, W = t(w.spins), t(w.a), t(w.b), t(w.W)
        ham = nqs.Hamiltonian(w.N, w.ham.sites, w.ham.paulis, w.ham.coeffs)
        # the fused call keeps tanh(theta) and therefore runs the multi-launch kernels: compare with the same kernels
        # (the single-launch kernel for small problems is another arithmetic, judged against the oracle elsewhere)
        nqs.set_option("small_path", 1)
        try:
            e1, l1 = ham.local_energy(spins, a, b, W)
        finally:
            nqs.set_option("small_path", 0)
        F1, s1 = nqs.forces(spins, a, b, W, e1, want_stats=True)
        e2, l2, F2, s2 = ham.local_energy_forces(spins, a, b, W)
        torch.cuda.synchronize()
        assert torch.equal(e1, e2) and torch.equal(l1, l2) and torch.equal(F1, F2) and torch.equal(s1, s2)
