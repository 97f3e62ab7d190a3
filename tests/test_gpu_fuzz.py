"""Randomised shapes through every device entry point against the oracle (ragged tiles, odd sizes,
chains and batches that are not multiples of any block): the cheap stand-in for a memory checker."""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu


def test_random_shapes_all_entry_points(oracle):
    import torch

    import paper_2108_03409_b200 as nqs

    d = torch.device("cuda:0")
    t = lambda x: torch.from_numpy(np.ascontiguousarray(x)).to(d)  # noqa: E731
    rng = np.random.default_rng(2024)
    for case in range(24):
        N = int(rng.integers(2, 150))
        M = int(rng.integers(1, 130))
        B = int(rng.integers(1, 700))
        T = int(rng.integers(1, 3 * N))
        sigma = float(rng.choice([0.02, 0.1, 0.25]))
        w = wl.make_random(N, M, B, T, sigma, 1000 + case)
        what = f"case {case}: N={N} M={M} B={w.B} T={T} sigma={sigma}"
        sp, a, b, W = t(w.spins), t(w.a), t(w.b), t(w.W)
        ham = nqs.Hamiltonian(w.N, w.ham.sites, w.ham.paulis, w.ham.coeffs)
        e, l, F, st = ham.local_energy_forces(sp, a, b, W)
        torch.cuda.synchronize()
        e, l, F = (x.cpu().numpy().astype(np.complex128) for x in (e, l, F))
        e_ref, l_ref = oracle.local_energy_fast(w.spins, w.a, w.b, w.W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
        tol_e = 1e-4 * np.maximum(1.0, np.abs(e_ref))
        assert np.all(np.abs(e.real - e_ref.real) <= tol_e) and np.all(np.abs(e.imag - e_ref.imag) <= tol_e), what
        tol_l = 1e-5 * np.maximum(1.0, np.abs(l_ref))
        dim = (l.imag - l_ref.imag + np.pi) % (2 * np.pi) - np.pi
        assert np.all(np.abs(l.real - l_ref.real) <= tol_l) and np.all(np.abs(dim) <= tol_l), what
        # the plain call (single-launch kernel where its tables fit, else the multi-launch path)
        e1, l1 = ham.local_energy(sp, a, b, W)
        torch.cuda.synchronize()
        e1, l1 = (x.cpu().numpy().astype(np.complex128) for x in (e1, l1))
        assert np.all(np.abs(e1.real - e_ref.real) <= tol_e) and np.all(np.abs(e1.imag - e_ref.imag) <= tol_e), what
        dim = (l1.imag - l_ref.imag + np.pi) % (2 * np.pi) - np.pi
        assert np.all(np.abs(l1.real - l_ref.real) <= tol_l) and np.all(np.abs(dim) <= tol_l), what
        # forces from the GPU's own E_loc bytes (complex64), as the fused call used them
        e32 = e.astype(np.complex64)
        F_ref = oracle.forces(w.spins, w.a, w.b, w.W, e32)
        theta = w.spins.astype(np.float64) @ w.W.astype(np.complex128).T + w.b.astype(np.complex128)[None, :]
        S = np.abs(e32 - e32.mean()).mean() * max(1.0, np.abs(np.tanh(theta)).max())
        assert np.abs(F - F_ref).max() <= 2e-6 * S + 1e-30, what
        # a few Metropolis steps
        steps = int(rng.integers(1, 3 * N))
        sites = rng.integers(0, N, (steps, w.B)).astype(np.int32)
        u = rng.random((steps, w.B), dtype=np.float32)
        chains = sp.clone()
        acc, dec = nqs.metropolis(chains, a, b, W, t(sites), t(u), trace=True)
        torch.cuda.synchronize()
        final, acc, dec = chains.cpu().numpy(), acc.cpu().numpy(), dec.cpu().numpy()
        ref_final, ref_acc, _, ref_dec, ref_mar = oracle.metropolis(w.spins, w.a, w.b, w.W, sites, u, trace=True)
        # every chain: identical decisions => identical result; else the first differing decision was a near-tie
        assert set(np.unique(final)) <= {-1, 1}, what
        assert np.array_equal(dec.sum(axis=0), acc), what
        differ = dec != ref_dec
        parted = differ.any(axis=0)
        assert np.array_equal(final[~parted], ref_final[~parted]) and np.array_equal(acc[~parted], ref_acc[~parted]), what
        if parted.any():
            first = differ.argmax(axis=0)[parted]
            assert np.all(ref_mar[first, np.flatnonzero(parted)] < 2e-4), what
        ham.close()
