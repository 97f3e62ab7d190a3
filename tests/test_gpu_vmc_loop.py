"""The pieces compose into the paper's ground-state search (Eq. 6-9): log psi ->
weights p = |psi|^2 over the full basis (exact sampling, :486 ExactSampler) -> E_loc -> mean (Eq. 3)
-> force vector (Eq. 16) -> theta <- theta - tau F.  Everything on the GPU path; the target is the
closed-form ground energy of the N = 8 TFIM ring (tests/golden, PAPER.md:588 ref. [66]).  A wrong
sign or conjugation anywhere in nqs_forces makes the energy go up instead of down."""
import json
import os

import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu


def test_gradient_descent_reaches_the_tfim_ground_energy():
    import torch

    import paper_2108_03409_b200 as nqs

    golden = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "tfim_ring_ground_energy.json")))
    e0 = next(c["E0"] for c in golden["cases"] if c["N"] == 8 and c["h"] == 1.0)
    w = wl.make_config(1)  # N = 8, M = 8, all 256 basis states, H = -sum ZZ - sum X
    d = torch.device("cuda:0")
    spins = torch.from_numpy(w.spins).to(d)
    a, b, W = (torch.from_numpy(x).to(d) for x in (w.a, w.b, w.W))
    ham = nqs.Hamiltonian(w.N, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    N, M = w.N, w.M
    tau, energies = 0.05, []
    for it in range(400):
        eloc, logpsi = ham.local_energy(spins, a, b, W)
        lw = 2.0 * logpsi.real
        p = torch.exp(lw - lw.max()).to(torch.float32).contiguous()
        F, st = nqs.forces(spins, a, b, W, eloc, weights=p, want_stats=True)
        energies.append(float(st[0].item()))
        assert abs(float(st[1].item())) < 1e-3  # Hermitian H: <H> is real
        a = (a - tau * F[:N]).contiguous()
        b = (b - tau * F[N:N + M]).contiguous()
        W = (W - tau * F[N + M:].reshape(M, N)).contiguous()
    energies = np.array(energies)
    assert energies[0] > -9.0  # random start: about -8
    assert np.all(np.diff(energies) < 1e-4)  # plain gradient descent with a small step never goes up
    assert e0 - 1e-3 <= energies[-1] < e0 + 0.05, (energies[-1], e0)  # variational: never below E0
