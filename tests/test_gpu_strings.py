"""k-site Pauli strings ("tensor products of branch-free operators") through the
C ABI (nqs_hamiltonian_create_k / nqs_local_energy_k) against the float64 oracle's definition mode, on both a5 paths.
Tolerances are the hot path's: 1e-4 max(1, |E_loc|) per real / imaginary part, 1e-5 max(1, |log psi|)."""
import numpy as np
import pytest

import workloads as wl
from test_gpu_parity import check_eloc, check_logpsi, gpu_eloc, oracle_on

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def nqs():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests need a B200")
    import paper_2108_03409_b200 as m

    m.load_library()
    yield m
    m.set_option("a5_path", 0)


def run(nqs, w, path):
    nqs.set_option("a5_path", nqs.A5_PATHS[path])
    try:
        e, l = gpu_eloc(nqs, w)
        took = nqs.debug_last_a5()
    finally:
        nqs.set_option("a5_path", 0)
    return e, l, took


@pytest.mark.parametrize("N,M,B,T,K,sigma,seed", [
    (5, 4, 32, 30, 3, 0.3, 501),      # all 2^5 states; 3-slot strings
    (7, 6, 128, 40, 4, 0.25, 502),    # all 2^7 states; up to four flipping sites
    (12, 9, 300, 80, 6, 0.2, 503),    # six slots: several Z riders per string
    (20, 17, 517, 150, 8, 0.1, 504),  # eight slots, ragged batch
])
def test_random_strings_vs_definition_product_form(nqs, oracle, N, M, B, T, K, sigma, seed):
    w = wl.make_random(N, M, B, 4, sigma, seed)
    w.ham = wl.random_strings(N, T, K, np.random.default_rng([seed, 3]))
    e, l, took = run(nqs, w, "product")
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "definition")
    check_eloc(e, e_ref, f"strings K={K} product")
    check_logpsi(l, l_ref, f"strings K={K}")


@pytest.mark.parametrize("N,M,B,T,K,sigma,seed", [
    (7, 6, 128, 40, 4, 0.004, 512),
    (20, 17, 517, 150, 8, 0.002, 514),
])
def test_random_strings_vs_definition_series(nqs, oracle, N, M, B, T, K, sigma, seed):
    """The tensor-core series path alone (fallback disabled) on k-site strings: 3- and 4-site flip sets with all their
    relative-sign columns, terms with more than two Z factors (the epilogue's general term list)."""
    w = wl.make_random(N, M, B, 4, sigma, seed)
    w.ham = wl.random_strings(N, T, K, np.random.default_rng([seed, 3]))
    e, l, took = run(nqs, w, "series_only")
    assert took["path"] == "series" and not took["guard_failed"], took
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "definition")
    check_eloc(e, e_ref, f"strings K={K} series")


def test_hand_written_strings_and_handle(nqs, oracle):
    import torch

    N, M = 5, 3
    w = wl.make_random(N, M, 1 << N, 1, 0.3, 19)
    X, Y, Z = 1, 2, 3
    sites = np.array([[0, 1, 2, -1], [1, 2, 3, -1], [0, 2, 4, -1], [0, 1, 2, 3], [1, 2, 3, 4]], np.int32)
    paulis = np.array([[X, X, X, 0], [Y, Y, Y, 0], [X, Y, Z, 0], [Z, Z, Z, Z], [X, Z, Z, X]], np.uint8)
    coeffs = np.array([0.5, -0.25 + 0.5j, 1.5, -1.0, 0.75j], np.complex64)
    w.ham = wl.Hamiltonian(sites, paulis, coeffs)
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "definition")
    e, l, _ = run(nqs, w, "product")
    check_eloc(e, e_ref, "hand-written strings")
    # compiled handle: flip sets, enumerator (Eq. 39 as data) against the oracle's term-by-term list
    ham = nqs.Hamiltonian(N, sites, paulis, coeffs)
    assert ham.flip_sites4.tolist() == [[0, 1, 2, -1], [1, 2, 3, -1], [0, 2, -1, -1], [1, 4, -1, -1]]
    spins = torch.from_numpy(w.spins).cuda()
    sp, mel = nqs.enumerate_connected_h(ham, spins)
    torch.cuda.synchronize()
    sp, mel = sp.cpu().numpy(), mel.cpu().numpy().astype(np.complex128)
    sp_ref, mel_ref = oracle.connected(w.spins, sites, paulis, coeffs)
    for bidx in range(w.B):
        agg = {}
        for t in range(len(coeffs)):
            key = sp_ref[bidx, t].tobytes()
            agg[key] = agg.get(key, 0) + mel_ref[bidx, t]
        for slot in range(ham.G + 1):
            key = sp[bidx, slot].tobytes()
            assert abs(agg.get(key, 0) - mel[bidx, slot]) <= 1e-5 * max(1, abs(agg.get(key, 0)))
    e2, _ = ham.local_energy(spins, *(torch.from_numpy(x).cuda() for x in (w.a, w.b, w.W)))
    torch.cuda.synchronize()
    check_eloc(e2.cpu().numpy(), e_ref, "hand-written strings, handle API (single-launch kernel)")
    with pytest.raises(nqs.NqsError) as ei:
        nqs.Hamiltonian(6, np.array([[0, 1, 2, 3, 4]], np.int32), np.full((1, 5), X, np.uint8), np.ones(1, np.complex64))
    assert ei.value.code == -4


def test_plaquette_model_full_batch_both_paths(nqs, oracle):
    """A 6 x 6 periodic lattice with four-site plaquette terms -J Z Z Z Z - h X X X X on every plaquette plus a
    transverse field: 36 four-site flip sets (8 sign columns each) + 36 single flips, B = 4096, fast-mode oracle on
    the full batch; once through the product form and once through the guarded series."""
    L = 6
    N, M, B = L * L, 72, 4096
    a, b, W = wl.rbm_parameters(N, M, 0.004, [77, 0])
    rows_s, rows_p, cs = [], [], []
    for x in range(L):
        for y in range(L):
            plq = [x * L + y, x * L + (y + 1) % L, ((x + 1) % L) * L + y, ((x + 1) % L) * L + (y + 1) % L]
            rows_s += [plq, plq]
            rows_p += [[3, 3, 3, 3], [1, 1, 1, 1]]
            cs += [-1.0, -0.5]
    for i in range(N):
        rows_s.append([i, -1, -1, -1])
        rows_p.append([1, 0, 0, 0])
        cs.append(-0.7)
    ham = wl.Hamiltonian(np.array(rows_s, np.int32), np.array(rows_p, np.uint8), np.array(cs, np.complex64))
    w = wl.Workload("plaquette_6x6", N, M, B, wl.iid_spins(B, N, [77, 1]), a, b, W, ham)
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "fast")
    e_def, _ = oracle_on(oracle, w, slice(0, 64), "definition")
    assert np.abs(e_ref[:64] - e_def).max() < 1e-9
    ep, lp, _ = run(nqs, w, "product")
    check_eloc(ep, e_ref, "plaquette product")
    check_logpsi(lp, l_ref, "plaquette")
    es, _, took = run(nqs, w, "series_guarded")
    assert took["path"] == "series"
    check_eloc(es, e_ref, "plaquette series (guarded)")
