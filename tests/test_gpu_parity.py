"""Parity of the CUDA path (through the C ABI) against the float64 oracle, on a B200.

Tolerances are BASELINE.json's (north_star), per sample:
  |Re dE|, |Im dE| <= 1e-4 * max(1, |E_loc|)        (reading Q15)
  |Re dlogpsi|, |Im dlogpsi wrapped to (-pi, pi]| <= 1e-5 * max(1, |log psi|)   (reading Q6)
"""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu

E_RTOL = 1e-4
L_RTOL = 1e-5


@pytest.fixture(scope="module")
def nqs():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests need a B200")
    import paper_2108_03409_b200 as m

    m.load_library()  # fail loudly if the extension is missing
    return m


def _wrap(d):
    return (d + np.pi) % (2 * np.pi) - np.pi


def check_eloc(e_gpu, e_ref, what, rtol=E_RTOL):
    e_gpu = np.asarray(e_gpu, dtype=np.complex128)
    tol = rtol * np.maximum(1.0, np.abs(e_ref))
    dr, di = np.abs(e_gpu.real - e_ref.real), np.abs(e_gpu.imag - e_ref.imag)
    worst = max((dr / tol).max(), (di / tol).max())
    assert np.all(np.isfinite(e_gpu.view(np.float64))), f"{what}: non-finite E_loc"
    assert worst <= 1.0, f"{what}: E_loc error {worst:.3f} x tolerance (max |dRe| {dr.max():.3e}, |dIm| {di.max():.3e})"
    return worst


def check_logpsi(l_gpu, l_ref, what, rtol=L_RTOL):
    l_gpu = np.asarray(l_gpu, dtype=np.complex128)
    tol = rtol * np.maximum(1.0, np.abs(l_ref))
    dr = np.abs(l_gpu.real - l_ref.real)
    di = np.abs(_wrap(l_gpu.imag - l_ref.imag))
    worst = max((dr / tol).max(), (di / tol).max())
    assert worst <= 1.0, f"{what}: log psi error {worst:.3f} x tolerance (max |dRe| {dr.max():.3e}, |dIm| {di.max():.3e})"
    return worst


def to_dev(w):
    import torch

    d = torch.device("cuda:0")
    return (torch.from_numpy(w.spins).to(d), torch.from_numpy(w.a).to(d), torch.from_numpy(w.b).to(d),
            torch.from_numpy(w.W).to(d))


def gpu_eloc(nqs, w):
    import torch

    spins, a, b, W = to_dev(w)
    e, l = nqs.local_energy(spins, a, b, W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    torch.cuda.synchronize()
    return e.cpu().numpy(), l.cpu().numpy()


def oracle_on(oracle, w, idx, mode):
    fn = oracle.local_energy_definition if mode == "definition" else oracle.local_energy_fast
    return fn(w.spins[idx], w.a, w.b, w.W, w.ham.sites, w.ham.paulis, w.ham.coeffs)


# ------------------------------------------------------------------ the five configurations
def test_config1_all_basis_states_vs_definition(nqs, oracle):
    w = wl.make_config(1)
    e, l = gpu_eloc(nqs, w)
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "definition")
    check_eloc(e, e_ref, "c1")
    check_logpsi(l, l_ref, "c1")


def test_config2_full_batch(nqs, oracle):
    w = wl.make_config(2)
    e, l = gpu_eloc(nqs, w)
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "fast")
    check_eloc(e, e_ref, "c2 fast")
    check_logpsi(l, l_ref, "c2 fast")
    idx = np.arange(0, w.B, 37)
    e_def, l_def = oracle_on(oracle, w, idx, "definition")
    check_eloc(e[idx], e_def, "c2 definition")
    check_logpsi(l[idx], l_def, "c2 definition")


_ORACLE_CACHE = {}


def full_size_sample(k, B):
    """Outputs the oracle recomputes at full size: three whole 128-sample tiles (first, middle, last: every
    position inside a CTA of either a5 kernel, i.e. every b mod 128 and b mod 64) plus every 17th sample of
    the batch (every 7th at B = 32768; 17 and 7 are coprime to the tile sizes, so every residue is hit)."""
    mid = (B // 2) // 128 * 128
    stride = 17 if B >= 65536 else 7
    idx = np.concatenate([np.arange(0, 128), np.arange(mid, mid + 128), np.arange(B - 128, B), np.arange(0, B, stride)])
    idx = np.unique(idx)
    d_idx = np.unique(np.concatenate([np.linspace(0, B - 1, 124).astype(np.int64), [63, 64, 127, 128, B - 129, B - 128]]))
    return idx, d_idx


def oracle_full_size(oracle, k):
    if k not in _ORACLE_CACHE:
        w = wl.make_config(k)
        idx, d_idx = full_size_sample(k, w.B)
        _ORACLE_CACHE[k] = (w, idx, oracle_on(oracle, w, idx, "fast"), d_idx, oracle_on(oracle, w, d_idx, "definition"))
    return _ORACLE_CACHE[k]


@pytest.mark.parametrize("path", ["auto", "product"])
@pytest.mark.parametrize("k", [3, 4, 5])
def test_full_size_configs_sampled_outputs(nqs, oracle, k, path):
    """GPU runs the FULL batch in bench.py's launch configuration, once through the default a5 path (the
    tensor-core series with its guard at these sizes) and once through the FP32 product form; the oracle
    recomputes >= 4096 sampled outputs in fast mode and >= 128 in definition mode (see full_size_sample)."""
    w, idx, (e_ref, l_ref), d_idx, (e_def, l_def) = oracle_full_size(oracle, k)
    assert idx.size >= 4096 and d_idx.size >= 128
    nqs.set_option("a5_path", nqs.A5_PATHS[path])
    try:
        e, l = gpu_eloc(nqs, w)
        took = nqs.debug_last_a5()
    finally:
        nqs.set_option("a5_path", 0)
    if path == "auto":
        assert took["path"] == "series" and not took["guard_failed"], took  # the configs sit well inside the guard
    else:
        assert took["path"] == "product", took
    assert np.all(np.isfinite(e.view(np.float32))) and np.all(np.isfinite(l.view(np.float32)))
    check_eloc(e[idx], e_ref, f"c{k} fast [{path}]")
    check_logpsi(l[idx], l_ref, f"c{k} fast [{path}]")
    check_eloc(e[d_idx], e_def, f"c{k} definition [{path}]")
    check_logpsi(l[d_idx], l_def, f"c{k} definition [{path}]")
    # property that holds at any size (TFIM: zero-parameter closed form is tested separately);
    # here: the batch mean is finite and the imaginary parts are small against the real ones
    assert abs(e.imag.mean()) < 0.05 * abs(e.real.mean())


@pytest.mark.parametrize("k", [3, 5])
def test_zero_parameter_closed_form_full_size(nqs, k):
    """P3 at full size: a = b = W = 0 => E_loc = -J sum s_i s_k - h N exactly (integers)."""
    w = wl.make_config(k)
    w.a[:] = 0
    w.b[:] = 0
    w.W[:] = 0
    e, l = gpu_eloc(nqs, w)
    spec = wl.config_spec(k)
    s = w.spins.astype(np.float64)
    zz = sum(s[:, i] * s[:, j] for i, j in wl.square_bonds(spec["L"]))
    expect = -spec["J"] * zz - spec["h"] * w.N
    assert np.array_equal(e.real.astype(np.float64), expect)
    assert np.all(e.imag == 0) and np.all(l == 0)


# ------------------------------------------------------------------ log psi entry point
@pytest.mark.parametrize("k,B", [(1, None), (2, 1000), (3, 300), (5, 130)])
def test_log_psi_entry_point(nqs, oracle, k, B):
    import torch

    w = wl.make_config(k, B=B) if B else wl.make_config(k)
    spins, a, b, W = to_dev(w)
    l = nqs.log_psi(spins, a, b, W)
    torch.cuda.synchronize()
    l_ref = oracle.log_psi(w.spins, w.a, w.b, w.W, stable=False)
    check_logpsi(l.cpu().numpy(), l_ref, f"log_psi c{k}")
    l_host = nqs.log_psi_host(w.spins, w.a, w.b, w.W)
    assert np.array_equal(l_host, l.cpu().numpy())


# ------------------------------------------------------------------ general term lists, ragged shapes
@pytest.mark.parametrize("N,M,B,T,sigma,seed", [
    (6, 5, 64, 40, 0.3, 101),      # all 2^N states, every Pauli type, complex coefficients
    (9, 17, 77, 60, 0.2, 102),     # ragged: B, M not multiples of any tile
    (13, 7, 257, 90, 0.2, 103),
    (33, 40, 515, 200, 0.05, 104),
    (70, 33, 300, 400, 0.03, 105),  # > 16*5 columns: several column tiles + ragged tail
])
def test_random_terms_vs_definition(nqs, oracle, N, M, B, T, sigma, seed):
    w = wl.make_random(N, M, B, T, sigma, seed)
    e, l = gpu_eloc(nqs, w)
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "definition")
    check_eloc(e, e_ref, f"random N={N}")
    check_logpsi(l, l_ref, f"random N={N}")


def test_pair_flip_both_parities_and_y_terms(nqs, oracle):
    """XX alone needs both parity columns; XY / YX / YY carry the -i s factors."""
    N, M, B = 8, 12, 200
    w = wl.make_random(N, M, B, 1, 0.25, 7)
    rows = []
    for i in range(N):
        k = (i + 3) % N
        rows += [(i, 1, k, 1, 0.7 + 0.1j), (i, 1, k, 2, -0.3j), (i, 2, k, 1, 0.2), (i, 2, k, 2, 1.1)]
    rows += [(2, 2, -1, 0, 0.5), (-1, 0, 5, 2, 0.25j), (3, 1, 6, 3, 0.4), (3, 2, 1, 3, -0.6), (-1, 0, -1, 0, 2.5)]
    w.ham = wl._terms(rows)
    e, l = gpu_eloc(nqs, w)
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "definition")
    check_eloc(e, e_ref, "pair flips")
    check_logpsi(l, l_ref, "pair flips")


def test_degenerate_term_lists(nqs, oracle):
    import torch

    w = wl.make_random(10, 6, 50, 5, 0.2, 9)
    spins, a, b, W = to_dev(w)
    # no terms at all: E_loc = 0, log psi still produced
    e, l = nqs.local_energy(spins, a, b, W, np.zeros((0, 2), np.int32), np.zeros((0, 2), np.uint8),
                            np.zeros(0, np.complex64))
    torch.cuda.synchronize()
    assert np.all(e.cpu().numpy() == 0)
    check_logpsi(l.cpu().numpy(), oracle.log_psi(w.spins, w.a, w.b, w.W), "T=0")
    # diagonal only (ZZ, Z, constant)
    ham = wl._terms([(0, 3, 1, 3, -1.0), (4, 3, -1, 0, 0.5 + 0.5j), (-1, 0, -1, 0, 3.0), (2, 0, 7, 0, 1.0)])
    e = nqs.local_energy(spins, a, b, W, ham.sites, ham.paulis, ham.coeffs, want_logpsi=False)
    torch.cuda.synchronize()
    e_ref, _ = oracle.local_energy_definition(w.spins, w.a, w.b, w.W, ham.sites, ham.paulis, ham.coeffs)
    check_eloc(e.cpu().numpy(), e_ref, "diagonal only")
    # B = 0 is a no-op, B = 1 works
    e0 = nqs.local_energy(spins[:0], a, b, W, w.ham.sites, w.ham.paulis, w.ham.coeffs, want_logpsi=False)
    assert e0.numel() == 0
    e1 = nqs.local_energy(spins[:1].contiguous(), a, b, W, w.ham.sites, w.ham.paulis, w.ham.coeffs, want_logpsi=False)
    torch.cuda.synchronize()
    e1_ref, _ = oracle.local_energy_definition(w.spins[:1], w.a, w.b, w.W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    check_eloc(e1.cpu().numpy(), e1_ref, "B=1")


def test_singlet_and_zero_matrix_elements(nqs):
    """P5 on the GPU: E_loc(up,down) = E_loc(down,up) = -3; parallel bonds have element 0."""
    q = 0.25j * np.pi
    ham = wl.heisenberg([(0, 1)])
    e, _ = nqs.local_energy_host(np.array([[1, -1], [-1, 1]], np.int8), np.array([q, -q], np.complex64),
                                 np.zeros(1, np.complex64), np.array([[q, q]], np.complex64), ham.sites, ham.paulis,
                                 ham.coeffs)
    assert np.allclose(e, -3.0, atol=1e-5)


# ------------------------------------------------------------------ enumerator (Eq. 39)
def test_enumerator_against_oracle_connected(nqs, oracle):
    import torch

    w = wl.make_random(11, 4, 40, 70, 0.1, 55)
    ham = nqs.Hamiltonian(w.N, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    spins = torch.from_numpy(w.spins).cuda()
    sp, mel, G = nqs.enumerate_connected(spins, w.ham.sites, w.ham.paulis, w.ham.coeffs)  # SURVEY 8(b) form
    sp_h, mel_h = nqs.enumerate_connected_h(ham, spins)                                   # handle form
    torch.cuda.synchronize()
    assert G == ham.G and torch.equal(sp, sp_h) and torch.equal(mel, mel_h)
    sp, mel = sp.cpu().numpy(), mel.cpu().numpy().astype(np.complex128)
    sp_ref, mel_ref = oracle.connected(w.spins, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    assert sp.shape == (w.B, ham.G + 1, w.N)
    for bidx in range(w.B):
        # aggregate the oracle's term-by-term list by s'
        agg = {}
        for t in range(w.ham.T):
            key = sp_ref[bidx, t].tobytes()
            agg[key] = agg.get(key, 0) + mel_ref[bidx, t]
        seen = set()
        for slot in range(ham.G + 1):
            key = sp[bidx, slot].tobytes()
            assert key not in seen, "two slots reach the same s'"
            seen.add(key)
            assert abs(agg.get(key, 0) - mel[bidx, slot]) <= 1e-5 * max(1, abs(agg.get(key, 0)))
        assert set(agg) <= seen
    # bit-exact index work: slot 0 is s itself, slot 1+g flips exactly the group's sites
    assert np.array_equal(sp[:, 0, :], w.spins)
    for g, (f0, f1) in enumerate(ham.flip_sites):
        diff = sp[:, 1 + g, :] != w.spins
        expect = np.zeros(w.N, bool)
        expect[f0] = True
        if f1 >= 0:
            expect[f1] = True
        assert np.array_equal(diff, np.broadcast_to(expect, diff.shape))


# ------------------------------------------------------------------ robustness set (pin P10)
def test_p10_sigma_0p1_full_tolerance(nqs, oracle):
    w = wl.make_robustness(0.1, B=256)
    e, l = gpu_eloc(nqs, w)
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "fast")
    check_eloc(e, e_ref, "P10 sigma=0.1")
    check_logpsi(l, l_ref, "P10 sigma=0.1")


@pytest.mark.parametrize("sigma", [0.3, 0.5])
def test_p10_large_parameters_finite_and_close(nqs, oracle, sigma):
    w = wl.make_robustness(sigma, B=128)
    e, l = gpu_eloc(nqs, w)
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "fast")
    assert np.all(np.isfinite(e.view(np.float32)))
    rel = np.abs(e.astype(np.complex128) - e_ref) / np.maximum(1.0, np.abs(e_ref))
    assert rel.max() <= 1e-3, f"relative error {rel.max():.3e}"
    check_logpsi(l, l_ref, f"P10 sigma={sigma}", rtol=1e-4)


def test_running_product_range_safety(nqs, oracle):
    """M = 1600 hidden units with |W| large enough that prod_j |r_j| leaves the float32 range."""
    w = wl.make_config(5, B=64, sigma=0.12, seed=77)
    e, l = gpu_eloc(nqs, w)
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "fast")
    assert np.all(np.isfinite(e.view(np.float32)))
    rel = np.abs(e.astype(np.complex128) - e_ref) / np.maximum(1.0, np.abs(e_ref))
    assert rel.max() <= 1e-3, f"relative error {rel.max():.3e}"


# ------------------------------------------------------------------ API behaviour
def test_determinism_and_handle_api(nqs):
    import torch

    w = wl.make_config(3, B=3000)
    spins, a, b, W = to_dev(w)
    ham = nqs.Hamiltonian(w.N, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    e1, l1 = ham.local_energy(spins, a, b, W)
    e2, l2 = ham.local_energy(spins, a, b, W)
    e3, l3 = nqs.local_energy(spins, a, b, W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    torch.cuda.synchronize()
    assert torch.equal(e1, e2) and torch.equal(l1, l2)  # run-to-run deterministic (reading Q16)
    assert torch.equal(e1, e3) and torch.equal(l1, l3)
    eh, lh = nqs.local_energy_host(w.spins, w.a, w.b, w.W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    assert np.array_equal(eh, e1.cpu().numpy()) and np.array_equal(lh, l1.cpu().numpy())


def test_host_entry_point_in_chunks(nqs, oracle):
    """nqs_local_energy_host sends large batches through the device in chunks (copy of chunk k + 1 under the kernels of
    chunk k).  Every sample is independent, so 1, 2, 3 and 5 chunks of a ragged batch (pageable and pinned host
    buffers) must give the bits of the device-pointer call of each chunk; sampled outputs against the oracle."""
    import torch

    w = wl.make_config(3, B=70001)
    pin = lambda x: torch.from_numpy(x).pin_memory().numpy()  # noqa: E731
    bufs = {"pageable": (w.spins, w.a, w.b, w.W), "pinned": tuple(pin(x) for x in (w.spins, w.a, w.b, w.W))}
    out = {}
    try:
        for kind, (hs, ha, hb, hW) in bufs.items():
            for ch in (1, 2, 3, 5, 0):
                nqs.set_option("host_chunks", ch)
                out[kind, ch] = nqs.local_energy_host(hs, ha, hb, hW, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    finally:
        nqs.set_option("host_chunks", 0)
    e1, l1 = out["pageable", 1]
    for key, (e, l) in out.items():
        assert np.array_equal(e, e1) and np.array_equal(l, l1), key
    spins, a, b, W = to_dev(w)
    ed, ld = nqs.local_energy(spins, a, b, W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    assert np.array_equal(e1, ed.cpu().numpy()) and np.array_equal(l1, ld.cpu().numpy())
    idx = np.unique(np.concatenate([np.arange(0, 70001, 997), [35071, 35072, 35073, 69999, 70000]]))
    e_ref, l_ref = oracle.local_energy_fast(w.spins[idx], w.a, w.b, w.W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    tol = 1e-4 * np.maximum(1, np.abs(e_ref))
    assert np.all(np.abs(e1[idx].real - e_ref.real) <= tol) and np.all(np.abs(e1[idx].imag - e_ref.imag) <= tol)


def test_non_default_stream(nqs, oracle):
    import torch

    w = wl.make_config(2, B=512)
    spins, a, b, W = to_dev(w)
    st = torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(st):
        e, l = nqs.local_energy(spins, a, b, W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    st.synchronize()
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "fast")
    check_eloc(e.cpu().numpy(), e_ref, "stream")


def test_cached_hamiltonian_shared_between_streams(nqs, oracle):
    """a term list compiled on a cache miss is uploaded in the order of the stream that missed.  A hit
    from ANOTHER (non-blocking) stream must wait for that upload, and an eviction must wait for the readers on every
    stream.  Miss on s1 behind a long-running kernel, immediate hit on s2, then nine other term lists push the entry
    out while both streams still hold work."""
    import torch

    w = wl.make_config(3, B=4096)
    coeffs = (w.ham.coeffs * np.complex64(1.25 - 0.5j)).astype(np.complex64)  # a term list no other test has cached
    spins, a, b, W = to_dev(w)
    small = wl.make_config(1)
    sp1, a1, b1, W1 = to_dev(small)
    nqs.release()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(s1):
        torch.cuda._sleep(400_000_000)  # ~0.2 s: the upload of the miss below is still pending when s2 hits
        e1, l1 = nqs.local_energy(spins, a, b, W, w.ham.sites, w.ham.paulis, coeffs)
    with torch.cuda.stream(s2):
        e2, l2 = nqs.local_energy(spins, a, b, W, w.ham.sites, w.ham.paulis, coeffs)
        for k in range(9):  # the cache holds eight entries
            nqs.local_energy(sp1, a1, b1, W1, small.ham.sites, small.ham.paulis,
                             (small.ham.coeffs * np.complex64(2.0 + k)).astype(np.complex64))
    with torch.cuda.stream(s1):
        e3, _ = nqs.local_energy(spins, a, b, W, w.ham.sites, w.ham.paulis, coeffs)  # a miss again: recompiled
    torch.cuda.synchronize()
    e_ref, l_ref = oracle.local_energy_fast(w.spins, w.a, w.b, w.W, w.ham.sites, w.ham.paulis, coeffs)
    check_eloc(e1.cpu().numpy(), e_ref, "miss on s1")
    check_logpsi(l1.cpu().numpy(), l_ref, "miss on s1")
    assert torch.equal(e1, e2) and torch.equal(l1, l2) and torch.equal(e1, e3)


def test_error_codes(nqs):
    import torch

    w = wl.make_config(1)
    spins, a, b, W = to_dev(w)
    with pytest.raises(nqs.NqsError) as ei:
        nqs.local_energy(spins, a, b, W, [[0, 99]], [[3, 3]], [1.0])
    assert ei.value.code == -2
    with pytest.raises(nqs.NqsError) as ei:
        nqs.local_energy(spins, a, b, W, [[0, 1]], [[3, 7]], [1.0])
    assert ei.value.code == -2
    with pytest.raises(nqs.NqsError) as ei:
        nqs.local_energy(spins, a, b, W, [[-1, 1]], [[3, 3]], [1.0])
    assert ei.value.code == -2
    host = nqs.Hamiltonian(w.N, w.ham.sites, w.ham.paulis, w.ham.coeffs, host_only=True)
    with pytest.raises(nqs.NqsError) as ei:
        host.local_energy(spins, a, b, W)
    assert ei.value.code == -1
    torch.cuda.synchronize()


def test_large_N_takes_the_simt_theta_kernel(nqs, oracle):
    """N > 512 is outside the tensor-core theta kernel (its spins tile lives in shared memory); the
    FP32 SIMT theta_kernel takes over.  Same tolerances; also through nqs_log_psi alone."""
    import torch

    N, M, B = 530, 48, 300
    a, b, W = wl.rbm_parameters(N, M, 0.03, [91, 0])
    ham = wl.tfim(wl.chain_bonds(N), N, 1.0, 0.8)
    spins = wl.iid_spins(B, N, [91, 1])
    w = wl.Workload("chain_N530", N, M, B, spins, a, b, W, ham)
    e, l = gpu_eloc(nqs, w)
    e_ref, l_ref = oracle.local_energy_fast(w.spins, w.a, w.b, w.W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    check_eloc(e, e_ref, "N=530")
    check_logpsi(l, l_ref, "N=530")
    sp, ad, bd, Wd = to_dev(w)
    l2 = nqs.log_psi(sp, ad, bd, Wd)
    torch.cuda.synchronize()
    check_logpsi(l2.cpu().numpy(), l_ref, "N=530 nqs_log_psi")


def test_nqs_validate_rejects_bad_spin_values(nqs, monkeypatch):
    """spin values other than +1/-1 are undefined behaviour in release and checked when NQS_VALIDATE=1
    (read at every call): every device entry point that takes spins then returns NQS_ERR_INVALID_ARG."""
    import torch

    w = wl.make_config(2, B=300)
    spins, a, b, W = to_dev(w)
    bad = spins.clone()
    bad[17, 5] = 0
    bad[200, 39] = 3
    monkeypatch.setenv("NQS_VALIDATE", "1")
    e, l = nqs.local_energy(spins, a, b, W, w.ham.sites, w.ham.paulis, w.ham.coeffs)  # valid spins pass
    torch.cuda.synchronize()
    for call in (lambda: nqs.local_energy(bad, a, b, W, w.ham.sites, w.ham.paulis, w.ham.coeffs),
                 lambda: nqs.log_psi(bad, a, b, W),
                 lambda: nqs.metropolis(bad.clone(), a, b, W, torch.zeros((1, w.B), dtype=torch.int32, device=bad.device),
                                        torch.zeros((1, w.B), dtype=torch.float32, device=bad.device))):
        with pytest.raises(nqs.NqsError) as ei:
            call()
        assert ei.value.code == -1 and "2 spin values" in str(ei.value)
    monkeypatch.delenv("NQS_VALIDATE")
    nqs.log_psi(bad, a, b, W)  # release mode: not checked (undefined values, no error)
    torch.cuda.synchronize()


def test_two_devices_in_one_process(nqs, oracle):
    """ADVICE (round 1): kernel attributes and the scratch pool are per device.  Needs two GPUs; skipped otherwise."""
    import torch

    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices in one process")
    w = wl.make_config(3, B=4096)
    e_ref, _ = oracle_on(oracle, w, np.arange(0, w.B, 64), "fast")
    for dev in (0, 1):
        d = torch.device("cuda", dev)
        with torch.cuda.device(d):
            args = [torch.from_numpy(x).to(d) for x in (w.spins, w.a, w.b, w.W)]
            e, _ = nqs.local_energy(*args, w.ham.sites, w.ham.paulis, w.ham.coeffs)
            F = nqs.forces(*args, e)
            torch.cuda.synchronize(d)
            check_eloc(e.cpu().numpy()[::64], e_ref, f"device {dev}")
            assert torch.isfinite(torch.view_as_real(F)).all()
