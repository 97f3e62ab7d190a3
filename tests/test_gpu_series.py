"""The guarded tensor-core series path of step a5 (csrc/nqs_series.cuh) against the
float64 oracle, through the C ABI.

  log psi(s')/psi(s) = log kappa_c - 2 sigma A_c - sigma ODD - EVEN,  truncated at k = 3, FP16 operands
  (hi + lo split for k = 1) on tcgen05 with FP32 accumulators, and a per-sample a-posteriori error bound
  (the guard) that sends the whole call back to the FP32 product form when it exceeds
  0.5e-4 max(1, |E_loc|).

Tolerances are the hot path's (north_star): |Re dE|, |Im dE| <= 1e-4 max(1, |E_loc|) per sample.
nqs_set_option(NQS_OPT_A5_PATH): 2 = series + guard + fallback at any size, 3 = series only (the guard is
recorded, nothing is recomputed) -- the latter is how the guard's SUFFICIENCY is tested: whenever the guard
passes, the series result alone must already meet the tolerance.
"""
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


@pytest.mark.parametrize("N,M,B,T,sigma,seed", [
    (6, 5, 64, 40, 0.02, 301),      # all 2^N states; every Pauli type, complex coefficients; M, C ragged
    (9, 17, 77, 60, 0.02, 302),     # B not a multiple of the 128-sample tile
    (13, 7, 257, 90, 0.01, 303),    # three sample tiles, the last one with one live row
    (33, 40, 515, 200, 0.003, 304),  # > 128 columns: two column tiles
    (70, 33, 300, 700, 0.001, 305),  # many pair-flip groups, both parities
])
@pytest.mark.parametrize("narrow_only", [0, 1])
def test_series_only_random_terms_vs_definition(nqs, oracle, N, M, B, T, sigma, seed, narrow_only):
    """Small parameters (inside the guard), general term lists: the series kernel ALONE (no fallback) against
    definition mode -- matrix elements, parities, diagonal, ragged tiles; with the default tiling (wide two-pass
    column tiles where there are more than 128 columns) and with narrow tiles only.  (Random complex coefficients
    make sum |m| large against |E_loc|, so the guard is strict here: sigma is chosen small.)"""
    w = wl.make_random(N, M, B, T, sigma, seed)
    nqs.set_option("series_wide", narrow_only)
    try:
        e, l, took = run(nqs, w, "series_only")
    finally:
        nqs.set_option("series_wide", 0)
    assert took["path"] == "series" and not took["guard_failed"], took
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "definition")
    check_eloc(e, e_ref, f"series N={N}")
    check_logpsi(l, l_ref, f"series N={N}")


def test_series_pair_flip_parities_and_y_terms(nqs, oracle):
    N, M, B = 8, 12, 200
    w = wl.make_random(N, M, B, 1, 0.02, 7)
    rows = []
    for i in range(N):
        k = (i + 3) % N
        rows += [(i, 1, k, 1, 0.7 + 0.1j), (i, 1, k, 2, -0.3j), (i, 2, k, 1, 0.2), (i, 2, k, 2, 1.1)]
    rows += [(2, 2, -1, 0, 0.5), (-1, 0, 5, 2, 0.25j), (3, 1, 6, 3, 0.4), (3, 2, 1, 3, -0.6), (-1, 0, -1, 0, 2.5)]
    w.ham = wl._terms(rows)
    e, l, took = run(nqs, w, "series_only")
    assert took["path"] == "series" and not took["guard_failed"], took
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "definition")
    check_eloc(e, e_ref, "series pair flips")


@pytest.mark.parametrize("sigma", [0.1, 0.3, 0.5])
def test_p10_takes_the_fallback(nqs, oracle, sigma):
    """Pin P10 (large parameters): the guard must refuse the series and the product form must answer."""
    w = wl.make_robustness(sigma, B=256 if sigma == 0.1 else 128)  # the sizes of the P10 cases in test_gpu_parity
    e, l, took = run(nqs, w, "series_guarded")
    assert took["path"] == "series" and took["guard_failed"] and took["samples_over"] > 0, took
    e_prod, _, took_p = run(nqs, w, "product")
    assert took_p["path"] == "product"
    assert np.array_equal(e, e_prod)  # the fallback IS the product-form result, bit for bit
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "fast")
    if sigma == 0.1:
        check_eloc(e, e_ref, "P10 sigma=0.1 via fallback")
    else:
        rel = np.abs(e.astype(np.complex128) - e_ref) / np.maximum(1.0, np.abs(e_ref))
        assert np.all(np.isfinite(e.view(np.float32))) and rel.max() <= 1e-3


def test_guard_boundary_inside_and_outside(nqs, oracle):
    """Config-3 shapes with growing parameter scale.  The guard decision must be monotone in sigma; wherever it
    PASSES, the series alone meets the tolerance (sufficiency: checked with the fallback disabled); outside,
    the guarded call returns the product form's result bit for bit (which meets the full tolerance up to
    sigma = 0.04 here; beyond that E_loc is a cancelling sum of large ratios and float32 is only asked for 1e-3,
    as in pin P10)."""
    sigmas = [0.01, 0.014, 0.02, 0.028, 0.04, 0.056, 0.08]
    passed = []
    for sg in sigmas:
        w = wl.make_config(3, B=384, sigma=sg, seed=31)
        e_ref, l_ref = oracle_on(oracle, w, slice(None), "fast")
        e3, _, took3 = run(nqs, w, "series_only")
        passed.append(not took3["guard_failed"])
        if passed[-1]:
            check_eloc(e3, e_ref, f"series only, sigma={sg} (guard passed)")
        e2, _, took2 = run(nqs, w, "series_guarded")
        assert took2["guard_failed"] == took3["guard_failed"]
        if took2["guard_failed"]:
            ep, _, _ = run(nqs, w, "product")
            assert np.array_equal(e2, ep), f"sigma={sg}: the fallback is not the product-form result"
        check_eloc(e2, e_ref, f"guarded, sigma={sg}", rtol=1e-4 if sg <= 0.04 else 1e-3)
    assert passed[0], "config 3's own sigma must be inside the guard"
    assert not passed[-1], "sigma = 0.08 at M = 400 must be outside the guard"
    first_fail = passed.index(False)
    assert not any(passed[first_fail:]), f"guard decision is not monotone in sigma: {list(zip(sigmas, passed))}"


def test_series_is_deterministic_and_matches_product_within_tolerance(nqs, oracle):
    import torch

    w = wl.make_config(3, B=3000)
    e1, l1, t1 = run(nqs, w, "series_only")
    e2, l2, t2 = run(nqs, w, "series_only")
    assert np.array_equal(e1, e2) and np.array_equal(l1, l2)
    ep, lp, _ = run(nqs, w, "product")
    assert np.array_equal(l1, lp)  # log psi does not depend on the a5 path
    tol = 1e-4 * np.maximum(1.0, np.abs(ep))
    assert np.all(np.abs(e1.real - ep.real) <= 2 * tol) and np.all(np.abs(e1.imag - ep.imag) <= 2 * tol)
    torch.cuda.synchronize()


def test_auto_threshold(nqs):
    """Automatic choice: small problems stay on the product form (the series' packing does not pay below
    2^28 triples), large ones take the series."""
    w = wl.make_config(2, B=2000)
    _, _, took = run(nqs, w, "auto")
    assert took["path"] == "small"  # the single-launch kernel (tests/test_gpu_small.py)
    w = wl.make_config(3, B=500)    # tables too large for it: the multi-launch product form
    _, _, took = run(nqs, w, "auto")
    assert took["path"] == "product"
    w = wl.make_config(3, B=8192)  # 8192 * 100 * 400 = 3.3e8 >= 2^28
    _, _, took = run(nqs, w, "auto")
    assert took["path"] == "series" and not took["guard_failed"]


def test_series_with_the_simt_theta_kernel(nqs, oracle):
    """N > 512 is outside the tensor-core theta kernel: theta_kernel (FP32 SIMT) writes tanh(theta) and
    series_pack_kernel builds the FP16 planes and the row norms from it; also through the NQS_OPT_THETA_PATH switch
    at a size both theta kernels cover (the two ways to the planes must agree within the tolerance)."""
    N, M, B = 530, 48, 300
    a, b, W = wl.rbm_parameters(N, M, 0.004, [92, 0])
    ham = wl.tfim(wl.chain_bonds(N), N, 1.0, 0.8)
    w = wl.Workload("chain_N530", N, M, B, wl.iid_spins(B, N, [92, 1]), a, b, W, ham)
    e, l, took = run(nqs, w, "series_only")
    assert took["path"] == "series" and not took["guard_failed"], took
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "fast")
    check_eloc(e, e_ref, "series, N=530")
    check_logpsi(l, l_ref, "series, N=530")
    w3 = wl.make_config(3, B=700)
    e_ref, l_ref = oracle_on(oracle, w3, slice(None), "fast")
    nqs.set_option("theta_path", 1)
    try:
        e1, l1, took = run(nqs, w3, "series_only")
    finally:
        nqs.set_option("theta_path", 0)
    assert took["path"] == "series" and not took["guard_failed"], took
    check_eloc(e1, e_ref, "series, SIMT theta, config 3")
    check_logpsi(l1, l_ref, "series, SIMT theta, config 3")


def test_theta_split_over_ctas(nqs, oracle):
    """On the series path the hidden-unit tiles of a sample tile are split over S CTAs of the theta kernel (S chosen
    for whole waves; partial log psi and row norms combined in a fixed order).  The operand planes do not depend on the
    split, so E_loc must have the same bits as with NQS_OPT_THETA_SPLIT = 1; log psi is the same float64 sum in another
    order (<= 1 ulp of the float32 result) and is checked against the oracle either way; deterministic run to run."""
    for k, B in ((5, 2000), (3, 4500), (4, 1300)):   # 16 / 36 / 11 sample tiles: S = 8, 8, 8 resp. what fits M
        w = wl.make_config(k, B=B)
        e_ref, l_ref = oracle_on(oracle, w, slice(None), "fast")
        out = {}
        for split in (1, 0, 0):
            nqs.set_option("theta_split", split)
            try:
                e, l, took = run(nqs, w, "series_only")
            finally:
                nqs.set_option("theta_split", 0)
            assert took["path"] == "series" and not took["guard_failed"], took
            check_logpsi(l, l_ref, f"c{k} theta_split={split}")
            out.setdefault(split, []).append((e, l))
        (e1, l1), = out[1]
        (e0, l0), (e0b, l0b) = out[0]
        check_eloc(e0, e_ref, f"c{k} split")
        assert np.array_equal(e1, e0), "E_loc must not depend on the split of the theta kernel"
        assert np.array_equal(e0, e0b) and np.array_equal(l0, l0b), "run-to-run determinism"
        assert np.abs(l1 - l0).max() <= 2e-7 * max(1.0, np.abs(l_ref).max())


def test_wide_column_tiles(nqs, oracle):
    """More than 128 table columns: the series GEMM tiles them in column tiles of up to 224 and makes two passes over the
    hidden units (EVEN, parked in a scratch array, then ODD) with one accumulator pair in TMEM at a time.  Every
    accumulator element sees the same addends in the same order as with tiles of <= 128 columns (NQS_OPT_SERIES_WIDE =
    1); only the order in which a row's columns are summed changes with the tiling, so the two agree to float32
    rounding of that sum (not bit for bit) and each is judged against the oracle: TFIM (affine columns), Heisenberg
    pair flips, a ragged batch; deterministic run to run."""
    for k, B in ((5, 1000), (4, 777), (5, 129)):
        w = wl.make_config(k, B=B)
        e_ref, l_ref = oracle_on(oracle, w, slice(None), "fast")
        out = {}
        for mode in (1, 0, 0):
            nqs.set_option("series_wide", mode)
            try:
                e, l, took = run(nqs, w, "series_only")
            finally:
                nqs.set_option("series_wide", 0)
            assert took["path"] == "series" and not took["guard_failed"]
            check_eloc(e, e_ref, f"c{k} B={B} series_wide={mode}")
            out.setdefault(mode, []).append(e)
        assert np.array_equal(out[0][0], out[0][1]), "run-to-run determinism"
        scale = np.abs(e_ref).max()
        assert np.abs(out[1][0] - out[0][0]).max() <= 4e-6 * scale, (k, B, np.abs(out[1][0] - out[0][0]).max(), scale)


def test_refusal_latch_skips_the_series_after_a_refused_call(nqs, oracle):
    """ADVICE / VERDICT round 2: in automatic mode a handle remembers that the guard refused its series.  Config-3 shapes
    at trained-scale parameters (sigma = 0.05, far outside the guard's window), B large enough for the automatic path to
    choose the series: call 1 attempts it and is refused; the next 8 calls enqueue the product form alone; call 10
    probes again, is refused again, and 16 product-only calls follow.  Every call returns the product-form bits.  A
    fresh handle with in-window parameters is untouched, and NQS_OPT_SERIES_LATCH = 1 restores an attempt per call."""
    import torch

    from test_gpu_parity import to_dev

    w = wl.make_config(3, B=8192, sigma=0.05, seed=77)
    spins, a, b, W = to_dev(w)
    e_prod, _, took = run(nqs, w, "product")
    assert took["path"] == "product"
    ham = nqs.Hamiltonian(w.N, w.ham.sites, w.ham.paulis, w.ham.coeffs)  # a fresh handle: a fresh latch
    paths, launches = [], []
    for call in range(27):
        n0 = nqs.launch_count()
        e, _ = ham.local_energy(spins, a, b, W)
        launches.append(nqs.launch_count() - n0)
        took = nqs.debug_last_a5()  # synchronises: the latch record of this call has landed
        paths.append(took["path"] + ("!" if took["guard_failed"] else ""))
        assert np.array_equal(e.cpu().numpy(), e_prod), f"call {call}"
    assert paths == ["series!"] + ["product"] * 8 + ["series!"] + ["product"] * 16 + ["series!"], paths
    assert max(launches[1:9]) < launches[0] and len(set(launches[1:9])) == 1, launches
    # without the latch every call attempts the series
    nqs.set_option("series_latch", 1)
    try:
        for _ in range(3):
            ham.local_energy(spins, a, b, W)
            took = nqs.debug_last_a5()
            assert took["path"] == "series" and took["guard_failed"], took
    finally:
        nqs.set_option("series_latch", 0)
    # the latch belongs to the handle: still refusing here ...
    ham.local_energy(spins, a, b, W)
    assert nqs.debug_last_a5()["path"] == "product"
    ham.close()
    # ... while another handle, with parameters inside the window, takes the series at once and keeps taking it
    w_ok = wl.make_config(3, B=8192)
    ham2 = nqs.Hamiltonian(w_ok.N, w_ok.ham.sites, w_ok.ham.paulis, w_ok.ham.coeffs)
    s2, a2, b2, W2 = to_dev(w_ok)
    for _ in range(3):
        e2, _ = ham2.local_energy(s2, a2, b2, W2)
        took = nqs.debug_last_a5()
        assert took["path"] == "series" and not took["guard_failed"], took
    ham2.close()
    idx = np.arange(0, w_ok.B, 64)
    e_ref, _ = oracle_on(oracle, w_ok, idx, "fast")
    check_eloc(e2.cpu().numpy()[idx], e_ref, "in-window handle")
    torch.cuda.synchronize()


@pytest.mark.parametrize("M", [4096, 8192])
def test_same_sign_accumulation_at_the_guard_boundary(nqs, oracle, M):
    """ADVICE / VERDICT round 2: the guard bounds truncation and FP16 operand rounding, not the FP32 accumulation of the
    tensor cores, which truncates and drifts on same-sign chains (csrc/nqs_fisher.cuh met it).  Purely REAL a, b, W make
    the EVEN sum  sum_j t_j^2 T_jc^2 / 2  such a chain -- every term >= 0 -- and M = 4096 / 8192 hidden units make it
    256 / 512 MMA steps long.  sigma walks down a ladder; at the LARGEST sigma the guard passes, the series alone (no
    fallback) must meet the hot path's tolerance against the float64 oracle, with half of it to spare for the
    accumulation as DESIGN.md section 12 assumes."""
    N, B = 64, 256
    ham = wl.tfim(wl.chain_bonds(N), N, 1.0, 1.0)
    spins = wl.iid_spins(B, N, [401, 1])
    passed = None
    for sigma in (0.02, 0.014, 0.01, 0.007, 0.005, 0.0035, 0.0025):
        a, b, W = wl.rbm_parameters(N, M, sigma, [401, M])
        a, b, W = (np.ascontiguousarray(x.real.astype(np.float32)).astype(np.complex64) for x in (a, b, W))
        w = wl.Workload(f"real_chain_N64_M{M}_sigma{sigma}", N, M, B, spins, a, b, np.ascontiguousarray(W), ham)
        e, l, took = run(nqs, w, "series_only")
        assert took["path"] == "series"
        if not took["guard_failed"]:
            passed = (sigma, w, e, l)
            break
    assert passed is not None, "the guard refused every sigma of the ladder"
    sigma, w, e, l = passed
    e_ref, l_ref = oracle_on(oracle, w, slice(None), "fast")
    worst = check_eloc(e, e_ref, f"real parameters, M = {M}, sigma = {sigma}")
    check_logpsi(l, l_ref, f"real parameters, M = {M}")
    print(f"M = {M}: guard passes at sigma = {sigma}; series error = {worst:.3f} x tolerance")
    assert worst <= 0.75, f"accumulation leaves too little of the tolerance: {worst:.3f}"
