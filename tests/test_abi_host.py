"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/nqs.h declares,
and its host logic (Hamiltonian compile: validation + flip grouping, step a0) is right.
No compute entry point is exercised here beyond its no-device error path."""
import ctypes
import os
import re

import numpy as np
import pytest

import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def nqs():
    from paper_2108_03409_b200 import build

    build.build()
    import paper_2108_03409_b200 as m

    m.load_library()
    return m


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "nqs.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(nqs_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(nqs):
    lib = ctypes.CDLL(nqs.lib_path())
    names = declared_symbols()
    assert {"nqs_log_psi", "nqs_local_energy", "nqs_local_energy_host", "nqs_last_error"} <= set(names)
    for name in names:
        assert hasattr(lib, name), f"{name} is declared in include/nqs.h but not exported"
    assert nqs.version().endswith("sm_100a")


def test_binding_covers_every_declared_symbol(nqs):
    """binding.py sets argtypes/restype for every entry point (a typo there is silent in ctypes)."""
    src = open(os.path.join(ROOT, "paper_2108_03409_b200", "binding.py")).read()
    for name in declared_symbols():
        assert name in src, f"{name} has no binding"


def test_product_package_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_2108_03409_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.lower(), f"{f} mentions the oracle"


@pytest.mark.parametrize("k,G,C,n_diag,n_grp", [(1, 8, 8, 8, 8), (2, 40, 40, 40, 40), (3, 100, 100, 200, 100),
                                                  (4, 200, 200, 200, 400), (5, 400, 400, 800, 400)])
def test_compile_counts_of_the_five_configs(nqs, k, G, C, n_diag, n_grp):
    spec = wl.config_spec(k)
    w = wl.make_config(k, B=4)
    info = nqs.hamiltonian_info_host(spec["N"], w.ham.sites, w.ham.paulis, w.ham.coeffs)
    assert (info["G"], info["C"], info["n_diag"], info["n_group_terms"]) == (G, C, n_diag, n_grp)
    if k != 4:  # TFIM: group g flips site g only
        assert np.array_equal(info["flip_sites"][:, 0], np.arange(spec["N"]))
        assert np.all(info["flip_sites"][:, 1] == -1)
    else:  # Heisenberg: one group per bond (XX and YY share it), sites sorted
        bonds = np.sort(np.array(wl.square_bonds(10), dtype=np.int32), axis=1)
        assert np.array_equal(info["flip_sites"], bonds)


def test_compile_groups_by_flip_set_in_order_of_first_appearance(nqs):
    X, Y, Z, I = wl.PAULI_X, wl.PAULI_Y, wl.PAULI_Z, wl.PAULI_I
    rows = [(3, X, 1, Y, 1.0),      # flips {1,3}
            (2, Z, -1, I, 0.5),     # diagonal
            (-1, I, 0, X, 2.0),     # flips {0}, site in slot 1
            (1, X, 3, X, 1j),       # flips {1,3} again (other slot order)
            (0, Y, 2, Z, -1.0),     # flips {0}: Z on 2 rides along
            (-1, I, -1, I, 7.0),    # constant
            (0, I, 4, Z, 1.0)]      # identity on a real site + Z: diagonal
    ham = wl._terms(rows)
    info = nqs.hamiltonian_info_host(5, ham.sites, ham.paulis, ham.coeffs)
    assert info["G"] == 2 and info["n_diag"] == 3 and info["n_group_terms"] == 4
    assert info["flip_sites"].tolist() == [[1, 3], [0, -1]]
    # X1Y3 + i X1X3: element c1*(-i s3) + i -> never identically zero for either parity -> 2 columns
    assert info["C"] == 3


def test_pair_group_emits_only_parities_with_nonzero_element(nqs):
    X, Y = wl.PAULI_X, wl.PAULI_Y
    # XX + YY: element 1 - s_i s_k -> zero for parallel spins: one column (antiparallel parity)
    ham = wl._terms([(0, X, 1, X, 1.0), (0, Y, 1, Y, 1.0)])
    assert nqs.hamiltonian_info_host(2, ham.sites, ham.paulis, ham.coeffs)["C"] == 1
    # XX - YY: element 1 + s_i s_k -> zero for antiparallel: one column
    ham = wl._terms([(0, X, 1, X, 1.0), (0, Y, 1, Y, -1.0)])
    assert nqs.hamiltonian_info_host(2, ham.sites, ham.paulis, ham.coeffs)["C"] == 1
    # XX alone: both parities
    ham = wl._terms([(0, X, 1, X, 1.0)])
    assert nqs.hamiltonian_info_host(2, ham.sites, ham.paulis, ham.coeffs)["C"] == 2
    # XX - XX: cancels identically -> no column at all
    ham = wl._terms([(0, X, 1, X, 1.0), (1, X, 0, X, -1.0)])
    info = nqs.hamiltonian_info_host(2, ham.sites, ham.paulis, ham.coeffs)
    assert info["G"] == 1 and info["C"] == 0


@pytest.mark.parametrize("row,what", [((0, 1, 0, 1, 1.0), "same site twice"),
                                      ((5, 1, -1, 0, 1.0), "site out of range"),
                                      ((0, 4, -1, 0, 1.0), "Pauli code > 3"),
                                      ((-1, 1, 0, 0, 1.0), "Pauli on unused slot"),
                                      ((-2, 0, 0, 1, 1.0), "site < -1")])
def test_invalid_terms_are_rejected(nqs, row, what):
    ham = wl._terms([row])
    with pytest.raises(nqs.NqsError) as ei:
        nqs.hamiltonian_info_host(5, ham.sites, ham.paulis, ham.coeffs)
    assert ei.value.code == -2, what
    assert "term 0" in str(ei.value)


def test_empty_term_list_and_bad_sizes(nqs):
    e = np.zeros((0, 2))
    info = nqs.hamiltonian_info_host(3, e.astype(np.int32), e.astype(np.uint8), np.zeros(0, np.complex64))
    assert info["G"] == 0 and info["C"] == 0 and info["n_diag"] == 0
    with pytest.raises(nqs.NqsError) as ei:
        nqs.hamiltonian_info_host(0, e.astype(np.int32), e.astype(np.uint8), np.zeros(0, np.complex64))
    assert ei.value.code == -1


def test_no_cpu_fallback_without_a_device(nqs):
    """On a machine without a GPU every compute entry point fails with NQS_ERR_CUDA."""
    import torch

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    w = wl.make_config(1)
    with pytest.raises(nqs.NqsError) as ei:
        nqs.local_energy_host(w.spins, w.a, w.b, w.W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    assert ei.value.code == -3
    with pytest.raises(nqs.NqsError) as ei:
        nqs.log_psi_host(w.spins, w.a, w.b, w.W)
    assert ei.value.code == -3


def test_missing_library_fails_loudly(nqs, monkeypatch):
    from paper_2108_03409_b200 import binding

    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "_LIB_PATH", "/nonexistent/libnqs_b200.so")
    with pytest.raises(FileNotFoundError):
        binding.load_library()


# ------------------------------------------------------------------ k-site Pauli strings
def test_k_site_strings_compile(nqs):
    X, Y, Z = wl.PAULI_X, wl.PAULI_Y, wl.PAULI_Z
    sites = np.array([[0, 1, 2, -1], [2, 0, 1, -1], [0, 1, 2, 3], [4, 1, -1, 5], [3, 2, 1, 0], [1, 3, -1, -1]], np.int32)
    paulis = np.array([[X, X, X, 0], [Y, X, Y, 0], [Z, Z, Z, Z], [X, Z, 0, Z], [X, Y, X, Y], [Z, X, 0, 0]], np.uint8)
    coeffs = np.array([1.0, 0.5j, -1.0, 2.0, 0.25, 1.0], np.complex64)
    info = nqs.hamiltonian_info_host(6, sites, paulis, coeffs)
    # flip sets: {0,1,2} (terms 0, 1), {} (term 2), {4} (term 3), {0,1,2,3} (term 4), {3} (term 5)
    assert info["G"] == 4 and info["n_diag"] == 1 and info["n_group_terms"] == 5
    assert info["flip_sites4"].tolist() == [[0, 1, 2, -1], [4, -1, -1, -1], [0, 1, 2, 3], [3, -1, -1, -1]]
    # columns: a flip set of m sites has 2^(m-1) relative-sign patterns, dropped only if provably zero:
    #   {0,1,2}: XXX + (i/2) Y X Y over sites (2,0,1): element 1 + (i/2)(-s_2 s_1): never zero -> 4
    #   {4}: 1;  {0,1,2,3}: XYXY alone: element -(s_2 s_0) * 0.25: never zero -> 8;  {3}: 1
    assert info["C"] == 4 + 1 + 8 + 1
    # XXX - XXX cancels identically -> no column; XXX + (XYY over the same sites): 1 - s_1 s_2 -> half the patterns
    s3 = np.array([[0, 1, 2], [0, 1, 2]], np.int32)
    assert nqs.hamiltonian_info_host(3, s3, np.array([[X, X, X], [X, X, X]], np.uint8),
                                     np.array([1.0, -1.0], np.complex64))["C"] == 0
    assert nqs.hamiltonian_info_host(3, s3, np.array([[X, X, X], [X, Y, Y]], np.uint8),
                                     np.array([1.0, 1.0], np.complex64))["C"] == 2


def test_k_site_strings_invalid_and_unsupported(nqs):
    X = wl.PAULI_X
    five = np.array([[0, 1, 2, 3, 4]], np.int32)
    with pytest.raises(nqs.NqsError) as ei:  # five flipping sites: 16 sign columns per group -- not supported
        nqs.hamiltonian_info_host(6, five, np.full((1, 5), X, np.uint8), np.ones(1, np.complex64))
    assert ei.value.code == -4
    with pytest.raises(nqs.NqsError) as ei:  # the same site in slots 0 and 3
        nqs.hamiltonian_info_host(6, np.array([[2, 1, 0, 2]], np.int32), np.full((1, 4), X, np.uint8),
                                  np.ones(1, np.complex64))
    assert ei.value.code == -2
    with pytest.raises(nqs.NqsError) as ei:  # nine slots
        nqs.hamiltonian_info_host(12, np.arange(9, dtype=np.int32)[None, :], np.full((1, 9), 3, np.uint8),
                                  np.ones(1, np.complex64))
    assert ei.value.code == -1


@pytest.mark.parametrize("N,T,K,seed", [(8, 50, 6, 17), (9, 40, 8, 18), (8, 60, 8, 21)])
def test_flip_sets_beyond_four_sites_are_refused_not_miscompiled(nqs, N, T, K, seed):
    """The term lists on which tests/test_oracle_pins.py pins the oracle beyond the kernels' limit (flip sets of five to
    eight sites): the host compiler must answer NQS_ERR_UNSUPPORTED for them -- and accept the same lists once the
    strings with more than four X / Y factors are taken out."""
    ham = wl.random_strings(N, T, K, np.random.default_rng([seed, 3]), max_flips=K)
    n_flips = ((ham.paulis == wl.PAULI_X) | (ham.paulis == wl.PAULI_Y)).sum(axis=1)
    assert n_flips.max() > 4
    with pytest.raises(nqs.NqsError) as ei:
        nqs.hamiltonian_info_host(N, ham.sites, ham.paulis, ham.coeffs)
    assert ei.value.code == -4
    keep = n_flips <= 4
    info = nqs.hamiltonian_info_host(N, ham.sites[keep], ham.paulis[keep], ham.coeffs[keep])
    assert info["G"] >= 1
