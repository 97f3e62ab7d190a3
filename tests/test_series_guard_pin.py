"""CPU pin of the GUARD of the tensor-core series path (csrc/nqs_series.cuh).

The series kernel replaces  log psi(s')/psi(s) = log kappa_c - 2 sigma A_c + sum_j log(1 - sigma t_bj T_jc)
by its Taylor series to k = 3 with FP16 operands (k = 1 split hi + lo), and bounds the error it makes by

    delta_bc = 2 [2^-21 n2t n2T + sqrt(M) (2^-29 n2T + 2^-31 n2t)] + 2^-10 n4t n4T + (2/3) 2^-10 n6t n6T + (1/2) n8t n8T,
    nPt_b = sqrt(sum_j |t_bj|^P),  nPT_c = sqrt(sum_j |T_jc|^P),   valid while max_j |t_bj| max_j |T_jc| <= 1/2,

weighted per sample as  eps_b = sum_c |m_bc R_bc| delta_bc  and compared with 0.5e-4 max(1, |E_loc|).

This file evaluates, in float64 numpy and independently of the CUDA code, (i) the exact log-ratio, (ii) the
truncated series with the same operand roundings (numpy float16, scales 16 / 64 / 2048 as in the kernel; the
accumulation itself in float64, so that what is measured is truncation + operand rounding -- what delta bounds),
and asserts  |exact - series| <= delta_bc  for every (sample, column) inside the validity range; and that the
resulting decision is "series" at the five configurations' parameters (c3, c4-like pairs, c5) and "fallback" on
the robustness set P10 (sigma = 0.1, 0.3, 0.5).  A wrong power, a missing 1/k, a wrong norm or scale in the
formula fails the bound on one of these sets.
"""
import numpy as np
import pytest

import workloads as wl

SA, SB1, SB2 = 16.0, 64.0, 2048.0


def f16(x):
    return x.astype(np.float16).astype(np.float64)


def split16(x):
    hi = f16(x)
    return hi, f16(x - hi)


def series_vs_exact(w, nb, cols):
    """Single-flip columns `cols` (sites) of the first nb samples: exact log R, series log R, delta, |m R| data."""
    s = w.spins[:nb].astype(np.float64)
    W = w.W.astype(np.complex128)
    a = w.a.astype(np.complex128)
    theta = s @ W.T + w.b.astype(np.complex128)[None, :]                      # [nb, M]
    # what the kernels hold: t and T as float32 complex numbers
    t = np.tanh(theta).astype(np.complex64).astype(np.complex128)
    T = np.tanh(2.0 * W[:, cols]).astype(np.complex64).astype(np.complex128)    # [M, C]
    sig = s[:, cols]                                                            # [nb, C]
    # exact: sum_j [lncosh(theta_j - 2 sigma W_jc) - lncosh(theta_j)] - 2 sigma a_c
    exact = np.empty((nb, len(cols)), np.complex128)
    for k, c in enumerate(cols):
        thp = theta - 2.0 * sig[:, k:k + 1] * W[None, :, c]
        exact[:, k] = (np.log(np.cosh(thp)) - np.log(np.cosh(theta))).sum(axis=1) - 2.0 * sig[:, k] * a[c]
    # series with the kernel's operand roundings
    def planes(z, scale):
        return f16(z.real * scale) + 1j * f16(z.imag * scale)
    th_r, tl_r = split16(t.real * SA)
    th_i, tl_i = split16(t.imag * SA)
    Th_r, Tl_r = split16(T.real * SB1)
    Th_i, Tl_i = split16(T.imag * SB1)
    thi, tlo, Thi, Tlo = th_r + 1j * th_i, tl_r + 1j * tl_i, Th_r + 1j * Th_i, Tl_r + 1j * Tl_i
    odd = (thi @ Thi + thi @ Tlo + tlo @ Thi + planes(t ** 3, SA) @ planes(T ** 3 / 3.0, SB1)) / (SA * SB1)
    even = (planes(t ** 2, SA) @ planes(T ** 2 / 2.0, SB2)) / (SA * SB2)
    logk = np.log(np.cosh(2.0 * W[:, cols])).sum(axis=0)
    series = logk[None, :] - sig * (2.0 * a[cols][None, :] + odd) - even
    # the guard's bound
    M = W.shape[0]
    nt = lambda P: np.sqrt((np.abs(t) ** P).sum(axis=1))[:, None]   # noqa: E731
    nT = lambda P: np.sqrt((np.abs(T) ** P).sum(axis=0))[None, :]   # noqa: E731
    delta = (2.0 * (2.0 ** -21 * nt(2) * nT(2) + np.sqrt(M) * (2.0 ** -29 * nT(2) + 2.0 ** -31 * nt(2)))
             + 2.0 ** -10 * nt(4) * nT(4) + (2.0 / 3.0) * 2.0 ** -10 * nt(6) * nT(6) + 0.5 * nt(8) * nT(8))
    X = np.abs(t).max(axis=1)[:, None] * np.abs(T).max(axis=0)[None, :]
    return exact, series, delta, X


def tfim_guard(w, nb):
    """Per-sample guard decision for a TFIM workload (all single flips, element -h, diagonal from Z Z bonds)."""
    N = w.N
    exact, series, delta, X = series_vs_exact(w, nb, list(range(N)))
    h = w.meta.get("h", None)
    spec = wl.config_spec(w.meta["config"])
    h, J = spec["h"], spec["J"]
    R = np.exp(exact)
    s = w.spins[:nb].astype(np.float64)
    bonds = wl.square_bonds(spec["L"]) if spec["lattice"] == "square" else wl.chain_bonds(N)
    diag = -J * sum(s[:, i] * s[:, k] for i, k in bonds)
    E = diag + (-h * R).sum(axis=1)
    eps = np.where(X <= 0.5, np.abs(h * R) * delta, np.inf).sum(axis=1)
    ok = eps <= 0.5e-4 * np.maximum(1.0, np.abs(E))
    return exact, series, delta, X, ok, eps, E


@pytest.mark.parametrize("k,nb", [(5, 6), (3, 24), (2, 64), (1, 256)])
def test_bound_holds_and_configs_pass(k, nb):
    w = wl.make_config(k, B=nb) if k != 1 else wl.make_config(1)
    exact, series, delta, X, ok, eps, E = tfim_guard(w, nb)
    inside = X <= 0.5
    err = np.abs(exact - series)
    assert inside.all()
    assert np.all(err <= delta), f"c{k}: bound violated, worst ratio {(err / delta).max():.3f}"
    assert (err / delta).max() > 1e-3, "the bound should not be vacuous by many orders of magnitude"
    if k in (3, 5):  # the benchmark configurations must sit inside the guard, with margin
        assert ok.all() and (eps / (0.5e-4 * np.maximum(1.0, np.abs(E)))).max() < 0.6, (eps, E)


@pytest.mark.filterwarnings("ignore::RuntimeWarning")  # float16 overflow of the operands IS the refusal at 0.3, 0.5
@pytest.mark.parametrize("sigma", [0.1, 0.3, 0.5])
def test_p10_is_refused(sigma):
    w = wl.make_robustness(sigma, B=12)
    w.meta["config"] = 3
    exact, series, delta, X, ok, eps, E = tfim_guard(w, 12)
    assert not ok.any(), "every sample of the robustness set must fail the guard"
    inside = X <= 0.5
    if inside.any():  # where the bound claims validity it must still hold
        err = np.abs(exact - series)
        assert np.all(err[inside] <= delta[inside] * (1 + 1e-9))


def test_threshold_scan_config3_shapes():
    """Where the guard flips for config-3 shapes (N = 100, M = 400) as sigma grows: config 3's own sigma = 0.01
    passes (at ~0.4 of the threshold), sigma = 0.014 is already refused -- the window the GPU test
    (test_gpu_series.test_guard_boundary_inside_and_outside) must reproduce -- and the decision is monotone.  The
    bound is a worst-case one (every rounding error aligned, Cauchy-Schwarz on the norms): the float64 evaluation
    shows the actual error 8 x to 50 x below it over the whole scan, so a refusal means "not provably inside the
    tolerance", not "wrong"."""
    decisions = {}
    for sigma in (0.01, 0.014, 0.02, 0.028):
        w = wl.make_config(3, B=16, sigma=sigma, seed=31)
        exact, series, delta, X, ok, eps, E = tfim_guard(w, 16)
        decisions[sigma] = bool(ok.all())
        inside = X <= 0.5
        err = np.abs(exact - series)
        assert np.all(err[inside] <= delta[inside])
        assert (err[inside] / delta[inside]).max() < 0.5
        # the actual weighted series error is within HALF the tolerance wherever the guard passes -- and, the
        # bound being conservative, also one step beyond
        if sigma <= 0.014:
            actual = (np.abs(3.0 * np.exp(exact)) * err).sum(axis=1)
            assert np.all(actual <= 0.5e-4 * np.maximum(1.0, np.abs(E)))
    assert decisions == {0.01: True, 0.014: False, 0.02: False, 0.028: False}, decisions
