"""Pins of oracle.metropolis (CPU only).

PM1 the acceptance rule, move by move, against the independent dense psi (dense_reference.psi_all):
    a proposal is accepted iff u < |psi(s')/psi(s)|^2 -- probed with u just below and just above the
    ratio for every basis state and site (a wrong power, a wrong site or a flipped inequality fails)
PM2 the stationary distribution: many chains, final states distributed as |psi|^2 / <psi|psi>
    (PAPER.md:56-61 p_theta(s); :70 Metropolis-Hastings) within 4.5 standard errors per state
PM3 bookkeeping (and the per-step trace: decisions and margins of every step of multi-step chains
    replayed against the dense psi): u = 0 accepts everything (two flips of a site restore the state), u ~ 1 with
    psi == const accepts nothing; chains are independent (a permutation of chains permutes outputs)
"""
import numpy as np

import workloads as wl
from dense_reference import all_states, psi_all


def test_pm1_acceptance_rule_against_dense_psi(oracle):
    N, M = 4, 3
    w = wl.make_random(N, M, 1 << N, 4, 0.5, 61)
    psi = psi_all(N, w.a, w.b, w.W)
    states = all_states(N).astype(np.int8)
    index = {tuple(s): k for k, s in enumerate(states)}
    for site in range(N):
        flipped = states.copy()
        flipped[:, site] *= -1
        ratio = np.array([abs(psi[index[tuple(f)]] / psi[k]) ** 2 for k, f in enumerate(flipped)])
        for factor, expect_accept in ((0.98, True), (1.02, False)):
            u = (ratio * factor).astype(np.float32)
            ok = u < 1.0  # only probes with a valid uniform number
            sites = np.full((1, 1 << N), site, dtype=np.int32)
            u = np.minimum(u, np.float32(0.999))
            final, acc, margin = oracle.metropolis(states, w.a, w.b, w.W, sites, u[None, :])
            assert np.array_equal(acc[ok] == 1, np.full(ok.sum(), expect_accept)), (site, factor)
            want = flipped if expect_accept else states
            assert np.array_equal(final[ok], want[ok])
            assert np.allclose(margin[ok], np.abs(np.log(ratio[ok]) - np.log(u[ok].astype(np.float64))), atol=1e-9)
            # the per-step trace (decision bit and margin of every single proposal) against the same dense ratios
            _, _, _, dec, mar = oracle.metropolis(states, w.a, w.b, w.W, sites, u[None, :], trace=True)
            assert dec.shape == mar.shape == (1, 1 << N)
            assert np.array_equal(dec[0, ok] == 1, np.full(ok.sum(), expect_accept))
            assert np.allclose(mar[0, ok], np.abs(np.log(ratio[ok]) - np.log(u[ok].astype(np.float64))), atol=1e-9)
        # ratio >= 1: accepted for every u in [0, 1)
        big = ratio >= 1.0
        if big.any():
            u = np.full((1, 1 << N), 0.999999, dtype=np.float32)
            _, acc, _ = oracle.metropolis(states, w.a, w.b, w.W, np.full((1, 1 << N), site, np.int32), u)
            assert np.all(acc[big] == 1)


def test_pm2_stationary_distribution(oracle):
    N, M, C, S = 3, 2, 40000, 40
    w = wl.make_random(N, M, 1 << N, 4, 0.3, 62)
    p = np.abs(psi_all(N, w.a, w.b, w.W)) ** 2
    p /= p.sum()
    assert p.min() > 0.005  # every state is visited often enough for the test below
    rng = np.random.default_rng(63)
    start = all_states(N).astype(np.int8)[rng.integers(0, 1 << N, C)]
    final, acc, _ = oracle.metropolis(start, w.a, w.b, w.W, rng.integers(0, N, (S, C)), rng.random((S, C), dtype=np.float32))
    idx = ((1 - final.astype(np.int64)) // 2) @ (1 << np.arange(N - 1, -1, -1))
    freq = np.bincount(idx, minlength=1 << N) / C
    sigma = np.sqrt(p * (1 - p) / C)
    assert np.all(np.abs(freq - p) < 4.5 * sigma), (freq, p)
    assert 0.2 < acc.mean() / S < 0.95


def test_pm3_bookkeeping(oracle):
    N, M, C = 7, 5, 50
    w = wl.make_random(N, M, C, 4, 0.3, 64)
    rng = np.random.default_rng(65)
    sites = np.repeat(rng.integers(0, N, (6, C)), 2, axis=0).astype(np.int32)  # every proposal twice in a row
    final, acc, _ = oracle.metropolis(w.spins, w.a, w.b, w.W, sites, np.zeros(sites.shape, np.float32))
    assert np.all(acc == 12) and np.array_equal(final, w.spins)
    zero = np.zeros_like(w.a), np.zeros_like(w.b), np.zeros_like(w.W)  # psi == 1: ratio 1, u < 1 accepts
    final, acc, _ = oracle.metropolis(w.spins, *zero, sites[:1], np.full((1, C), 0.999, np.float32))
    assert np.all(acc == 1)
    S = 30
    sites, u = rng.integers(0, N, (S, C)).astype(np.int32), rng.random((S, C), dtype=np.float32)
    f1, a1, m1 = oracle.metropolis(w.spins, w.a, w.b, w.W, sites, u)
    perm = rng.permutation(C)
    f2, a2, m2 = oracle.metropolis(w.spins[perm], w.a, w.b, w.W, sites[:, perm], u[:, perm])
    assert np.array_equal(f1[perm], f2) and np.array_equal(a1[perm], a2) and np.array_equal(m1[perm], m2)
    assert set(np.unique(f1)) <= {-1, 1}
    # trace: the decisions replayed by hand reproduce the final state and the counters; the per-step
    # margins reduce to min_margin; every step of a multi-step chain is checked against the dense psi
    f3, a3, m3, dec, mar = oracle.metropolis(w.spins, w.a, w.b, w.W, sites, u, trace=True)
    assert np.array_equal(f3, f1) and np.array_equal(a3, a1) and np.array_equal(m3, m1)
    assert np.array_equal(dec.sum(axis=0), a1) and np.array_equal(mar.min(axis=0), m1)
    psi = psi_all(N, w.a, w.b, w.W)
    idx_of = lambda s: int(((1 - s.astype(np.int64)) // 2) @ (1 << np.arange(N - 1, -1, -1)))  # noqa: E731
    for c in range(0, C, 7):
        s = w.spins[c].copy()
        for t in range(S):
            sp = s.copy()
            sp[sites[t, c]] *= -1
            lr = np.log(abs(psi[idx_of(sp)] / psi[idx_of(s)]) ** 2)
            lu = np.log(np.float64(u[t, c])) if u[t, c] > 0 else -np.inf
            assert dec[t, c] == (lu < lr) and abs(mar[t, c] - abs(lr - lu)) < 1e-9, (c, t)
            if dec[t, c]:
                s = sp
        assert np.array_equal(s, f1[c])
