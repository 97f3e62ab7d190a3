"""Parity of nqs_metropolis against the float64 oracle.

Floating point decides an integer here (accept / reject), and the kernel takes the decision in
float32 from a product form the oracle does not use.  Several chains are therefore correct; what is
unique is checked on EVERY chain (reading Q19): both sides emit their per-step
accept bits (nqs_metropolis_trace / oracle.metropolis(trace=True)), and
  * a chain whose decisions never differ from the oracle's must be bit-identical in final spins and
    accepted count;
  * where a chain differs, the FIRST step at which the two decide differently must be a near-tie for the
    oracle at that very step: margin |2 Re dlog psi - log u| < MARGIN.  (After that step the two chains are
    in different states and are no longer comparable; the chain must still be a valid configuration and
    consistent with its own accept bits.)
MARGIN = 2e-4 is about 10x the float32 error of log |ratio|^2 seen at these sizes; it was set empirically
in round 1 and has not been changed.  There is no robust-fraction floor any more: it judged the inputs.
"""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu

MARGIN = 2e-4


@pytest.fixture(scope="module")
def nqs():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests need a B200")
    import paper_2108_03409_b200 as m

    m.load_library()
    return m


def proposals(S, C, N, seed):
    rng = np.random.default_rng([seed, 9])
    return rng.integers(0, N, (S, C)).astype(np.int32), rng.random((S, C), dtype=np.float32)


def gpu_metropolis(nqs, spins, a, b, W, sites, u, trace=False):
    import torch

    d = torch.device("cuda:0")
    t = lambda x: torch.from_numpy(np.ascontiguousarray(x)).to(d)  # noqa: E731
    sp = t(spins.copy())
    out = nqs.metropolis(sp, t(a), t(b), t(W), t(sites), t(u), trace=trace)
    torch.cuda.synchronize()
    if trace:
        return sp.cpu().numpy(), out[0].cpu().numpy(), out[1].cpu().numpy()
    return sp.cpu().numpy(), out.cpu().numpy()


def replay(start, sites, dec):
    """The chain states implied by a table of accept bits (bit-exact index work, no arithmetic)."""
    s = start.copy()
    cols = np.arange(s.shape[0])
    for t in range(sites.shape[0]):
        acc = dec[t].astype(bool)
        s[cols[acc], sites[t, acc]] *= -1
    return s


def compare(start, sites, final, acc, dec, ref_final, ref_acc, ref_dec, ref_mar, what):
    """Every chain is judged: identical decisions => identical result; otherwise the first differing
    decision must have been a near-tie in float64.  Returns the number of chains that parted ways."""
    assert set(np.unique(final)) <= {-1, 1}, what
    assert set(np.unique(dec)) <= {0, 1}, what
    # the kernel's outputs are consistent with its own trace
    assert np.array_equal(dec.sum(axis=0), acc), f"{what}: accepted count != number of accept bits"
    assert np.array_equal(replay(start, sites, dec), final), f"{what}: final spins do not follow from the accept bits"
    differ = dec != ref_dec
    parted = differ.any(axis=0)
    same = ~parted
    assert np.array_equal(final[same], ref_final[same]) and np.array_equal(acc[same], ref_acc[same]), what
    if parted.any():
        first = differ.argmax(axis=0)[parted]
        m = ref_mar[first, np.flatnonzero(parted)]
        bad = np.flatnonzero(m >= MARGIN)
        assert bad.size == 0, (f"{what}: {bad.size} chains part from the oracle at a decision that was no tie: "
                               f"chains {np.flatnonzero(parted)[bad[:5]]}, steps {first[bad[:5]]}, margins {m[bad[:5]]}")
    return int(parted.sum())


@pytest.mark.parametrize("N,M,C,S,sigma,seed", [
    (8, 8, 256, 64, 0.3, 1),        # config-1 shapes
    (40, 80, 1000, 200, 0.05, 2),   # config-2 shapes, 5 sweeps
    (37, 45, 333, 150, 0.2, 3),     # ragged sizes, chains not a multiple of the block
    (100, 400, 2048, 100, 0.03, 4), # config-3 shapes, one sweep
    (20, 30, 64, 2000, 0.25, 5),    # long chains: drift of the in-place update over 100 sweeps
    (142, 95, 463, 227, 0.25, 6),   # saturated hidden units (|Re theta| up to ~13): range of the ratio product
])
def test_metropolis_vs_oracle(nqs, oracle, N, M, C, S, sigma, seed):
    w = wl.make_random(N, M, C, 4, sigma, 200 + seed)
    sites, u = proposals(S, w.B, N, seed)
    final, acc, dec = gpu_metropolis(nqs, w.spins, w.a, w.b, w.W, sites, u, trace=True)
    ref_final, ref_acc, _, ref_dec, ref_mar = oracle.metropolis(w.spins, w.a, w.b, w.W, sites, u, trace=True)
    parted = compare(w.spins, sites, final, acc, dec, ref_final, ref_acc, ref_dec, ref_mar,
                     f"N={N} M={M} C={w.B} S={S}")
    assert parted <= 0.5 * w.B  # sanity only: the judgement is per chain, above
    assert 0.05 < acc.mean() / S <= 1.0
    # the untraced entry point gives the same chains
    f2, a2 = gpu_metropolis(nqs, w.spins, w.a, w.b, w.W, sites, u)
    assert np.array_equal(f2, final) and np.array_equal(a2, acc)


def test_metropolis_config5_full_size_sampled_chains(nqs, oracle):
    """Config 5 at full size (65536 chains, the launch configuration of the sampler bench): chains are
    independent, so the oracle replays 48 sampled chains one by one; every chain is checked against its
    own accept bits."""
    w = wl.make_config(5)
    S = 24
    sites, u = proposals(S, w.B, w.N, 55)
    final, acc, dec = gpu_metropolis(nqs, w.spins, w.a, w.b, w.W, sites, u, trace=True)
    assert set(np.unique(final)) <= {-1, 1}
    assert np.array_equal(dec.sum(axis=0), acc)
    assert np.array_equal(replay(w.spins, sites, dec), final)
    sel = np.sort(np.random.default_rng(56).choice(w.B, size=48, replace=False))
    sel[0], sel[-1] = 0, w.B - 1
    ref_final, ref_acc, _, ref_dec, ref_mar = oracle.metropolis(w.spins[sel], w.a, w.b, w.W, sites[:, sel], u[:, sel],
                                                                trace=True)
    compare(w.spins[sel], sites[:, sel], final[sel], acc[sel], dec[:, sel], ref_final, ref_acc, ref_dec, ref_mar,
            "config 5 sampled chains")


def gpu_metropolis_shared(nqs, spins, a, b, W, sites, u):
    import torch

    d = torch.device("cuda:0")
    t = lambda x: torch.from_numpy(np.ascontiguousarray(x)).to(d)  # noqa: E731
    sp = t(spins.copy())
    acc, dec = nqs.metropolis_shared(sp, t(a), t(b), t(W), t(sites), t(u), trace=True)
    torch.cuda.synchronize()
    return sp.cpu().numpy(), acc.cpu().numpy(), dec.cpu().numpy()


@pytest.mark.parametrize("N,M,C,S,sigma,seed", [
    (8, 8, 256, 64, 0.3, 11),         # one hidden-unit pair record per lane (PPL = 1)
    (40, 80, 1000, 200, 0.05, 12),    # config-2 shapes, 5 sweeps, chains not a multiple of the 12-chain block
    (37, 45, 333, 150, 0.2, 13),      # ragged
    (100, 400, 2048, 100, 0.03, 14),  # config-3 shapes (PPL = 8)
    (20, 30, 64, 2000, 0.25, 15),     # long chains: 100 sweeps, theta refreshed every 2 N steps
    (142, 95, 463, 227, 0.25, 16),    # saturated hidden units
    (50, 700, 100, 120, 0.02, 17),    # PPL = 13
    (30, 1900, 40, 70, 0.01, 18),     # PPL = 32 (8-warp blocks)
])
def test_metropolis_shared_site_vs_oracle(nqs, oracle, N, M, C, S, sigma, seed):
    """nqs_metropolis_shared: every chain proposes the same site at a step.  Same oracle (the site schedule is
    broadcast to [S, C]), same per-chain rule."""
    w = wl.make_random(N, M, C, 4, sigma, 300 + seed)
    rng = np.random.default_rng([seed, 9])
    sites1 = rng.integers(0, N, S).astype(np.int32)
    u = rng.random((S, w.B), dtype=np.float32)
    sites = np.ascontiguousarray(np.broadcast_to(sites1[:, None], (S, w.B)))
    final, acc, dec = gpu_metropolis_shared(nqs, w.spins, w.a, w.b, w.W, sites1, u)
    ref_final, ref_acc, _, ref_dec, ref_mar = oracle.metropolis(w.spins, w.a, w.b, w.W, sites, u, trace=True)
    parted = compare(w.spins, sites, final, acc, dec, ref_final, ref_acc, ref_dec, ref_mar,
                     f"shared N={N} M={M} C={w.B} S={S}")
    assert parted <= 0.5 * w.B
    assert 0.05 < acc.mean() / S <= 1.0


def test_metropolis_shared_config5_full_size_sampled_chains(nqs, oracle):
    """The launch configuration of the sampler bench (65536 chains, N = 400, M = 1600: PPL = 25, 12-chain blocks)."""
    w = wl.make_config(5)
    S = 24
    rng = np.random.default_rng(57)
    sites1 = rng.integers(0, w.N, S).astype(np.int32)
    u = rng.random((S, w.B), dtype=np.float32)
    final, acc, dec = gpu_metropolis_shared(nqs, w.spins, w.a, w.b, w.W, sites1, u)
    sites = np.ascontiguousarray(np.broadcast_to(sites1[:, None], (S, w.B)))
    assert np.array_equal(dec.sum(axis=0), acc) and np.array_equal(replay(w.spins, sites, dec), final)
    sel = np.sort(np.random.default_rng(58).choice(w.B, size=48, replace=False))
    sel[0], sel[1], sel[-1] = 0, 11, w.B - 1
    ref_final, ref_acc, _, ref_dec, ref_mar = oracle.metropolis(w.spins[sel], w.a, w.b, w.W, sites[:, sel], u[:, sel],
                                                                trace=True)
    compare(w.spins[sel], sites[:, sel], final[sel], acc[sel], dec[:, sel], ref_final, ref_acc, ref_dec, ref_mar,
            "config 5 shared-site sampled chains")


def test_metropolis_shared_samples_the_born_distribution(nqs):
    """A fixed site schedule shared by all chains still samples |psi|^2 (each chain is a valid Metropolis chain)."""
    from dense_reference import all_states, psi_all

    N, M, C, S = 5, 4, 60000, 100
    w = wl.make_random(N, M, 1 << N, 4, 0.3, 98)
    p = np.abs(psi_all(N, w.a, w.b, w.W)) ** 2
    p /= p.sum()
    rng = np.random.default_rng(99)
    start = all_states(N).astype(np.int8)[rng.integers(0, 1 << N, C)]
    sites1 = rng.integers(0, N, S).astype(np.int32)
    u = rng.random((S, C), dtype=np.float32)
    final, _, _ = gpu_metropolis_shared(nqs, start, w.a, w.b, w.W, sites1, u)
    idx = ((1 - final.astype(np.int64)) // 2) @ (1 << np.arange(N - 1, -1, -1))
    freq = np.bincount(idx, minlength=1 << N) / C
    assert np.all(np.abs(freq - p) < 4.5 * np.sqrt(p * (1 - p) / C)), np.abs(freq - p).max()


def test_metropolis_properties(nqs):
    import torch

    N, M, C = 24, 16, 100
    w = wl.make_random(N, M, C, 4, 0.2, 77)
    rng = np.random.default_rng(78)
    sites = np.repeat(rng.integers(0, N, (8, C)), 2, axis=0).astype(np.int32)
    final, acc = gpu_metropolis(nqs, w.spins, w.a, w.b, w.W, sites, np.zeros(sites.shape, np.float32))
    assert np.all(acc == 16) and np.array_equal(final, w.spins)  # u = 0 accepts; double flips restore
    sites, u = proposals(50, C, N, 79)
    f1, a1 = gpu_metropolis(nqs, w.spins, w.a, w.b, w.W, sites, u)
    f2, a2 = gpu_metropolis(nqs, w.spins, w.a, w.b, w.W, sites, u)
    assert np.array_equal(f1, f2) and np.array_equal(a1, a2)  # deterministic
    f0, a0 = gpu_metropolis(nqs, w.spins, w.a, w.b, w.W, sites[:0], u[:0])
    assert np.array_equal(f0, w.spins) and np.all(a0 == 0)  # S = 0
    d = torch.device("cuda:0")
    with pytest.raises(ValueError):
        nqs.metropolis(torch.from_numpy(w.spins).to(d), torch.from_numpy(w.a).to(d), torch.from_numpy(w.b).to(d),
                       torch.from_numpy(w.W).to(d), torch.from_numpy(sites[:, :5]).to(d), torch.from_numpy(u).to(d))


def test_metropolis_samples_the_born_distribution(nqs):
    """End to end, no oracle: 2^5 states, 60000 chains from uniform starts; the final states follow
    |psi|^2 (dense psi from tests/dense_reference.py) within 4.5 standard errors."""
    from dense_reference import all_states, psi_all

    N, M, C, S = 5, 4, 60000, 80
    w = wl.make_random(N, M, 1 << N, 4, 0.3, 88)
    p = np.abs(psi_all(N, w.a, w.b, w.W)) ** 2
    p /= p.sum()
    rng = np.random.default_rng(89)
    start = all_states(N).astype(np.int8)[rng.integers(0, 1 << N, C)]
    sites, u = proposals(S, C, N, 90)
    final, _ = gpu_metropolis(nqs, start, w.a, w.b, w.W, sites, u)
    idx = ((1 - final.astype(np.int64)) // 2) @ (1 << np.arange(N - 1, -1, -1))
    freq = np.bincount(idx, minlength=1 << N) / C
    assert np.all(np.abs(freq - p) < 4.5 * np.sqrt(p * (1 - p) / C)), np.abs(freq - p).max()


def test_saturated_chain_is_reported_not_frozen(nqs):
    """ADVICE (round 1): with the state exp(2 theta), |Re theta| >~ 22 overflows float32 and the chain would stop
    accepting silently.  It must be reported instead: accepted = -1 for such a chain, for both sampler kernels; chains
    of the same call that stay in range are unaffected."""
    import torch

    N, M, C, S = 16, 12, 40, 30
    w = wl.make_random(N, M, C, 4, 0.05, 123)
    W = w.W.copy()
    W[3, :] = 2.0  # hidden unit 3: theta = b_3 + 2 sum_i s_i, i.e. |Re theta| = 32 for the aligned configurations
    spins = w.spins.copy()
    spins[0, :] = 1     # chain 0: Re theta_3 = +32 -> exp(64) overflows
    spins[1, :] = -1    # chain 1: Re theta_3 = -32 -> exp(-64) underflows to 0: |E + 1|^2 = 1, stays finite
    spins[2, : N // 2] = 1
    spins[2, N // 2:] = -1  # chain 2: Re theta_3 ~ 0
    rng = np.random.default_rng(124)
    sites1 = rng.integers(0, N, S).astype(np.int32)
    u = rng.random((S, C), dtype=np.float32)
    d = torch.device("cuda:0")
    t = lambda x: torch.from_numpy(np.ascontiguousarray(x)).to(d)  # noqa: E731
    sites = np.ascontiguousarray(np.broadcast_to(sites1[:, None], (S, C)))
    acc_a = nqs.metropolis(t(spins), t(w.a), t(w.b), t(W), t(sites), t(u)).cpu().numpy()
    acc_b = nqs.metropolis_shared(t(spins), t(w.a), t(w.b), t(W), t(sites1), t(u)).cpu().numpy()
    for acc in (acc_a, acc_b):
        assert acc[0] == -1, "the overflowing chain must be flagged"
    assert np.array_equal(acc_a, acc_b)
    # (the strong unit pulls other chains towards alignment too; whichever saturate are flagged the same way by both
    # kernels.)  With the original small parameters nothing is flagged:
    acc_ok = nqs.metropolis_shared(t(spins), t(w.a), t(w.b), t(w.W), t(sites1), t(u)).cpu().numpy()
    assert np.all(acc_ok >= 0)


def test_shared_site_kernel_refuses_shapes_beyond_its_shared_memory(nqs):
    """the shared-site kernel keeps every site's table offsets and each chain's spins in shared memory;
    a lattice too large for the 227 KB of a block must come back as NQS_ERR_UNSUPPORTED (as include/nqs.h documents)
    before anything is launched -- not as a CUDA error from the launch.  nqs_metropolis takes the same shape."""
    import torch

    N, M, C, S = 12000, 16, 4, 3
    rng = np.random.default_rng(77)
    d = torch.device("cuda:0")
    t = lambda x: torch.from_numpy(np.ascontiguousarray(x)).to(d)  # noqa: E731
    spins0 = np.where(rng.random((C, N)) < 0.5, 1, -1).astype(np.int8)
    a = (1e-3 * (rng.standard_normal(N) + 1j * rng.standard_normal(N))).astype(np.complex64)
    b = (1e-3 * (rng.standard_normal(M) + 1j * rng.standard_normal(M))).astype(np.complex64)
    W = (1e-3 * (rng.standard_normal((M, N)) + 1j * rng.standard_normal((M, N)))).astype(np.complex64)
    sites1 = rng.integers(0, N, S).astype(np.int32)
    u = rng.random((S, C), dtype=np.float32)
    spins = t(spins0)
    n0 = nqs.launch_count()
    with pytest.raises(nqs.NqsError) as err:
        nqs.metropolis_shared(spins, t(a), t(b), t(W), t(sites1), t(u))
    assert err.value.code == -4 and "shared memory" in str(err.value), err.value
    assert nqs.launch_count() == n0
    torch.cuda.synchronize()
    assert np.array_equal(spins.cpu().numpy(), spins0)
    sites = np.ascontiguousarray(np.broadcast_to(sites1[:, None], (S, C)))
    acc = nqs.metropolis(spins, t(a), t(b), t(W), t(sites), t(u)).cpu().numpy()
    assert np.all((acc >= 0) & (acc <= S))
