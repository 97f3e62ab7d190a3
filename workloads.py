"""Seeded synthetic inputs for the five BASELINE.json configurations (+ the robustness set).

This module is the ONLY code shared by the float64 oracle (`oracle/`) and the CUDA path
(`paper_2108_03409_b200/`).  It holds none of the method's arithmetic: it draws random
parameters and spin configurations, and writes Hamiltonians down as lists of <=2-site
Pauli terms.  Nothing here evaluates log psi, a matrix element or a local energy.

Recipe:
  * numpy PCG64: parameters from default_rng([seed, 0]), spins from default_rng([seed, 1]),
    seed = configuration number 1..5.
  * draw order a.re[N], a.im[N], b.re[M], b.im[M], W.re[M,N], W.im[M,N]; each is
    standard_normal() * sigma cast to float32.  complex64 a[N], b[M], W[M,N] (row-major,
    W[j, i] couples hidden unit j to site i; Eq. 38, reading Q1).
  * spins are int8 +1/-1 [B, N]; +1 == "up" == sigma^z = +1 (reading Q2).

The inputs stand in for the paper's workloads (TFIM chains / 2-D TFIM next to g_c,
PAPER.md:565-577, :612-618) with an RBM (Eq. 38) as the ansatz; the paper uses no public
dataset, so nothing external is replaced.

Term-list format (the C-ABI's): sites int32 [T,2] (-1 = unused slot), paulis uint8 [T,2]
(0=I, 1=X, 2=Y, 3=Z), coeffs complex64 [T].
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

PAULI_I, PAULI_X, PAULI_Y, PAULI_Z = 0, 1, 2, 3


@dataclass
class Hamiltonian:
    """A list of at most 2-site Pauli terms (PAPER.md:418-426 Eq. 39; :473 Pauli products)."""

    sites: np.ndarray  # int32 [T,2]
    paulis: np.ndarray  # uint8 [T,2]
    coeffs: np.ndarray  # complex64 [T]
    name: str = ""

    @property
    def T(self) -> int:
        return int(self.sites.shape[0])


@dataclass
class Workload:
    name: str
    N: int
    M: int
    B: int
    spins: np.ndarray  # int8 [B,N]
    a: np.ndarray  # complex64 [N]
    b: np.ndarray  # complex64 [M]
    W: np.ndarray  # complex64 [M,N]
    ham: Hamiltonian
    meta: dict = field(default_factory=dict)


# ----------------------------------------------------------------------------------------
# term lists
# ----------------------------------------------------------------------------------------
def _terms(rows) -> Hamiltonian:
    T = len(rows)
    sites = np.full((T, 2), -1, dtype=np.int32)
    paulis = np.zeros((T, 2), dtype=np.uint8)
    coeffs = np.zeros((T,), dtype=np.complex64)
    for t, (s0, p0, s1, p1, c) in enumerate(rows):
        sites[t] = (s0, s1)
        paulis[t] = (p0, p1)
        coeffs[t] = c
    return Hamiltonian(sites, paulis, coeffs)


def chain_bonds(N: int):
    """Periodic chain: bonds (l, (l+1) % N), N bonds (reading Q11)."""
    return [(l, (l + 1) % N) for l in range(N)]


def square_bonds(L: int):
    """Periodic L x L square lattice, site (x, y) -> i = x*L + y; bonds to (x, y+1) and
    (x+1, y): 2*L*L bonds (reading Q11; L = 2 would double count and is not used)."""
    bonds = []
    for x in range(L):
        for y in range(L):
            i = x * L + y
            bonds.append((i, x * L + (y + 1) % L))
            bonds.append((i, ((x + 1) % L) * L + y))
    return bonds


def tfim(bonds, N: int, J: float, h: float) -> Hamiltonian:
    """H = -J sum_<ik> Z_i Z_k - h sum_i X_i (PAPER.md:585 Eq. 41, :616 Eq. 44; reading Q10)."""
    rows = [(i, PAULI_Z, k, PAULI_Z, -J) for (i, k) in bonds]
    rows += [(i, PAULI_X, -1, PAULI_I, -h) for i in range(N)]
    ham = _terms(rows)
    ham.name = f"tfim(J={J},h={h})"
    return ham


def heisenberg(bonds) -> Hamiltonian:
    """H = sum_<ik> (X_i X_k + Y_i Y_k + Z_i Z_k), Pauli matrices, coefficient +1 (reading Q9)."""
    rows = []
    for (i, k) in bonds:
        rows.append((i, PAULI_X, k, PAULI_X, 1.0))
        rows.append((i, PAULI_Y, k, PAULI_Y, 1.0))
        rows.append((i, PAULI_Z, k, PAULI_Z, 1.0))
    ham = _terms(rows)
    ham.name = "heisenberg"
    return ham


def random_terms(N: int, T: int, rng: np.random.Generator, allow_identity: bool = True) -> Hamiltonian:
    """Random 1- and 2-site Pauli terms of every type with complex coefficients (pin P1)."""
    rows = []
    for _ in range(T):
        kind = int(rng.integers(0, 4))
        c = complex(rng.standard_normal(), rng.standard_normal())
        if kind == 0 and allow_identity:  # constant / single-site
            s0 = int(rng.integers(0, N))
            p0 = int(rng.integers(0, 4))
            rows.append((s0, p0, -1, PAULI_I, c))
        elif kind == 1:  # single-site in slot 1 only
            s1 = int(rng.integers(0, N))
            p1 = int(rng.integers(1, 4))
            rows.append((-1, PAULI_I, s1, p1, c))
        else:  # two distinct sites
            s0, s1 = (int(v) for v in rng.choice(N, size=2, replace=False))
            p0 = int(rng.integers(0, 4))
            p1 = int(rng.integers(0, 4))
            rows.append((s0, p0, s1, p1, c))
    ham = _terms(rows)
    ham.name = f"random({T})"
    return ham


def random_strings(N: int, T: int, K: int, rng: np.random.Generator, max_flips: int = 4) -> Hamiltonian:
    """Random Pauli strings on up to K distinct sites (term arrays [T,K]):
    every Pauli type, complex coefficients, at most `max_flips` X/Y factors per string (the flip set), unused
    slots (-1) anywhere in the row."""
    sites = np.full((T, K), -1, dtype=np.int32)
    paulis = np.zeros((T, K), dtype=np.uint8)
    coeffs = np.zeros((T,), dtype=np.complex64)
    for t in range(T):
        m = int(rng.integers(0, min(K, N) + 1))  # number of sites the string acts on (0: constant term)
        where = rng.choice(K, size=m, replace=False)
        which = rng.choice(N, size=m, replace=False)
        flips = 0
        for slot, site in zip(where, which):
            p = int(rng.integers(0, 4))
            if p in (PAULI_X, PAULI_Y):
                if flips == max_flips:
                    p = PAULI_Z
                else:
                    flips += 1
            sites[t, slot] = site
            paulis[t, slot] = p
        coeffs[t] = complex(rng.standard_normal(), rng.standard_normal())
    ham = Hamiltonian(sites, paulis, coeffs)
    ham.name = f"strings({T},K={K})"
    return ham


# ----------------------------------------------------------------------------------------
# parameters and spins
# ----------------------------------------------------------------------------------------
def rbm_parameters(N: int, M: int, sigma: float, seed) -> tuple[np.ndarray, np.ndarray, np.ndarray]:
    rng = np.random.default_rng(seed)

    def draw(shape):
        return (rng.standard_normal(shape) * sigma).astype(np.float32)

    a_re, a_im = draw(N), draw(N)
    b_re, b_im = draw(M), draw(M)
    W_re, W_im = draw((M, N)), draw((M, N))
    a = (a_re + 1j * a_im).astype(np.complex64)
    b = (b_re + 1j * b_im).astype(np.complex64)
    W = (W_re + 1j * W_im).astype(np.complex64)
    return a, b, np.ascontiguousarray(W)


def basis_states(N: int) -> np.ndarray:
    """All 2^N configurations in index order; s_i = +1 iff bit (N-1-i) of k is 0 (pin P1)."""
    k = np.arange(1 << N, dtype=np.int64)[:, None]
    bits = (k >> (N - 1 - np.arange(N, dtype=np.int64))[None, :]) & 1
    return (1 - 2 * bits).astype(np.int8)


def iid_spins(B: int, N: int, seed) -> np.ndarray:
    rng = np.random.default_rng(seed)
    return (rng.integers(0, 2, size=(B, N), dtype=np.int8) * 2 - 1).astype(np.int8)


def zero_magnetisation_spins(B: int, N: int, seed) -> np.ndarray:
    """Per sample a random permutation of N/2 up and N/2 down spins (config 4)."""
    rng = np.random.default_rng(seed)
    base = np.concatenate([np.ones(N // 2, np.int8), -np.ones(N - N // 2, np.int8)])
    return rng.permuted(np.broadcast_to(base, (B, N)), axis=1).astype(np.int8)


# ----------------------------------------------------------------------------------------
# the five configurations (BASELINE.json "configs") and the robustness set (pin P10)
# ----------------------------------------------------------------------------------------
_SPECS = {
    1: dict(name="c1_tfim_chain_N8", lattice="chain", L=8, alpha=1, B=256, sigma=0.05, J=1.0, h=1.0),
    2: dict(name="c2_tfim_chain_N40", lattice="chain", L=40, alpha=2, B=16384, sigma=0.02, J=1.0, h=1.0),
    3: dict(name="c3_tfim_10x10", lattice="square", L=10, alpha=4, B=65536, sigma=0.01, J=1.0, h=3.0),
    4: dict(name="c4_heisenberg_10x10", lattice="square", L=10, alpha=2, B=32768, sigma=0.01),
    5: dict(name="c5_tfim_20x20", lattice="square", L=20, alpha=4, B=65536, sigma=0.005, J=1.0, h=3.0),
}


def config_spec(k: int) -> dict:
    spec = dict(_SPECS[k])
    L = spec["L"]
    spec["N"] = L if spec["lattice"] == "chain" else L * L
    spec["M"] = spec["alpha"] * spec["N"]
    return spec


def make_config(k: int, B: int | None = None, sigma: float | None = None, seed: int | None = None) -> Workload:
    """Configuration k in 1..5.  `B` truncates/extends the batch (spins are drawn for the
    requested B from the same stream, so the first rows agree between sizes only for the
    i.i.d. generators when drawn row-major -- tests that need a prefix slice the full batch)."""
    spec = config_spec(k)
    N, M = spec["N"], spec["M"]
    seed = k if seed is None else seed
    sig = spec["sigma"] if sigma is None else sigma
    nB = spec["B"] if B is None else B
    a, b, W = rbm_parameters(N, M, sig, [seed, 0])
    bonds = chain_bonds(N) if spec["lattice"] == "chain" else square_bonds(spec["L"])
    if k == 4:
        ham = heisenberg(bonds)
        spins = zero_magnetisation_spins(nB, N, [seed, 1])
    else:
        ham = tfim(bonds, N, spec["J"], spec["h"])
        if k == 1:
            spins = basis_states(N)
            if B is not None:
                spins = spins[:nB]
        else:
            spins = iid_spins(nB, N, [seed, 1])
    return Workload(spec["name"], N, M, int(spins.shape[0]), np.ascontiguousarray(spins), a, b, W, ham,
                    meta=dict(config=k, sigma=sig, seed=seed, lattice=spec["lattice"], L=spec["L"]))


def make_robustness(sigma: float, B: int = 512, seed: int = 103) -> Workload:
    """Pin P10: config-3 shapes (10x10 TFIM, N=100, M=400) with larger parameters."""
    w = make_config(3, B=B, sigma=sigma, seed=seed)
    w.name = f"p10_tfim_10x10_sigma{sigma}"
    return w


def make_random(N: int, M: int, B: int, T: int, sigma: float, seed: int) -> Workload:
    """Small random problem: random terms of all Pauli types, random spins and parameters."""
    a, b, W = rbm_parameters(N, M, sigma, [seed, 0])
    rng = np.random.default_rng([seed, 2])
    ham = random_terms(N, T, rng)
    spins = iid_spins(B, N, [seed, 1]) if B < (1 << N) or N > 16 else basis_states(N)
    return Workload(f"random_N{N}_M{M}_T{T}", N, M, int(spins.shape[0]), spins, a, b, W, ham,
                    meta=dict(sigma=sigma, seed=seed))
