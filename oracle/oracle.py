"""ctypes front end of oracle/nqs_oracle.c (float64 CPU oracle; TEST INFRASTRUCTURE ONLY).

`build()` compiles the C file with gcc (-O2 -fopenmp) into oracle/liboracle_nqs.so;
every other function marshals numpy arrays and calls it.  No arithmetic of the method
lives in this file.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nqs_oracle.c")
_LIB = os.path.join(_HERE, "liboracle_nqs.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle (gcc, float64, OpenMP over samples).  Returns the .so path."""
    with _lock:
        stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _LIB + f".tmp{os.getpid()}"
            cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
            subprocess.run(cmd, check=True)
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        vp, i64, i32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int
        lib.oracle_lncosh.argtypes = [vp, i64, i32, vp]
        lib.oracle_lncosh.restype = None
        lib.oracle_log_psi.argtypes = [vp, i64, i32, i32, vp, vp, vp, i32, vp]
        lib.oracle_log_psi.restype = None
        for fn in (lib.oracle_local_energy_definition, lib.oracle_local_energy_fast):
            fn.argtypes = [vp, i64, i32, i32, vp, vp, vp, i32, i32, vp, vp, vp, vp, vp]
            fn.restype = None
        lib.oracle_connected.argtypes = [vp, i64, i32, i32, i32, vp, vp, vp, vp, vp]
        lib.oracle_connected.restype = None
        lib.oracle_mean_variance.argtypes = [vp, vp, i64, vp]
        lib.oracle_mean_variance.restype = None
        lib.oracle_log_derivatives.argtypes = [vp, i64, i32, i32, vp, vp, vp, vp]
        lib.oracle_log_derivatives.restype = None
        lib.oracle_forces.argtypes = [vp, i64, i32, i32, vp, vp, vp, vp, vp, vp]
        lib.oracle_forces.restype = None
        lib.oracle_metropolis.argtypes = [vp, i64, i32, i32, vp, vp, vp, i32, vp, vp, vp, vp, vp, vp]
        lib.oracle_metropolis.restype = None
        lib.oracle_num_threads.restype = i32
        lib.oracle_set_num_threads.argtypes = [i32]
        _lib = lib
    return _lib


def _p(x: np.ndarray):
    return x.ctypes.data_as(ctypes.c_void_p)


def _c(x, dtype):
    x = np.ascontiguousarray(x, dtype=dtype)
    return x


def _params(spins, a, b, W):
    spins = _c(spins, np.int8)
    a, b, W = _c(a, np.complex64), _c(b, np.complex64), _c(W, np.complex64)
    B, N = spins.shape
    M = b.shape[0]
    assert a.shape == (N,) and W.shape == (M, N), (a.shape, b.shape, W.shape, spins.shape)
    return spins, a, b, W, B, N, M


def _terms(sites, paulis, coeffs):
    """Term arrays [T,K]: K slots per term (K = 2 for the five configurations; k-site Pauli strings use more)."""
    sites, paulis, coeffs = _c(sites, np.int32), _c(paulis, np.uint8), _c(coeffs, np.complex64)
    T = coeffs.shape[0]
    K = sites.shape[1] if sites.ndim == 2 else 2
    sites, paulis = sites.reshape(T, K), paulis.reshape(T, K)
    assert 1 <= K <= 16
    return sites, paulis, coeffs, T, K


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().oracle_set_num_threads(int(n))


def lncosh(z: np.ndarray, stable: bool) -> np.ndarray:
    """Pointwise log cosh: libm definition (stable=False) or formula F1 (stable=True)."""
    z = _c(z, np.complex128).ravel()
    out = np.empty_like(z)
    _load().oracle_lncosh(_p(z), z.size, int(stable), _p(out))
    return out


def log_psi(spins, a, b, W, stable: bool = False) -> np.ndarray:
    """complex128 [B]: Eq. 38."""
    spins, a, b, W, B, N, M = _params(spins, a, b, W)
    out = np.empty(B, dtype=np.complex128)
    _load().oracle_log_psi(_p(spins), B, N, M, _p(a), _p(b), _p(W), int(stable), _p(out))
    return out


def _eloc(fn, spins, a, b, W, sites, paulis, coeffs):
    spins, a, b, W, B, N, M = _params(spins, a, b, W)
    sites, paulis, coeffs, T, K = _terms(sites, paulis, coeffs)
    eloc = np.empty(B, dtype=np.complex128)
    logpsi = np.empty(B, dtype=np.complex128)
    fn(_p(spins), B, N, M, _p(a), _p(b), _p(W), T, K, _p(sites), _p(paulis), _p(coeffs), _p(eloc), _p(logpsi))
    return eloc, logpsi


def local_energy_definition(spins, a, b, W, sites, paulis, coeffs):
    """(E_loc, log psi) complex128 [B]; definition mode -- the parity authority."""
    return _eloc(_load().oracle_local_energy_definition, spins, a, b, W, sites, paulis, coeffs)


def local_energy_fast(spins, a, b, W, sites, paulis, coeffs):
    """(E_loc, log psi) complex128 [B]; fast mode (flip grouping + low-rank theta update)."""
    return _eloc(_load().oracle_local_energy_fast, spins, a, b, W, sites, paulis, coeffs)


def connected(spins, sites, paulis, coeffs):
    """Eq. 39 as data, term by term: s' int8 [B,T,N] and matrix elements complex128 [B,T]."""
    spins = _c(spins, np.int8)
    B, N = spins.shape
    sites, paulis, coeffs, T, K = _terms(sites, paulis, coeffs)
    sp = np.empty((B, T, N), dtype=np.int8)
    mel = np.empty((B, T), dtype=np.complex128)
    _load().oracle_connected(_p(spins), B, N, T, K, _p(sites), _p(paulis), _p(coeffs), _p(sp), _p(mel))
    return sp, mel


def _weights(weights, B):
    if weights is None:
        return None
    w = _c(weights, np.float64)
    assert w.shape == (B,)
    return w


def mean_variance(x, weights=None):
    """Eq. 5 / Eq. 3: (mean complex, variance, sum of weights) of x [B] complex."""
    x = _c(x, np.complex128)
    w = _weights(weights, x.shape[0])
    out = np.empty(4, dtype=np.float64)
    _load().oracle_mean_variance(_p(x), _p(w) if w is not None else None, x.shape[0], _p(out))
    return complex(out[0], out[1]), float(out[2]), float(out[3])


def log_derivatives(spins, a, b, W) -> np.ndarray:
    """Eq. 8: O [B,K] complex128, K = N + M + M*N in the order a, b, W (row-major)."""
    spins, a, b, W, B, N, M = _params(spins, a, b, W)
    out = np.empty((B, N + M + M * N), dtype=np.complex128)
    _load().oracle_log_derivatives(_p(spins), B, N, M, _p(a), _p(b), _p(W), _p(out))
    return out


def forces(spins, a, b, W, eloc, weights=None) -> np.ndarray:
    """Eq. 16: F [K] complex128 = <<O_k^* E_loc>> - <<O_k^*>><<E_loc>>."""
    spins, a, b, W, B, N, M = _params(spins, a, b, W)
    eloc = _c(eloc, np.complex128)
    assert eloc.shape == (B,)
    w = _weights(weights, B)
    out = np.empty(N + M + M * N, dtype=np.complex128)
    _load().oracle_forces(_p(spins), B, N, M, _p(a), _p(b), _p(W), _p(eloc), _p(w) if w is not None else None, _p(out))
    return out


def metropolis(spins, a, b, W, sites, u, trace: bool = False):
    """Single-spin-flip Metropolis chains driven by the given proposals (sites [S,C] int32) and
    uniforms (u [S,C] float32).  Returns (final spins int8 [C,N], accepted int32 [C], min_margin f64 [C]);
    with trace=True also (decisions uint8 [S,C], margins f64 [S,C]): the accept bit and the distance of
    every single decision from a tie."""
    spins, a, b, W, C, N, M = _params(spins, a, b, W)
    spins = spins.copy()
    sites, u = _c(sites, np.int32), _c(u, np.float32)
    S = sites.shape[0]
    assert sites.shape == (S, C) and u.shape == (S, C)
    assert sites.min(initial=0) >= 0 and sites.max(initial=0) < N
    acc = np.empty(C, dtype=np.int32)
    mm = np.empty(C, dtype=np.float64)
    dec = np.empty((S, C), dtype=np.uint8) if trace else None
    mar = np.empty((S, C), dtype=np.float64) if trace else None
    _load().oracle_metropolis(_p(spins), C, N, M, _p(a), _p(b), _p(W), S, _p(sites), _p(u), _p(acc), _p(mm),
                              _p(dec) if trace else None, _p(mar) if trace else None)
    return (spins, acc, mm, dec, mar) if trace else (spins, acc, mm)
