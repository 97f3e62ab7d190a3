"""ctypes binding of libnqs_b200.so -- same names as include/nqs.h, marshalling only."""
from __future__ import annotations

import ctypes
import os
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libnqs_b200.so")
_lock = threading.Lock()
_lib = None

NQS_OK = 0
ERROR_NAMES = {-1: "NQS_ERR_INVALID_ARG", -2: "NQS_ERR_INVALID_TERM", -3: "NQS_ERR_CUDA", -4: "NQS_ERR_UNSUPPORTED"}


class NqsError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"{ERROR_NAMES.get(code, code)}: {message}")
        self.code = code


def lib_path() -> str:
    return _LIB_PATH


def load_library() -> ctypes.CDLL:
    """Loads libnqs_b200.so; raises if it has not been built (python -m paper_2108_03409_b200.build)."""
    global _lib
    with _lock:
        if _lib is None:
            if not os.path.exists(_LIB_PATH):
                raise FileNotFoundError(
                    f"{_LIB_PATH} is missing: build it with `python -m paper_2108_03409_b200.build` "
                    "(there is no CPU fallback)")
            lib = ctypes.CDLL(_LIB_PATH)
            vp, i64, i32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32
            lib.nqs_log_psi.argtypes = [vp, i64, i32, i32, vp, vp, vp, vp, vp]
            lib.nqs_local_energy.argtypes = [vp, i64, i32, i32, vp, vp, vp, i32, vp, vp, vp, vp, vp, vp]
            lib.nqs_local_energy_host.argtypes = [vp, i64, i32, i32, vp, vp, vp, i32, vp, vp, vp, vp, vp]
            lib.nqs_log_psi_host.argtypes = [vp, i64, i32, i32, vp, vp, vp, vp]
            lib.nqs_hamiltonian_create.argtypes = [i32, i32, vp, vp, vp, ctypes.POINTER(vp)]
            lib.nqs_hamiltonian_compile_host.argtypes = [i32, i32, vp, vp, vp, ctypes.POINTER(vp)]
            lib.nqs_hamiltonian_destroy.argtypes = [vp]
            lib.nqs_hamiltonian_info.argtypes = [vp, vp, vp]
            lib.nqs_local_energy_h.argtypes = [vp, vp, i64, i32, vp, vp, vp, vp, vp, vp]
            lib.nqs_enumerate_connected_h.argtypes = [vp, vp, i64, vp, vp, vp]
            lib.nqs_enumerate_connected.argtypes = [vp, i64, i32, i32, vp, vp, vp, vp, vp, vp, vp]
            lib.nqs_metropolis_trace.argtypes = [vp, i64, i32, i32, vp, vp, vp, i32, vp, vp, vp, vp, vp]
            lib.nqs_set_option.argtypes = [i32, i32]
            lib.nqs_get_option.argtypes = [i32, vp]
            lib.nqs_debug_last_a5.argtypes = [vp, vp]
            lib.nqs_launch_count.argtypes = [vp]
            lib.nqs_hamiltonian_create_k.argtypes = [i32, i32, i32, vp, vp, vp, ctypes.POINTER(vp)]
            lib.nqs_hamiltonian_compile_host_k.argtypes = [i32, i32, i32, vp, vp, vp, ctypes.POINTER(vp)]
            lib.nqs_hamiltonian_info_k.argtypes = [vp, vp, vp]
            lib.nqs_local_energy_k.argtypes = [vp, i64, i32, i32, vp, vp, vp, i32, i32, vp, vp, vp, vp, vp, vp]
            lib.nqs_metropolis_shared.argtypes = [vp, i64, i32, i32, vp, vp, vp, i32, vp, vp, vp, vp, vp]
            lib.nqs_fisher.argtypes = [vp, i64, i32, i32, vp, vp, vp, vp, vp, vp, vp]
            lib.nqs_vmc_step_h.argtypes = [vp, vp, i64, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
            lib.nqs_energy_stats.argtypes = [vp, vp, i64, vp, vp]
            lib.nqs_energy_stats_static.argtypes = [vp, vp, i64, vp, vp]
            lib.nqs_forces.argtypes = [vp, i64, i32, i32, vp, vp, vp, vp, vp, vp, vp, vp]
            lib.nqs_microbench.argtypes = [i32, i32, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_float)]
            lib.nqs_local_energy_forces_h.argtypes = [vp, vp, i64, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp]
            lib.nqs_metropolis.argtypes = [vp, i64, i32, i32, vp, vp, vp, i32, vp, vp, vp, vp]
            lib.nqs_profile_enable.argtypes = [i32]
            lib.nqs_profile_last.argtypes = [vp]
            lib.nqs_last_error.restype = ctypes.c_char_p
            lib.nqs_version.restype = ctypes.c_char_p
            for name in ("nqs_log_psi", "nqs_local_energy", "nqs_local_energy_host", "nqs_log_psi_host",
                         "nqs_hamiltonian_create", "nqs_hamiltonian_compile_host", "nqs_hamiltonian_destroy",
                         "nqs_hamiltonian_info", "nqs_local_energy_h", "nqs_enumerate_connected", "nqs_release",
                         "nqs_profile_enable", "nqs_profile_last", "nqs_microbench", "nqs_energy_stats",
                         "nqs_forces", "nqs_metropolis", "nqs_local_energy_forces_h", "nqs_enumerate_connected_h",
                         "nqs_metropolis_trace", "nqs_set_option", "nqs_get_option", "nqs_debug_last_a5",
                         "nqs_launch_count", "nqs_fisher", "nqs_vmc_step_h", "nqs_hamiltonian_create_k",
                         "nqs_hamiltonian_compile_host_k", "nqs_hamiltonian_info_k", "nqs_local_energy_k",
                         "nqs_metropolis_shared", "nqs_energy_stats_static"):
                getattr(lib, name).restype = ctypes.c_int
            _lib = lib
    return _lib


def last_error() -> str:
    return load_library().nqs_last_error().decode()


def version() -> str:
    return load_library().nqs_version().decode()


def release() -> None:
    _check(load_library().nqs_release())


def profile_enable(on: bool) -> None:
    _check(load_library().nqs_profile_enable(int(on)))


PROFILE_SEGMENTS = ("table", "theta", "series_pack", "series_gemm", "series_guard", "eloc", "finalize")


def profile_last() -> dict:
    """Milliseconds of the kernels of the most recent profiled nqs_local_energy* call (include/nqs.h)."""
    ms = (ctypes.c_float * len(PROFILE_SEGMENTS))()
    _check(load_library().nqs_profile_last(ms))
    return {k: ms[i] for i, k in enumerate(PROFILE_SEGMENTS)}


OPTIONS = {"a5_path": 0, "theta_path": 1, "host_chunks": 2, "small_path": 3, "theta_split": 4, "series_wide": 5,
           "series_latch": 6}
A5_PATHS = {"auto": 0, "product": 1, "series_guarded": 2, "series_only": 3}


def set_option(key: str, value: int) -> None:
    """nqs_set_option: process-wide test / benchmark switches (include/nqs.h)."""
    _check(load_library().nqs_set_option(OPTIONS[key], int(value)))


def get_option(key: str) -> int:
    v = ctypes.c_int32()
    _check(load_library().nqs_get_option(OPTIONS[key], ctypes.byref(v)))
    return int(v.value)


def launch_count() -> int:
    """nqs_launch_count: kernels launched by the library so far in this process."""
    v = ctypes.c_int64()
    _check(load_library().nqs_launch_count(ctypes.byref(v)))
    return int(v.value)


def debug_last_a5() -> dict:
    """nqs_debug_last_a5 (synchronises): which a5 path the last nqs_local_energy* call took."""
    out = (ctypes.c_int32 * 3)()
    _check(load_library().nqs_debug_last_a5(out, _stream()))
    return dict(path={1: "series", 2: "product", 3: "small"}.get(out[0], "none"), guard_failed=bool(out[1]), samples_over=int(out[2]))


MICROBENCH_KINDS = {"ffma": 0, "ffma2": 1, "a5_body_packed": 2, "a5_body_scalar": 3, "mufu_ex2": 4}


def microbench(kind: str, iters: int = 20000) -> dict:
    """nqs_microbench: measured pipe rate (lane-operations per second over the whole GPU)."""
    rate, ms = ctypes.c_double(), ctypes.c_float()
    _check(load_library().nqs_microbench(MICROBENCH_KINDS[kind], iters, ctypes.byref(rate), ctypes.byref(ms)))
    return dict(kind=kind, lane_ops_per_s=rate.value, ms=ms.value)


def _check(rc: int) -> None:
    if rc != NQS_OK:
        raise NqsError(rc, last_error())


def _np(x, dtype, shape_tail=None):
    x = np.ascontiguousarray(x, dtype=dtype)
    if shape_tail is not None:
        assert x.shape[1:] == shape_tail, (x.shape, shape_tail)
    return x


def _terms(sites, paulis, coeffs):
    """Term arrays [T,K]: K = 2 slots per term, or up to 8 for k-site Pauli strings (the *_k entry points)."""
    coeffs = _np(coeffs, np.complex64).reshape(-1)
    sites = _np(sites, np.int32)
    K = sites.shape[1] if sites.ndim == 2 and sites.shape[0] == coeffs.shape[0] else 2
    sites = sites.reshape(-1, K)
    paulis = _np(paulis, np.uint8).reshape(-1, K)
    assert sites.shape[0] == paulis.shape[0] == coeffs.shape[0]
    return sites, paulis, coeffs


def _hp(x: np.ndarray):
    return x.ctypes.data_as(ctypes.c_void_p)


def _stream():
    import torch

    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev(t, dtype, name):
    import torch

    if not (isinstance(t, torch.Tensor) and t.is_cuda):
        raise TypeError(f"{name} must be a CUDA tensor")
    if t.dtype != dtype:
        raise TypeError(f"{name} must have dtype {dtype}, got {t.dtype}")
    if not t.is_contiguous():
        raise ValueError(f"{name} must be contiguous")
    return ctypes.c_void_p(t.data_ptr())


def _shapes(spins, a, b, W):
    B, N = spins.shape
    M = b.shape[0]
    if tuple(a.shape) != (N,) or tuple(W.shape) != (M, N):
        raise ValueError(f"shape mismatch: spins {tuple(spins.shape)}, a {tuple(a.shape)}, b {tuple(b.shape)}, "
                         f"W {tuple(W.shape)}")
    return B, N, M


class Hamiltonian:
    """Compiled term list (nqs_hamiltonian_create / _compile_host / _destroy / _info)."""

    def __init__(self, N: int, sites, paulis, coeffs, host_only: bool = False):
        lib = load_library()
        sites, paulis, coeffs = _terms(sites, paulis, coeffs)
        self.N = int(N)
        self.T = int(coeffs.shape[0])
        self.K = int(sites.shape[1])
        self._h = ctypes.c_void_p()
        if self.K == 2:
            fn = lib.nqs_hamiltonian_compile_host if host_only else lib.nqs_hamiltonian_create
            _check(fn(self.N, self.T, _hp(sites), _hp(paulis), _hp(coeffs), ctypes.byref(self._h)))
        else:
            fn = lib.nqs_hamiltonian_compile_host_k if host_only else lib.nqs_hamiltonian_create_k
            _check(fn(self.N, self.T, self.K, _hp(sites), _hp(paulis), _hp(coeffs), ctypes.byref(self._h)))
        info = np.zeros(5, np.int32)
        _check(lib.nqs_hamiltonian_info(self._h, _hp(info), None))
        self.G, self.C, self.n_diag, self.n_group_terms = (int(v) for v in info[:4])
        flips = np.zeros((max(self.G, 1), 4), np.int32)
        _check(lib.nqs_hamiltonian_info_k(self._h, _hp(info), _hp(flips)))
        self.flip_sites4 = flips[: self.G].copy()
        self.flip_sites = self.flip_sites4[:, :2].copy()

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            load_library().nqs_hamiltonian_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def local_energy(self, spins, a, b, W, want_logpsi: bool = True):
        import torch

        B, N, M = _shapes(spins, a, b, W)
        if N != self.N:
            raise ValueError("N mismatch with the compiled Hamiltonian")
        eloc = torch.empty(B, dtype=torch.complex64, device=spins.device)
        logpsi = torch.empty(B, dtype=torch.complex64, device=spins.device) if want_logpsi else None
        args = (self._h, _dev(spins, torch.int8, "spins"), B, M, _dev(a, torch.complex64, "a"),
                _dev(b, torch.complex64, "b"), _dev(W, torch.complex64, "W"), ctypes.c_void_p(eloc.data_ptr()),
                ctypes.c_void_p(logpsi.data_ptr()) if want_logpsi else None)
        if spins.device.index == torch.cuda.current_device():  # the common case: no device switch to pay for
            _check(load_library().nqs_local_energy_h(*args, _stream()))
        else:
            with torch.cuda.device(spins.device):
                _check(load_library().nqs_local_energy_h(*args, _stream()))
        return (eloc, logpsi) if want_logpsi else eloc

    def local_energy_forces(self, spins, a, b, W, weights=None):
        """nqs_local_energy_forces_h: (E_loc [B], log psi [B], F [N + M + M*N], stats [4] float64)."""
        import torch

        B, N, M = _shapes(spins, a, b, W)
        if N != self.N:
            raise ValueError("N mismatch with the compiled Hamiltonian")
        dev = spins.device
        eloc = torch.empty(B, dtype=torch.complex64, device=dev)
        logpsi = torch.empty(B, dtype=torch.complex64, device=dev)
        F = torch.empty(N + M + M * N, dtype=torch.complex64, device=dev)
        stats = torch.empty(4, dtype=torch.float64, device=dev)
        with torch.cuda.device(dev):
            _check(load_library().nqs_local_energy_forces_h(
                self._h, _dev(spins, torch.int8, "spins"), B, M, _dev(a, torch.complex64, "a"),
                _dev(b, torch.complex64, "b"), _dev(W, torch.complex64, "W"),
                _dev(weights, torch.float32, "weights") if weights is not None else None,
                ctypes.c_void_p(eloc.data_ptr()), ctypes.c_void_p(logpsi.data_ptr()), ctypes.c_void_p(F.data_ptr()),
                ctypes.c_void_p(stats.data_ptr()), _stream()))
        return eloc, logpsi, F, stats


    def vmc_step(self, spins, a, b, W, weights=None):
        """nqs_vmc_step_h: (E_loc [B], log psi [B], F [K], S [K,K], <O> [K], stats [4] float64), K = N + M + M*N."""
        import torch

        B, N, M = _shapes(spins, a, b, W)
        if N != self.N:
            raise ValueError("N mismatch with the compiled Hamiltonian")
        dev, K = spins.device, N + M + M * N
        eloc = torch.empty(B, dtype=torch.complex64, device=dev)
        logpsi = torch.empty(B, dtype=torch.complex64, device=dev)
        F = torch.empty(K, dtype=torch.complex64, device=dev)
        S = torch.empty((K, K), dtype=torch.complex64, device=dev)
        Obar = torch.empty(K, dtype=torch.complex64, device=dev)
        stats = torch.empty(4, dtype=torch.float64, device=dev)
        with torch.cuda.device(dev):
            _check(load_library().nqs_vmc_step_h(
                self._h, _dev(spins, torch.int8, "spins"), B, M, _dev(a, torch.complex64, "a"),
                _dev(b, torch.complex64, "b"), _dev(W, torch.complex64, "W"),
                _dev(weights, torch.float32, "weights") if weights is not None else None,
                ctypes.c_void_p(eloc.data_ptr()), ctypes.c_void_p(logpsi.data_ptr()), ctypes.c_void_p(F.data_ptr()),
                ctypes.c_void_p(S.data_ptr()), ctypes.c_void_p(Obar.data_ptr()), ctypes.c_void_p(stats.data_ptr()),
                _stream()))
        return eloc, logpsi, F, S, Obar, stats


def fisher(spins, a, b, W, weights=None):
    """nqs_fisher: (S [K,K], <O> [K]) complex64 CUDA tensors, K = N + M + M*N in the order a, b, W."""
    import torch

    B, N, M = _shapes(spins, a, b, W)
    K = N + M + M * N
    if weights is not None and tuple(weights.shape) != (B,):
        raise ValueError("weights must have shape [B]")
    S = torch.empty((K, K), dtype=torch.complex64, device=spins.device)
    Obar = torch.empty(K, dtype=torch.complex64, device=spins.device)
    with torch.cuda.device(spins.device):
        _check(load_library().nqs_fisher(
            _dev(spins, torch.int8, "spins"), B, N, M, _dev(a, torch.complex64, "a"), _dev(b, torch.complex64, "b"),
            _dev(W, torch.complex64, "W"), _dev(weights, torch.float32, "weights") if weights is not None else None,
            ctypes.c_void_p(S.data_ptr()), ctypes.c_void_p(Obar.data_ptr()), _stream()))
    return S, Obar


def energy_stats(x, weights=None):
    """nqs_energy_stats: float64 CUDA tensor [4] = (Re mean, Im mean, variance, sum of weights) of x [B]."""
    import torch

    stats = torch.empty(4, dtype=torch.float64, device=x.device)
    with torch.cuda.device(x.device):
        _check(load_library().nqs_energy_stats(
            _dev(x, torch.complex64, "x"), _dev(weights, torch.float32, "weights") if weights is not None else None,
            x.shape[0], ctypes.c_void_p(stats.data_ptr()), _stream()))
    return stats


STATS_STATIC_MAX_B = 1 << 26  # NQS_STATS_STATIC_MAX_B of include/nqs.h


def energy_stats_static(x, weights=None, out=None):
    """nqs_energy_stats_static: nqs_energy_stats for a caller that can not let the library allocate.

    Meant for a program whose own allocator already holds the GPU's memory (a JAX/XLA process with preallocation
    on, as in the paper's set-up), or that runs under a memory budget or a latency bound: the library takes
    nothing from the CUDA allocator here, its partial sums sit in a fixed 8 KB array inside the library image.
    The caller brings the output too: `out` is a float64 CUDA tensor [4] from the caller's own memory and is
    returned filled with (Re mean, Im mean, variance, sum of weights).  Only when `out` is None does this wrapper
    make one with torch.empty, as a convenience for tests -- that allocation is torch's, outside the library.
    x.shape[0] must not exceed STATS_STATIC_MAX_B (NqsError NQS_ERR_UNSUPPORTED otherwise).  All calls on a
    device share the array: run them on one stream or order them with events, and make the first call on each
    device before any stream capture starts (include/nqs.h).
    """
    import torch

    stats = torch.empty(4, dtype=torch.float64, device=x.device) if out is None else out
    if stats.dtype != torch.float64 or stats.numel() != 4 or not stats.is_cuda or not stats.is_contiguous():
        raise ValueError("out must be a contiguous float64 CUDA tensor of 4 elements")
    with torch.cuda.device(x.device):
        _check(load_library().nqs_energy_stats_static(
            _dev(x, torch.complex64, "x"), _dev(weights, torch.float32, "weights") if weights is not None else None,
            x.shape[0], ctypes.c_void_p(stats.data_ptr()), _stream()))
    return stats


def forces(spins, a, b, W, eloc, weights=None, want_stats: bool = False):
    """nqs_forces: complex64 CUDA tensor [N + M + M*N] (order a, b, W row-major); optionally the stats of eloc."""
    import torch

    B, N, M = _shapes(spins, a, b, W)
    if tuple(eloc.shape) != (B,) or (weights is not None and tuple(weights.shape) != (B,)):
        raise ValueError("eloc / weights must have shape [B]")
    F = torch.empty(N + M + M * N, dtype=torch.complex64, device=spins.device)
    stats = torch.empty(4, dtype=torch.float64, device=spins.device) if want_stats else None
    with torch.cuda.device(spins.device):
        _check(load_library().nqs_forces(
            _dev(spins, torch.int8, "spins"), B, N, M, _dev(a, torch.complex64, "a"), _dev(b, torch.complex64, "b"),
            _dev(W, torch.complex64, "W"), _dev(eloc, torch.complex64, "eloc"),
            _dev(weights, torch.float32, "weights") if weights is not None else None, ctypes.c_void_p(F.data_ptr()),
            ctypes.c_void_p(stats.data_ptr()) if want_stats else None, _stream()))
    return (F, stats) if want_stats else F


def metropolis(spins, a, b, W, sites, u, want_accepted: bool = True, trace: bool = False):
    """nqs_metropolis: advances the chains `spins` [C,N] IN PLACE by S = sites.shape[0] steps.
    trace=True (nqs_metropolis_trace) also returns the accept bits uint8 [S,C]."""
    import torch

    C, N, M = _shapes(spins, a, b, W)
    S = int(sites.shape[0])
    if tuple(sites.shape) != (S, C) or tuple(u.shape) != (S, C):
        raise ValueError("sites and u must have shape [S, C]")
    accepted = torch.empty(C, dtype=torch.int32, device=spins.device) if want_accepted else None
    args = (_dev(spins, torch.int8, "spins"), C, N, M, _dev(a, torch.complex64, "a"), _dev(b, torch.complex64, "b"),
            _dev(W, torch.complex64, "W"), S, _dev(sites, torch.int32, "sites"), _dev(u, torch.float32, "u"),
            ctypes.c_void_p(accepted.data_ptr()) if want_accepted else None)
    with torch.cuda.device(spins.device):
        if trace:
            decisions = torch.empty((S, C), dtype=torch.uint8, device=spins.device)
            _check(load_library().nqs_metropolis_trace(*args, ctypes.c_void_p(decisions.data_ptr()), _stream()))
            return accepted, decisions
        _check(load_library().nqs_metropolis(*args, _stream()))
    return accepted


def metropolis_shared(spins, a, b, W, sites, u, trace: bool = False):
    """nqs_metropolis_shared: every chain proposes sites[t] at step t (sites [S] int32, u [S,C] float32).
    Advances `spins` [C,N] IN PLACE; returns accepted [C] (and the accept bits uint8 [S,C] with trace=True)."""
    import torch

    C, N, M = _shapes(spins, a, b, W)
    S = int(sites.shape[0])
    if tuple(sites.shape) != (S,) or tuple(u.shape) != (S, C):
        raise ValueError("sites must have shape [S] and u shape [S, C]")
    accepted = torch.empty(C, dtype=torch.int32, device=spins.device)
    decisions = torch.empty((S, C), dtype=torch.uint8, device=spins.device) if trace else None
    with torch.cuda.device(spins.device):
        _check(load_library().nqs_metropolis_shared(
            _dev(spins, torch.int8, "spins"), C, N, M, _dev(a, torch.complex64, "a"), _dev(b, torch.complex64, "b"),
            _dev(W, torch.complex64, "W"), S, _dev(sites, torch.int32, "sites"), _dev(u, torch.float32, "u"),
            ctypes.c_void_p(accepted.data_ptr()), ctypes.c_void_p(decisions.data_ptr()) if trace else None, _stream()))
    return (accepted, decisions) if trace else accepted


def hamiltonian_info_host(N: int, sites, paulis, coeffs) -> dict:
    """Host-only compile (no GPU needed): grouping of the term list by flip set."""
    h = Hamiltonian(N, sites, paulis, coeffs, host_only=True)
    out = dict(G=h.G, C=h.C, n_diag=h.n_diag, n_group_terms=h.n_group_terms, flip_sites=h.flip_sites,
               flip_sites4=h.flip_sites4)
    h.close()
    return out


def log_psi(spins, a, b, W):
    """nqs_log_psi: complex64 [B] CUDA tensor (Eq. 38)."""
    import torch

    B, N, M = _shapes(spins, a, b, W)
    out = torch.empty(B, dtype=torch.complex64, device=spins.device)
    with torch.cuda.device(spins.device):
        _check(load_library().nqs_log_psi(_dev(spins, torch.int8, "spins"), B, N, M, _dev(a, torch.complex64, "a"),
                                          _dev(b, torch.complex64, "b"), _dev(W, torch.complex64, "W"),
                                          ctypes.c_void_p(out.data_ptr()), _stream()))
    return out


def local_energy(spins, a, b, W, sites, paulis, coeffs, want_logpsi: bool = True):
    """nqs_local_energy: (E_loc, log psi) complex64 [B] CUDA tensors (Eq. 4)."""
    import torch

    B, N, M = _shapes(spins, a, b, W)
    sites, paulis, coeffs = _terms(sites, paulis, coeffs)
    eloc = torch.empty(B, dtype=torch.complex64, device=spins.device)
    logpsi = torch.empty(B, dtype=torch.complex64, device=spins.device) if want_logpsi else None
    K = int(sites.shape[1])
    head = (_dev(spins, torch.int8, "spins"), B, N, M, _dev(a, torch.complex64, "a"), _dev(b, torch.complex64, "b"),
            _dev(W, torch.complex64, "W"), int(coeffs.shape[0]))
    tail = (_hp(sites), _hp(paulis), _hp(coeffs), ctypes.c_void_p(eloc.data_ptr()),
            ctypes.c_void_p(logpsi.data_ptr()) if want_logpsi else None)
    with torch.cuda.device(spins.device):
        if K == 2:
            _check(load_library().nqs_local_energy(*head, *tail, _stream()))
        else:
            _check(load_library().nqs_local_energy_k(*head, K, *tail, _stream()))
    return (eloc, logpsi) if want_logpsi else eloc


def local_energy_host(spins, a, b, W, sites, paulis, coeffs, eloc_out=None, logpsi_out=None, want_logpsi=True):
    """nqs_local_energy_host: numpy (or pinned torch CPU) buffers in, numpy out; copies inside."""
    spins = _np(spins, np.int8)
    a, b, W = _np(a, np.complex64), _np(b, np.complex64), _np(W, np.complex64)
    B, N, M = _shapes(spins, a, b, W)
    sites, paulis, coeffs = _terms(sites, paulis, coeffs)
    eloc = np.empty(B, np.complex64) if eloc_out is None else eloc_out
    logpsi = (np.empty(B, np.complex64) if logpsi_out is None else logpsi_out) if want_logpsi else None
    _check(load_library().nqs_local_energy_host(
        _hp(spins), B, N, M, _hp(a), _hp(b), _hp(W), int(coeffs.shape[0]), _hp(sites), _hp(paulis), _hp(coeffs),
        _hp(eloc), _hp(logpsi) if want_logpsi else None))
    return (eloc, logpsi) if want_logpsi else eloc


def log_psi_host(spins, a, b, W):
    spins = _np(spins, np.int8)
    a, b, W = _np(a, np.complex64), _np(b, np.complex64), _np(W, np.complex64)
    B, N, M = _shapes(spins, a, b, W)
    out = np.empty(B, np.complex64)
    _check(load_library().nqs_log_psi_host(_hp(spins), B, N, M, _hp(a), _hp(b), _hp(W), _hp(out)))
    return out


def enumerate_connected_h(ham: Hamiltonian, spins):
    """nqs_enumerate_connected_h: s' int8 [B,G+1,N], elements complex64 [B,G+1] (slot 0 = diagonal)."""
    import torch

    B, N = spins.shape
    sp = torch.empty((B, ham.G + 1, N), dtype=torch.int8, device=spins.device)
    mel = torch.empty((B, ham.G + 1), dtype=torch.complex64, device=spins.device)
    with torch.cuda.device(spins.device):
        _check(load_library().nqs_enumerate_connected_h(ham._h, _dev(spins, torch.int8, "spins"), B,
                                                        ctypes.c_void_p(sp.data_ptr()),
                                                        ctypes.c_void_p(mel.data_ptr()), _stream()))
    return sp, mel


def connected_groups(N: int, sites, paulis, coeffs) -> int:
    """nqs_enumerate_connected with B = 0: the number G of flip groups of a term list (host only)."""
    sites, paulis, coeffs = _terms(sites, paulis, coeffs)
    G = ctypes.c_int32(-1)
    _check(load_library().nqs_enumerate_connected(None, 0, int(N), int(coeffs.shape[0]), _hp(sites), _hp(paulis),
                                                  _hp(coeffs), None, None, ctypes.byref(G), None))
    return int(G.value)


def enumerate_connected(spins, sites, paulis, coeffs):
    """nqs_enumerate_connected (term-list form): (s' int8 [B,G+1,N], elements complex64 [B,G+1], G)."""
    import torch

    B, N = spins.shape
    sites, paulis, coeffs = _terms(sites, paulis, coeffs)
    G = connected_groups(N, sites, paulis, coeffs)
    sp = torch.empty((B, G + 1, N), dtype=torch.int8, device=spins.device)
    mel = torch.empty((B, G + 1), dtype=torch.complex64, device=spins.device)
    G2 = ctypes.c_int32(-1)
    with torch.cuda.device(spins.device):
        _check(load_library().nqs_enumerate_connected(
            _dev(spins, torch.int8, "spins"), B, N, int(coeffs.shape[0]), _hp(sites), _hp(paulis), _hp(coeffs),
            ctypes.c_void_p(sp.data_ptr()), ctypes.c_void_p(mel.data_ptr()), ctypes.byref(G2), _stream()))
    assert G2.value == G
    return sp, mel, G
