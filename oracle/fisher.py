"""Quantum Fisher matrix of the RBM (float64 CPU oracle; TEST INFRASTRUCTURE ONLY -- see nqs_oracle.c).

Eq. 10-11:  S_{k,k'} = << (O_k)^* O_k' >>_c ,  O_k(s) = d log psi(s) / d theta_k  (Eq. 8, :93),
the connected correlation written out as its two terms (Algorithm 1 line 9, :163-194; jVMC's
get_global_covariance, :515):

    S_{k,k'} = sum_b w_b O_k(s_b)^* O_k'(s_b) / sum_b w_b  -  <O_k>^* <O_k'>,     <O_k> = sum_b w_b O_k(s_b) / sum_b w_b.

O comes from oracle_log_derivatives (nqs_oracle.c, pinned by PF1); the contraction over the samples is one
library matrix product (numpy matmul on complex128) -- a plain definition, no blocking, no reordering.
Pins: tests/test_oracle_pins_fisher.py (PS1 dense-basis identity by finite differences of the dense psi,
PS2 Hermitian / positive semi-definite / diagonal = variances, PS3 numpy.cov, PS4 shift invariance).
"""
from __future__ import annotations

import numpy as np

from . import oracle as _o


def fisher_from_derivatives(O: np.ndarray, weights=None):
    """S [K,K] complex128 and <O> [K] from the logarithmic derivatives O [B,K] (Eq. 11)."""
    O = np.asarray(O, dtype=np.complex128)
    B = O.shape[0]
    w = np.full(B, 1.0 / B) if weights is None else np.asarray(weights, dtype=np.float64) / np.sum(weights, dtype=np.float64)
    Obar = (w[:, None] * O).sum(axis=0)
    S = O.conj().T @ (w[:, None] * O) - np.outer(Obar.conj(), Obar)
    return S, Obar


def fisher(spins, a, b, W, weights=None):
    """S [K,K] complex128, K = N + M + M*N in the order a, b, W (row-major), and <O> [K]."""
    return fisher_from_derivatives(_o.log_derivatives(spins, a, b, W), weights)
