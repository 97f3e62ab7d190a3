"""Builds libnqs_b200.so (the C-ABI library of include/nqs.h) in-tree with nvcc for sm_100a.

    python -m paper_2108_03409_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The static CUDA runtime is linked, so the library loads
(and its host-only entry points work) on machines without a driver.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libnqs_b200.so")
SOURCES = ["nqs_api.cu", "nqs_hamiltonian.cpp"]
DEPS = SOURCES + ["nqs_kernels.cuh", "nqs_theta_mma.cuh", "nqs_forces.cuh", "nqs_fisher.cuh", "nqs_microbench.cuh", "nqs_sampler.cuh", "nqs_series.cuh", "nqs_small.cuh", "nqs_device.cuh", "nqs_hamiltonian.h", os.path.join("..", "..", "include", "nqs.h")]


def nvcc_command(out: str, verbose: bool = False) -> list[str]:
    cmd = [
        os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc"),
        "-gencode", "arch=compute_100a,code=sm_100a",
        "-O3", "-std=c++17", "-lineinfo",
        "-Xcompiler", "-fPIC,-O2",
        "--shared", "-cudart", "static",
        "-o", out,
    ]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += os.environ.get("NQS_NVCC_FLAGS", "").split()  # development switches, e.g. -DNQS_SERIES_TIMELINE
    cmd += [os.path.join(CSRC, s) for s in SOURCES]
    return cmd


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or is_stale():
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = nvcc_command(tmp, verbose)
        res = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
