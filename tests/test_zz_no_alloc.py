"""nqs_energy_stats_static: the batch statistics for callers that can not let the library allocate.

Some programs that want the mean and variance of E_loc (Eq. 5) have no device memory to spare for a
library: a JAX/XLA process that grabbed the whole GPU at start-up, a service running under a
fixed memory budget, a sampling loop that may not stall on the driver's allocator.  For them the library has one
entry point whose only scratch is a fixed 8 KB array inside the library image.  These tests check that it gives
what the ordinary entry point (nqs_energy_stats, scratch from the library's pool) gives -- to the 1e-12 relative
tolerance the statistics are tested to elsewhere (tests/test_gpu_forces.py), and in fact bit for bit, since the two
launch the same kernels in the same geometry -- on calls made back to back, where the second call finds the array
full of the first call's partial sums.

The static calls are made BEFORE the ordinary ones, so that when this file runs alone in a fresh process the entry
point is exercised in a library that has never created its pool.  The file sorts last on purpose: under
`pytest -x` a failure here must not hide another test.
"""
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
STATS_RTOL = 1e-12  # float64 sums of float32 inputs, as in tests/test_gpu_forces.py


@pytest.fixture(scope="module")
def nqs():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests need a B200")
    import paper_2108_03409_b200 as m

    m.load_library()
    return m


def local_energies(B, seed, device):
    """Seeded stand-in for E_loc [B] complex64 (any values do: the statistics are plain sums)."""
    import torch

    g = torch.Generator(device=device).manual_seed(1000 + seed)
    re = torch.empty(B, dtype=torch.float32, device=device).normal_(-50.0, 3.0, generator=g)
    im = torch.empty(B, dtype=torch.float32, device=device).normal_(0.0, 1.0, generator=g)
    return torch.complex(re, im)


def assert_same_stats(got, want, what):
    got, want = got.cpu().numpy(), want.cpu().numpy()
    assert np.all(np.isfinite(got)), f"{what}: {got}"
    mean = float(np.hypot(want[0], want[1]))
    scale = np.array([mean, mean, want[2], want[3]])  # Re / Im mean against |mean|, variance, sum of the weights
    assert np.all(np.abs(got - want) <= STATS_RTOL * scale), f"{what}: static {got} vs pooled {want}"
    assert np.array_equal(got, want), f"{what}: same kernels, same geometry, yet the bits differ: {got} vs {want}"


@pytest.mark.gpu
def test_static_scratch_matches_the_pooled_path_on_consecutive_calls(nqs):
    import torch

    d = torch.device("cuda:0")
    # (B, weighted): a batch that fills all 256 partial records, then a short one that fills 4 of them and must not
    # see the other 252 left over from the call before, then a weighted ragged one, then the first again
    cases = [(100_003, False), (1_000, False), (37_777, True), (100_003, False)]
    inputs = []
    for k, (B, weighted) in enumerate(cases):
        x = local_energies(B, k % 3, d)
        w = torch.rand(B, dtype=torch.float32, device=d, generator=torch.Generator(device=d).manual_seed(k)) if weighted else None
        inputs.append((x, w))
    # the caller's own output buffers: nothing is allocated between the static calls
    outs = [torch.empty(4, dtype=torch.float64, device=d) for _ in cases]
    torch.cuda.synchronize()
    for (x, w), out in zip(inputs, outs):  # back to back on one stream, no synchronisation in between
        r = nqs.energy_stats_static(x, w, out=out)
        assert r.data_ptr() == out.data_ptr()
    torch.cuda.synchronize()
    for k, ((x, w), out) in enumerate(zip(inputs, outs)):
        assert_same_stats(out, nqs.energy_stats(x, w), f"call {k} (B = {x.shape[0]}, weights = {w is not None})")
    # and against numpy, so that the pair is not merely consistently wrong
    x = inputs[0][0].cpu().numpy().astype(np.complex128)
    s = outs[0].cpu().numpy()
    assert abs(complex(s[0], s[1]) - x.mean()) <= 1e-12 * abs(x.mean()) and abs(s[2] - x.var()) <= 1e-9 * x.var()
    assert s[3] == x.shape[0]


@pytest.mark.gpu
def test_static_scratch_size_limit(nqs):
    """B up to NQS_STATS_STATIC_MAX_B runs (and agrees with the pooled path); one more is refused, nothing is launched."""
    import ctypes

    import torch

    d = torch.device("cuda:0")
    lib = nqs.load_library()
    small = local_energies(64, 5, d)
    out = torch.full((4,), -1.0, dtype=torch.float64, device=d)
    before = nqs.launch_count()
    rc = lib.nqs_energy_stats_static(ctypes.c_void_p(small.data_ptr()), None, nqs.STATS_STATIC_MAX_B + 1,
                                     ctypes.c_void_p(out.data_ptr()), None)
    assert rc == -4 and nqs.launch_count() == before  # NQS_ERR_UNSUPPORTED, before any launch
    msg = nqs.last_error()
    assert "NQS_STATS_STATIC_MAX_B" in msg and str(nqs.STATS_STATIC_MAX_B) in msg, msg
    torch.cuda.synchronize()
    assert np.all(out.cpu().numpy() == -1.0)
    assert lib.nqs_energy_stats_static(None, None, -1, None, None) == -1
    assert lib.nqs_energy_stats_static(None, None, 0, None, None) == 0  # B == 0: no-op like every entry point
    assert lib.nqs_energy_stats_static(None, None, 5, None, None) == -1
    big = local_energies(nqs.STATS_STATIC_MAX_B, 6, d)  # 512 MiB
    got = nqs.energy_stats_static(big, out=out)
    assert_same_stats(got, nqs.energy_stats(big), "B = NQS_STATS_STATIC_MAX_B")
    del big
    torch.cuda.empty_cache()


def test_static_entry_point_source_calls_no_allocator():
    """The promise 'allocates nothing' is kept by construction: the entry point and its helper name no allocating
    runtime call, no pool scratch and not device_state() (which creates the pool); the array is a file-scope
    `static __device__ __align__(256)` object whose device address comes from a checked cudaGetSymbolAddress."""
    src = open(os.path.join(ROOT, "paper_2108_03409_b200", "csrc", "nqs_api.cu")).read()
    bodies = []
    for head in (r"static int stats_static_scratch\(", r'extern "C" int nqs_energy_stats_static\('):
        m = re.search(head + r".*?\n}\n", src, flags=re.S)
        assert m, head
        bodies.append(re.sub(r"//[^\n]*", "", m.group(0)))
    text = "\n".join(bodies)
    for banned in ("cudaMalloc", "cudaFree", "cudaMemPool", "cudaHostAlloc", "Scratch", "device_state", "cudaStreamCreate",
                   "cudaEventCreate", "new ", "std::vector"):
        assert banned not in text, f"{banned} in the no-allocation entry point"
    assert re.search(r"static __device__ __align__\(256\) double g_stats_static_scratch\[", src)
    assert "NQS_CUDA(cudaGetSymbolAddress(&p, g_stats_static_scratch))" in bodies[0]
    assert "g_stats_static_scratch" not in bodies[1]  # the host-side name never reaches a kernel launch
