#!/usr/bin/env python
"""Benchmark of the batched RBM local-energy hot path (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 5]

A "step" is one pass of the whole hot path -- nqs_local_energy on one synthetic batch of the
configuration (default: config 5, 20x20 TFIM, N=400, M=1600, B=65536, the one the target
"% of the FP32 roofline" is quoted on) -- with inputs resident in HBM.  Rank 0 prints ONE JSON
line.  With N > 1 (torchrun) every rank runs its own batch (weak scaling, no collective on the
data path); the time is the max over ranks.

--impl reference times the float64 CPU oracle (oracle/, as it stands) on the host cores, each
step a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402

SM_COUNT = 148
FP32_LANES_PER_SM = 128
L2_FLUSH_BYTES = 256 << 20
# dram__bytes_read.sum + dram__bytes_write.sum of one eloc_kernel launch at config 5, from the
# ncu --set full capture summarised in profiles/ (None until a capture exists)
ELOC_KERNEL_DRAM_TRAFFIC_BYTES = 897_815_552  # profiles/r1_v3_ncu_summary.md: dram read + write per launch


def shard_plan(n_ranks: int, rank: int, config: int) -> dict:
    """Weak scaling: every rank draws its own batch of the configuration (its own spin seed),
    parameters and Hamiltonian replicated.  No data-path collective."""
    spec = wl.config_spec(config)
    return dict(config=config, B=spec["B"], spin_seed=[config, 1, rank], global_batch=spec["B"] * n_ranks)


def make_rank_workload(plan: dict) -> wl.Workload:
    k = plan["config"]
    w = wl.make_config(k)
    if plan["spin_seed"][-1] != 0:  # ranks > 0: same generator, different stream
        if k == 4:
            w.spins = wl.zero_magnetisation_spins(w.B, w.N, plan["spin_seed"])
        elif k != 1:
            w.spins = wl.iid_spins(w.B, w.N, plan["spin_seed"])
    return w


def fma_lane_ops(w: wl.Workload, C: int) -> dict:
    """Algorithmic FP32 lane-ops per step."""
    B, N, M = w.B, w.N, w.M
    return dict(a5=8.0 * B * C * M, a2=2.0 * B * N * M, a3=40.0 * B * M)


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index: int, period: float = 0.05):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._halt = threading.Event()
        self.ok = False
        try:
            import pynvml

            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
            nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
            nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake",
        }
        while not self._halt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self) -> dict:
        self._halt.set()
        self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return dict(sm_mhz=med, sm_max_mhz=self.max_mhz, reasons=sorted(self.reasons), samples=len(self.samples))


def cpu_baseline(w: wl.Workload, budget_s: float = 10.0) -> dict:
    """The float64 oracle (fast mode, OpenMP over samples), as it stands, on the host cores, on a
    bounded prefix of the same batch."""
    import oracle

    oracle.build()
    cores = oracle.num_threads()
    args = (w.a, w.b, w.W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    n0 = min(w.B, cores)
    t0 = time.perf_counter()
    oracle.local_energy_fast(w.spins[:n0], *args)
    dt0 = max(time.perf_counter() - t0, 1e-6)
    n = int(min(w.B, max(n0, (budget_s / dt0) * n0)))
    n = max(cores, n // cores * cores)
    t0 = time.perf_counter()
    oracle.local_energy_fast(w.spins[:n], *args)
    dt = time.perf_counter() - t0
    return dict(value=n / dt, unit="samples/s", cores=cores, kind="oracle",
                sample=f"fast mode (float64, flip grouping + low-rank theta update), first {n} of {w.B} samples "
                       f"of {w.name}, {dt:.2f} s wall, OpenMP {cores} threads"), n, dt


def run_reference(args) -> None:
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle

    oracle.build()
    plan = shard_plan(1, 0, args.config)
    w = make_rank_workload(plan)
    cores = oracle.num_threads()
    oargs = (w.a, w.b, w.W, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    # size one step to ~4 s of wall time
    n0 = min(w.B, cores)
    t0 = time.perf_counter()
    oracle.local_energy_fast(w.spins[:n0], *oargs)
    dt0 = max(time.perf_counter() - t0, 1e-6)
    total = max(args.steps + args.warmup, 1)
    per_step_budget = min(4.0, 150.0 / total)
    n = int(min(w.B, max(n0, per_step_budget / dt0 * n0)))
    n = max(cores, n // cores * cores)
    for _ in range(args.warmup):
        oracle.local_energy_fast(w.spins[:n], *oargs)
    times = []
    for _ in range(args.steps):
        t0 = time.perf_counter()
        oracle.local_energy_fast(w.spins[:n], *oargs)
        times.append(time.perf_counter() - t0)
    ms = 1e3 * float(np.mean(times))
    value = n / (ms * 1e-3)
    sample = (f"fast mode (float64), each step = first {n} of {w.B} samples of {w.name}, OpenMP {cores} threads")
    line = {
        "impl": "reference", "metric": "E_loc samples/s", "value": value, "unit": "samples/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "N": w.N, "M": w.M, "B": w.B, "terms": w.ham.T, "samples_per_step": n},
        "cpu_baseline": {"value": value, "unit": "samples/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "samples/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_ours(args) -> None:
    import torch
    import torch.distributed as dist

    import paper_2108_03409_b200 as nqs

    nqs.load_library()  # fail loudly when the CUDA extension is missing
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    plan = shard_plan(world, rank, args.config)
    w = make_rank_workload(plan)
    spins = torch.from_numpy(w.spins).to(dev)
    a, b, W = (torch.from_numpy(x).to(dev) for x in (w.a, w.b, w.W))
    ham = nqs.Hamiltonian(w.N, w.ham.sites, w.ham.paulis, w.ham.coeffs)
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        return ham.local_energy(spins, a, b, W)

    warm = max(args.warmup, 3)
    for _ in range(warm):
        e, l = step()
    torch.cuda.synchronize()

    # ---- timed region: K steps, each bracketed by CUDA events on the launching stream; the L2 is
    # flushed (256 MiB write) between steps, outside the event pairs.
    sampler = ClockSampler(local_rank)
    nqs.profile_enable(True)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    kern_ms = []
    barrier()
    sampler.start()
    for k in range(args.steps):
        flush.fill_(k & 0xFF)
        ev[k][0].record()
        e, l = step()
        ev[k][1].record()
        if k == args.steps - 1 or k % 4 == 3:
            kern_ms.append(nqs.profile_last())
    barrier()
    clocks = sampler.stop()
    nqs.profile_enable(False)
    step_ms = [s.elapsed_time(t) for s, t in ev]
    total_ms = float(np.sum(step_ms))
    if world > 1:
        tt = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        total_ms = float(tt.item())
    ms_per_step = total_ms / args.steps
    value = plan["global_batch"] / (ms_per_step * 1e-3)

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    pin = lambda x: torch.from_numpy(x).pin_memory()  # noqa: E731
    hs, ha, hb, hW = pin(w.spins), pin(w.a), pin(w.b), pin(w.W)
    he = torch.empty(w.B, dtype=torch.complex64).pin_memory()
    hl = torch.empty(w.B, dtype=torch.complex64).pin_memory()

    def e2e_step():
        nqs.local_energy_host(hs.numpy(), ha.numpy(), hb.numpy(), hW.numpy(), w.ham.sites, w.ham.paulis,
                              w.ham.coeffs, eloc_out=he.numpy(), logpsi_out=hl.numpy())

    for _ in range(2):
        e2e_step()
    n_e2e = max(2, min(args.steps, 5))
    barrier()
    t0 = time.perf_counter()
    for _ in range(n_e2e):
        e2e_step()
    torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / n_e2e
    if world > 1:
        tt = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        e2e_s = float(tt.item())
    h2d = int(w.spins.nbytes + w.a.nbytes + w.b.nbytes + w.W.nbytes)
    d2h = int(2 * w.B * 8)
    assert np.array_equal(he.numpy(), e.cpu().numpy()), "host and device entry points disagree"

    if rank == 0:
        ops = fma_lane_ops(w, ham.C)
        km = {k: float(np.median([d[k] for d in kern_ms])) for k in kern_ms[0]}
        f_max = (clocks["sm_max_mhz"] or 1965) * 1e6
        peak_tflops = SM_COUNT * FP32_LANES_PER_SM * 2 * f_max / 1e12
        a5_ms = max(km["eloc"], km["series_gemm"])
        achieved = 2.0 * ops["a5"] / (a5_ms * 1e-3) / 1e12
        path_floor_ms = (ops["a5"] + ops["a2"] + ops["a3"]) / (SM_COUNT * FP32_LANES_PER_SM * f_max) * 1e3
        line = {
            "metric": "E_loc samples/s", "value": value, "unit": "samples/s", "n_gpus": world, "steps": args.steps,
            "warmup": warm, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "N": w.N, "M": w.M, "B_per_gpu": w.B, "global_batch": plan["global_batch"],
                       "terms": w.ham.T, "flip_groups": ham.G, "table_columns": ham.C,
                       "connected_per_sample": ham.G + 1,
                       "l2": f"flushed between timed steps ({L2_FLUSH_BYTES >> 20} MiB write outside the event pairs)",
                       "parallelism": f"replicas over B x{world}, no collective"},
            "connected_evals_per_s": value * (ham.G + 1),
            "kernel_ms": km,
            "path_fraction_of_fp32_roofline": path_floor_ms / ms_per_step,
            "roofline": {"bound": "alu", "kernel": "eloc_kernel", "achieved": achieved, "peak": peak_tflops,
                         "unit": "TFLOP/s", "frac": achieved / peak_tflops,
                         "traffic": ELOC_KERNEL_DRAM_TRAFFIC_BYTES,
                         "peak_source": "148 SMs x 128 FP32 lanes x 2 x clocks.max.sm (DESIGN.md); FMA = 2 flop; "
                                        "algorithmic work = 8 FMA per (sample, column, hidden unit)"},
            "clocks": {k: clocks[k] for k in ("sm_mhz", "sm_max_mhz", "reasons")},
            "e2e": {"value": plan["global_batch"] / e2e_s, "unit": "samples/s", "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h},
            "gpu_launches": 6 * args.steps,  # table, pack_spins, pack_w, theta_mma, eloc, finalize
        }
        # SURVEY.md 8(f) items 1 + 3, reported beside the headline (not part of `value`): the force
        # vector of the same batch from the E_loc just computed (nqs_forces: stats, theta, pack, int8 GEMM)
        f_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(5)]
        for k in range(7):
            if k >= 2:
                flush.fill_(k)
                f_ev[k - 2][0].record()
            nqs.forces(spins, a, b, W, e)
            if k >= 2:
                f_ev[k - 2][1].record()
        torch.cuda.synchronize()
        f_ms = float(np.median([s0.elapsed_time(s1) for s0, s1 in f_ev]))
        line["forces"] = {"ms_per_call": f_ms, "samples_per_s": w.B / (f_ms * 1e-3), "parameters": w.N + w.M + w.M * w.N,
                          "what": "nqs_forces (Eq. 16) on the same batch, device-resident, median of 5, L2 flushed"}
        # one VMC evaluation step: E_loc + statistics + forces with theta computed once
        v_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(5)]
        for k in range(7):
            if k >= 2:
                flush.fill_(k)
                v_ev[k - 2][0].record()
            ham.local_energy_forces(spins, a, b, W)
            if k >= 2:
                v_ev[k - 2][1].record()
        torch.cuda.synchronize()
        v_ms = float(np.median([s0.elapsed_time(s1) for s0, s1 in v_ev]))
        line["vmc_step"] = {"ms_per_call": v_ms, "samples_per_s": w.B / (v_ms * 1e-3),
                            "what": "nqs_local_energy_forces_h: E_loc, mean/variance and force vector of one batch, "
                                    "theta and tanh(theta) computed once; median of 5, L2 flushed"}
        # one Metropolis sweep (N proposals per chain) of B chains, proposals and
        # uniforms drawn on the device beforehand (not timed), chains continue from the batch
        gen = torch.Generator(device=dev)
        gen.manual_seed(1234)
        m_sites = torch.randint(0, w.N, (w.N, w.B), device=dev, dtype=torch.int32, generator=gen)
        m_u = torch.rand((w.N, w.B), device=dev, dtype=torch.float32, generator=gen)
        chains = spins.clone()
        m_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(3)]
        acc = None
        for k in range(4):
            if k >= 1:
                m_ev[k - 1][0].record()
            acc = nqs.metropolis(chains, a, b, W, m_sites, m_u)
            if k >= 1:
                m_ev[k - 1][1].record()
        torch.cuda.synchronize()
        m_ms = float(np.median([s0.elapsed_time(s1) for s0, s1 in m_ev]))
        line["metropolis"] = {"ms_per_sweep": m_ms, "chains": w.B, "steps_per_sweep": w.N,
                              "proposals_per_s": w.B * w.N / (m_ms * 1e-3),
                              "acceptance": float(acc.float().mean().item()) / w.N,
                              "what": "nqs_metropolis, one sweep of all chains, median of 3"}
        del m_sites, m_u, chains
        # pipe rates measured on this box (nqs_microbench; register-only kernels, after the timed region)
        mb = {k: nqs.microbench(k)["lane_ops_per_s"] for k in nqs.MICROBENCH_KINDS}
        line["measured_peaks"] = {
            "ffma_tflops": 2 * mb["ffma"] / 1e12, "ffma2_tflops": 2 * mb["ffma2"] / 1e12,
            "a5_body_packed_tflops": 2 * mb["a5_body_packed"] / 1e12,
            "a5_body_scalar_tflops": 2 * mb["a5_body_scalar"] / 1e12,
            "mufu_ex2_gops": mb["mufu_ex2"] / 1e9,
            "how": "nqs_microbench: 2 x 320 threads per SM, operands in registers, best of 3; FMA = 2 flop"}
        line["roofline"]["frac_of_measured_ffma"] = achieved / (2 * max(mb["ffma"], mb["ffma2"]) / 1e12)
        if world == 1 and not args.no_cpu_baseline:
            cb, _, _ = cpu_baseline(w)
            line["cpu_baseline"] = cb
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
