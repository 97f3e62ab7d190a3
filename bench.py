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
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from `ncu --set full` captures
# summarised under profiles/ -- (workload, kernel) -> (bytes, file).  No capture for that pair => traffic is null.
NCU_DRAM_TRAFFIC = {
    ("c5_tfim_20x20", "eloc_kernel"): (897_815_552, "profiles/r1_v3_ncu_summary.md"),
    ("c5_tfim_20x20", "series_gemm_kernel"): (2_228_427_000, "profiles/r2e_ncu_summary.md"),
    ("c2_tfim_chain_N40", "small_eloc_kernel"): (780_800, "profiles/r2e_ncu_summary.md"),
}
# nominal ratio of the dense INT8 to the dense BF16/FP16 tensor peak (B200_PROFILING.md: 4.5 vs 2.25 P)
INT8_OVER_BF16 = 2.0


def measured_peaks() -> dict:
    """MEASURED_PEAKS.json (driver-written) or the profiling guide's stated fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return dict(bf16_tflops=float(d["bf16_tflops"]), bf16_tflops_sustained=float(d.get("bf16_tflops_sustained", 0.0)),
                    hbm_gbs=float(d["hbm_gbs"]), source="MEASURED_PEAKS.json (of measured)")
    return dict(bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, hbm_gbs=6650.0,
                source="B200_PROFILING.md fallback (of fallback)")


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


def algorithmic_work(w: wl.Workload, C: int) -> dict:
    """Algorithmic work per step (DESIGN.md sections 6 and 12).
    a5_fp32   product form: 8 FP32 FMA per (sample, column, hidden unit)
    a5_tensor series form: 5 complex FP16 products (k = 1 as hi.hi + hi.lo + lo.hi, k = 2, k = 3) = 20 real MACs
    a2_fp32   theta as FP32 add/sub: 2 N M lane-ops per sample (SIMT kernel)
    a2_int8   theta as 4 int8 digits x (re, im) = 8 N M int8 MACs per sample (tensor-core kernel)
    a3_fp32   ~40 FP32 per (sample, hidden unit)"""
    B, N, M = float(w.B), float(w.N), float(w.M)
    return dict(a5_fp32=8.0 * B * C * M, a5_tensor=20.0 * B * C * M, a2_fp32=2.0 * B * N * M, a2_int8=8.0 * B * N * M,
                a3_fp32=40.0 * B * M)


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
    """The float64 oracle, as it stands, on the host cores, on bounded prefixes of the same batch: fast mode
    (OpenMP over samples) on all threads -- the `value` -- plus the 1-thread figure and definition mode on a
    smaller subset (SURVEY.md 8(d) "Oracle timing")."""
    import oracle

    oracle.build()
    cores = oracle.num_threads()
    args = (w.a, w.b, w.W, w.ham.sites, w.ham.paulis, w.ham.coeffs)

    def timed(fn, n):
        t0 = time.perf_counter()
        fn(w.spins[:n], *args)
        return max(time.perf_counter() - t0, 1e-6)

    n0 = min(w.B, cores)
    dt0 = timed(oracle.local_energy_fast, n0)
    n = int(min(w.B, max(n0, (budget_s / dt0) * n0)))
    n = max(min(cores, w.B), n // cores * cores)
    dt = timed(oracle.local_energy_fast, n)
    # one thread, ~3 s
    oracle.set_num_threads(1)
    try:
        n1 = int(min(w.B, max(1, 3.0 / (dt / n * cores))))
        dt1 = timed(oracle.local_energy_fast, n1)
    finally:
        oracle.set_num_threads(cores)
    # definition mode (Algorithm 1 lines 6-8 literally), all threads, ~4 s
    nd0 = min(w.B, cores)
    dtd0 = timed(oracle.local_energy_definition, nd0)
    nd = int(min(w.B, max(nd0, (4.0 / dtd0) * nd0)))
    nd = max(min(cores, w.B), nd // cores * cores)
    dtd = timed(oracle.local_energy_definition, nd) if nd > nd0 else dtd0
    return dict(value=n / dt, unit="samples/s", cores=cores, kind="oracle",
                sample=f"fast mode (float64, flip grouping + low-rank theta update), first {n} of {w.B} samples "
                       f"of {w.name}, {dt:.2f} s wall, OpenMP {cores} threads",
                one_thread={"value": n1 / dt1, "unit": "samples/s", "sample": f"fast mode, first {n1} samples, {dt1:.2f} s"},
                definition_mode={"value": nd / dtd, "unit": "samples/s", "cores": cores,
                                 "sample": f"definition mode, first {nd} samples, {dtd:.2f} s wall"})


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

    def timed_steps(n_steps, n_warm):
        """n_warm untimed steps, then n_steps steps each bracketed by CUDA events on the launching stream; the L2
        is flushed (256 MiB write) between steps, outside the event pairs.  Returns (total ms, max over ranks;
        per-kernel ms; clocks; kernel launches in the timed steps; last outputs)."""
        for _ in range(n_warm):
            out = step()
        torch.cuda.synchronize()
        sampler = ClockSampler(local_rank)
        nqs.profile_enable(True)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_steps)]
        kern_ms = []
        barrier()
        launches0 = nqs.launch_count()
        sampler.start()
        for k in range(n_steps):
            flush.fill_(k & 0xFF)
            ev[k][0].record()
            out = step()
            ev[k][1].record()
            if k == n_steps - 1 or k % 4 == 3:
                kern_ms.append(nqs.profile_last())
        barrier()
        clocks = sampler.stop()
        launches = nqs.launch_count() - launches0
        nqs.profile_enable(False)
        total_ms = float(np.sum([s0.elapsed_time(s1) for s0, s1 in ev]))
        if world > 1:
            tt = torch.tensor([total_ms], dtype=torch.float64, device=dev)
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            total_ms = float(tt.item())
        km = {k: float(np.median([d[k] for d in kern_ms])) for k in kern_ms[0]}
        return total_ms, km, clocks, launches, out

    warm = max(args.warmup, 3)
    # ---- the product (default path: tensor-core series for a5 where it applies, guarded, FP32 fallback behind it)
    total_ms, km, clocks, launches, (e, l) = timed_steps(args.steps, warm)
    took = nqs.debug_last_a5()
    ms_per_step = total_ms / args.steps
    value = plan["global_batch"] / (ms_per_step * 1e-3)
    # ---- beside it: the same steps with a5 forced onto the FP32 product form (the round-1 path)
    nqs.set_option("a5_path", nqs.A5_PATHS["product"])
    try:
        n_prod = max(3, min(args.steps, 10))
        p_total_ms, p_km, _, _, (e_prod, _) = timed_steps(n_prod, 3)
    finally:
        nqs.set_option("a5_path", 0)
    p_ms_per_step = p_total_ms / n_prod

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
        work = algorithmic_work(w, ham.C)
        peaks = measured_peaks()
        f_max = (clocks["sm_max_mhz"] or 1965) * 1e6
        fp32_peak_lane = SM_COUNT * FP32_LANES_PER_SM * f_max          # lane-FMA / s
        fp32_peak_tflops = 2 * fp32_peak_lane / 1e12
        series = took["path"] == "series" and not took["guard_failed"]
        theta_on_tensor = w.N <= 512
        # dominant kernel of the step and its roofline
        if series:
            dom, dom_ms = "series_gemm_kernel", km["series_gemm"]
            achieved = 2.0 * work["a5_tensor"] / (dom_ms * 1e-3) / 1e12
            roof = {"bound": "tensor", "kernel": dom, "achieved": achieved, "peak": peaks["bf16_tflops"],
                    "unit": "TFLOP/s", "frac": achieved / peaks["bf16_tflops"],
                    "peak_source": f"{peaks['source']}: cuBLAS bf16 burst figure (FP16 and BF16 share the tcgen05 "
                                   "kind::f16 rate); algorithmic work = 20 real FP16 MACs per (sample, column, hidden "
                                   "unit), padding columns not counted",
                    "frac_of_sustained_peak": (achieved / peaks["bf16_tflops_sustained"]
                                               if peaks["bf16_tflops_sustained"] else None),
                    # SURVEY 8(f)4 counts the series as K = 3 complex GEMMs = 12 real MACs per triple; the other 8 of
                    # the 20 are the hi + lo split that FP16 operands need for the k = 1 term
                    "frac_12mac": achieved / peaks["bf16_tflops"] * 12.0 / 20.0}
        else:
            dom, dom_ms = ("small_eloc_kernel" if took["path"] == "small" else "eloc_kernel"), km["eloc"]
            achieved = 2.0 * work["a5_fp32"] / (dom_ms * 1e-3) / 1e12
            roof = {"bound": "alu", "kernel": dom, "achieved": achieved, "peak": fp32_peak_tflops, "unit": "TFLOP/s",
                    "frac": achieved / fp32_peak_tflops,
                    "peak_source": "148 SMs x 128 FP32 lanes x 2 x clocks.max.sm (DESIGN.md); FMA = 2 flop; "
                                   "algorithmic work = 8 FMA per (sample, column, hidden unit)"}
        traffic = NCU_DRAM_TRAFFIC.get((w.name, dom))
        if (w.name, dom) == ("c5_tfim_20x20", "series_gemm_kernel"):
            # context from the same ncu capture (not measured in this run): the chip is power-limited under tensor load
            roof["ncu_context"] = {"sm_ghz_during_kernel": 1.48, "tensor_pipe_active": 0.837,
                                   "l2_to_sm_fill_bytes": 9_121_392_000, "source": "profiles/r2e_ncu_summary.md"}
        roof["traffic"] = traffic[0] if traffic else None
        roof["traffic_source"] = traffic[1] if traffic else "no ncu --set full capture of this kernel at this workload"
        # FP32 floor of the cheapest FP32 formulation (SURVEY 8(d) rule (i)): product-form a5 + per-unit work, and a2
        # only when theta really runs on the FP32 pipe.  With a5 on the tensor cores the step can beat this floor;
        # the ratio is then > 1 and is a speed-up over the FP32 roofline, not a fraction of it.
        fp32_floor_ms = (work["a5_fp32"] + work["a3_fp32"] + (0.0 if theta_on_tensor else work["a2_fp32"])) / fp32_peak_lane * 1e3
        p_achieved = 2.0 * work["a5_fp32"] / (p_km["eloc"] * 1e-3) / 1e12
        line = {
            "metric": "E_loc samples/s", "value": value, "unit": "samples/s", "n_gpus": world, "steps": args.steps,
            "warmup": warm, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f16 x f16 -> f32 (tcgen05, k = 1 operands split hi + lo) for a5; int8 -> s32 for "
                                          "theta; f32 elsewhere" if series else "f32",
            "data": "synthetic",
            "config": {"workload": w.name, "N": w.N, "M": w.M, "B_per_gpu": w.B, "global_batch": plan["global_batch"],
                       "terms": w.ham.T, "flip_groups": ham.G, "table_columns": ham.C,
                       "connected_per_sample": ham.G + 1, "a5_path": "tensor-core series (guard passed)" if series else
                       ("FP32 product form (series guard failed)" if took["path"] == "series" else
                        "FP32 product form, single launch" if took["path"] == "small" else "FP32 product form"),
                       "l2": f"flushed between timed steps ({L2_FLUSH_BYTES >> 20} MiB write outside the event pairs)",
                       "parallelism": f"replicas over B x{world}, no collective"},
            "connected_evals_per_s": value * (ham.G + 1),
            "kernel_ms": km,
            "fp32_floor_ms": fp32_floor_ms,
            "path_fraction_of_fp32_roofline": fp32_floor_ms / ms_per_step,
            "roofline": roof,
            "clocks": {k: clocks[k] for k in ("sm_mhz", "sm_max_mhz", "reasons")},
            "e2e": {"value": plan["global_batch"] / e2e_s, "unit": "samples/s", "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h},
            "gpu_launches": int(launches),
            "product_form": {"ms_per_step": p_ms_per_step, "samples_per_s": plan["global_batch"] / (p_ms_per_step * 1e-3),
                             "kernel_ms": p_km, "steps": n_prod,
                             "roofline": {"bound": "alu", "kernel": "eloc_kernel", "achieved": p_achieved,
                                          "peak": fp32_peak_tflops, "unit": "TFLOP/s", "frac": p_achieved / fp32_peak_tflops},
                             "path_fraction_of_fp32_roofline": fp32_floor_ms / p_ms_per_step,
                             "max_abs_diff_vs_default_path": float((e_prod - e).abs().max().item()),
                             "what": "the same steps with NQS_OPT_A5_PATH = 1 (FP32 product form, the round-1 path)"},
        }
        if theta_on_tensor:
            th_tops = 2.0 * work["a2_int8"] / (km["theta"] * 1e-3) / 1e12
            int8_peak = INT8_OVER_BF16 * peaks["bf16_tflops"]
            line["theta_tensor"] = {"ms": km["theta"], "achieved_tops": th_tops, "peak_tops": int8_peak,
                                    "frac": th_tops / int8_peak,
                                    "what": "pack_spins + pack_w + theta_mma_kernel (a2 + a3); 8 N M int8 MACs per sample; "
                                            f"peak = {INT8_OVER_BF16:g} x measured bf16 (nominal int8 : bf16 ratio)"}
        if w.meta.get("config") == 4:
            # Q12: half of the pair-flip columns have a zero matrix element per sample (parallel bonds)
            s64 = w.spins.astype(np.int64)
            bonds = np.array(wl.square_bonds(w.meta["L"]))
            nonzero = float((s64[:, bonds[:, 0]] * s64[:, bonds[:, 1]] < 0).sum(axis=1).mean())
            roof["frac_of_nonzero_work"] = roof["frac"] * nonzero / ham.C
            line["product_form"]["roofline"]["frac_of_nonzero_work"] = p_achieved / fp32_peak_tflops * nonzero / ham.C
            line["config"]["nonzero_columns_per_sample"] = nonzero
            line["connected_evals_per_s_nonzero"] = value * (nonzero + 1)
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
        # trained-scale parameters (10 x the configuration's sigma: far outside the series guard's window), automatic
        # path, a fresh handle: the first call attempts the series and is refused; the refusal latch then sends the
        # following calls to the product form alone and probes the series again after 8, 16, ... calls
        if series:
            sig_t = 10.0 * w.meta["sigma"]
            ta, tb, tW = (torch.from_numpy(x).to(dev) for x in wl.rbm_parameters(w.N, w.M, sig_t, [w.meta["seed"], 9]))
            ham_t = nqs.Hamiltonian(w.N, w.ham.sites, w.ham.paulis, w.ham.coeffs)
            n_t = 20
            t_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_t)]
            t_paths = []
            for k in range(n_t):
                flush.fill_(k)
                t_ev[k][0].record()
                ham_t.local_energy(spins, ta, tb, tW)
                t_ev[k][1].record()
                tk = nqs.debug_last_a5()  # synchronises, as a VMC loop does when it reads the energies
                t_paths.append("series refused" if tk["path"] == "series" and tk["guard_failed"] else tk["path"])
            t_ms = [s0.elapsed_time(s1) for s0, s1 in t_ev]
            # the forced product form at the SAME parameters (larger theta: the closed-form log cosh / tanh branch)
            nqs.set_option("a5_path", nqs.A5_PATHS["product"])
            try:
                tp_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(5)]
                for k in range(7):
                    if k >= 2:
                        flush.fill_(k)
                        tp_ev[k - 2][0].record()
                    ham_t.local_energy(spins, ta, tb, tW)
                    if k >= 2:
                        tp_ev[k - 2][1].record()
                torch.cuda.synchronize()
            finally:
                nqs.set_option("a5_path", 0)
            tp_ms = float(np.median([s0.elapsed_time(s1) for s0, s1 in tp_ev]))
            ham_t.close()
            line["trained_scale"] = {
                "sigma": sig_t, "first_call_ms": t_ms[0], "refused_call_ms": float(np.mean(t_ms[1:])),
                "median_call_ms": float(np.median(t_ms[1:])), "calls": n_t,
                "series_attempts": int(sum(p_ != "product" for p_ in t_paths)),
                "product_form_ms": tp_ms, "paths": t_paths,
                "what": "same batch and Hamiltonian, parameters ~ N(0, sigma^2) at 10 x the configuration's sigma, automatic "
                        "a5 path on a fresh handle; refused_call_ms = mean over calls 2..20 (includes the latch's re-probe "
                        "after 8 product-form calls), median_call_ms = their median; product_form_ms = the forced product "
                        "form at the same parameters (median of 5)"}
        # SURVEY.md 8(f) items 1 + 3: the quantum Fisher matrix S = <<O* O>>_c of the same batch (K <= 8192 parameters)
        K = w.N + w.M + w.M * w.N
        if K <= 8192:
            s_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(5)]
            for k in range(7):
                if k >= 2:
                    flush.fill_(k)
                    s_ev[k - 2][0].record()
                nqs.fisher(spins, a, b, W)
                if k >= 2:
                    s_ev[k - 2][1].record()
            torch.cuda.synchronize()
            s_ms = float(np.median([s0.elapsed_time(s1) for s0, s1 in s_ev]))
            macs = 12.0 * w.B * K * (K + 128) / 2.0  # upper-triangle tiles, 3 split products x 4 real MACs
            line["fisher"] = {"ms_per_call": s_ms, "parameters": K, "achieved_tflops": 2.0 * macs / (s_ms * 1e-3) / 1e12,
                              "frac_of_bf16_peak": 2.0 * macs / (s_ms * 1e-3) / 1e12 / peaks["bf16_tflops"],
                              "what": "nqs_fisher (Eq. 10-11): theta, <O> (int8 GEMM), operand packing and the FP16 tcgen05 "
                                      "GEMM over the samples of the upper-triangle tile pairs; median of 5, L2 flushed"}
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
        # the shared-site variant: the same sweep with one proposal site per step for all chains
        m_sites1 = torch.randint(0, w.N, (w.N,), device=dev, dtype=torch.int32, generator=gen)
        chains = spins.clone()
        ms_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(3)]
        for k in range(4):
            if k >= 1:
                ms_ev[k - 1][0].record()
            acc_s = nqs.metropolis_shared(chains, a, b, W, m_sites1, m_u)
            if k >= 1:
                ms_ev[k - 1][1].record()
        torch.cuda.synchronize()
        ms_ms = float(np.median([s0.elapsed_time(s1) for s0, s1 in ms_ev]))
        line["metropolis_shared"] = {"ms_per_sweep": ms_ms, "chains": w.B, "steps_per_sweep": w.N,
                                     "proposals_per_s": w.B * w.N / (ms_ms * 1e-3),
                                     "acceptance": float(acc_s.float().mean().item()) / w.N,
                                     "what": "nqs_metropolis_shared (one proposal site per step for all chains: table rows "
                                             "staged once per block, chain state in registers), median of 3"}
        del m_sites, m_u, chains
        # pipe rates measured on this box (nqs_microbench; register-only kernels, after the timed region)
        mb = {k: nqs.microbench(k)["lane_ops_per_s"] for k in nqs.MICROBENCH_KINDS}
        line["measured_peaks"] = {
            "ffma_tflops": 2 * mb["ffma"] / 1e12, "ffma2_tflops": 2 * mb["ffma2"] / 1e12,
            "a5_body_packed_tflops": 2 * mb["a5_body_packed"] / 1e12,
            "a5_body_scalar_tflops": 2 * mb["a5_body_scalar"] / 1e12,
            "mufu_ex2_gops": mb["mufu_ex2"] / 1e9,
            "how": "nqs_microbench: 2 x 320 threads per SM, operands in registers, best of 3; FMA = 2 flop"}
        line["product_form"]["roofline"]["frac_of_measured_ffma"] = p_achieved / (2 * max(mb["ffma"], mb["ffma2"]) / 1e12)
        if not series:
            line["roofline"]["frac_of_measured_ffma"] = achieved / (2 * max(mb["ffma"], mb["ffma2"]) / 1e12)
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(w)
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
