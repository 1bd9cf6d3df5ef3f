#!/usr/bin/env python
"""bench.py — the headline measurement of BASELINE.json.

Metric: interactions/s (and ms per force evaluation = `ms_per_step`) of ONE force
evaluation — the whole hot path A1-A6 of DESIGN.md §1 (tree walk + interaction
list evaluation + write-back) — on config 3: Plummer sphere N = 2^20 (seed 3),
theta = 0.5, eps = 0.01, N_leaf = 16, N_group = 96 (tuned; option `n_group`), monopole+quadrupole, fp32.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A "step" is one `tc_forces` call through the C ABI on a tree that `tc_build`
(host, as in the paper — PAPER.md:17,41) built before the timed region.
  value : device-resident — particles, tree and outputs live in HBM; CUDA events
          on the launching stream around every step; L2 flushed between steps.
  e2e   : the call a user makes with HOST buffers every step —
          tc_set_particles(host) + tc_build (host tree, ONE bulk H2D) +
          tc_forces(host acc, pot) (D2H inside) — wall clock.
N > 1 (torchrun): the path shards over independent force evaluations — every rank
evaluates its own Plummer sphere (seed 3 + rank), no data-path collective; weak
scaling; time = max over ranks.

`--impl reference` times the fp64 CPU oracle (oracle/, test infrastructure) on a
bounded sample of the same workload; it is a baseline, not the target.
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

WORKLOAD = "plummer_1m"           # BASELINE.json configs[2]: the configuration the metric is quoted on
N_GROUP = 96
# flops per interaction, SASS convention (FFMA = 2, FADD/FMUL = 1, MUFU.RSQ = 1) — DESIGN.md §6
FLOPS_PC, FLOPS_PP = 54, 20
# paper convention (fn. 3)
PAPER_FLOPS_PC, PAPER_FLOPS_PP = 70, 38
# FP32 ALU peak: SMs x 128 lanes x 2 flops x clock
N_SM, LANES = 148, 128
L2_FLUSH_BYTES = 256 << 20        # > 126 MB L2
# DRAM bytes of one launch of the force kernel at config 3, from the committed ncu capture (profiles/)
DRAM_TRAFFIC_BYTES = 74562048


def fp32_peak_tflops(mhz: float) -> float:
    return N_SM * LANES * 2 * mhz * 1e6 / 1e12


class ClockSampler(threading.Thread):
    """Samples SM clock / throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period: float = 0.02):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.sm, self.reasons, self.power = [], set(), []
        self.sm_max = None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.nv = None

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        # NVML clocks-event-reason bits
        names = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
                 0x80: "hw_power_brake_slowdown"}
        while not self._stop_evt.is_set():
            try:
                self.sm.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, nm in names.items():
                    if r & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self) -> dict:
        self._stop_evt.set()
        if self.is_alive():
            self.join()
        if not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(self.sm)), "sm_max_mhz": self.sm_max, "reasons": sorted(self.reasons),
                "power_w_max": max(self.power) if self.power else None, "samples": len(self.sm)}


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def max_over_ranks(x: float, world: int, device=None) -> float:
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float, world: int, device=None) -> float:
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def cpu_baseline(pos, mass, theta, eps, n_leaf, target_s: float = 15.0) -> dict:
    """The fp64 oracle as it stands, timed on this box's host cores on a bounded sample of groups."""
    import oracle
    o = oracle.Oracle(pos, mass, n_leaf, N_GROUP)
    ng = o.n_groups
    probe = np.unique(np.linspace(0, ng - 1, min(ng, 128)).astype(np.int64))
    t0 = time.perf_counter()
    r = o.forces(theta, eps, shadow32=True, groups=probe)
    dt = time.perf_counter() - t0
    k = int(min(ng, max(len(probe), len(probe) * target_s / max(dt, 1e-3))))
    sel = np.unique(np.linspace(0, ng - 1, k).astype(np.int64))
    t0 = time.perf_counter()
    r = o.forces(theta, eps, shadow32=True, groups=sel)
    dt = time.perf_counter() - t0
    return {"value": r["interactions"] / dt, "unit": "interactions/s", "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"{len(sel)} of {ng} groups (evenly spaced in Morton order), {r['interactions']} interactions, "
                      f"{dt:.2f} s walk+evaluate in fp64 (tree build excluded)",
            "seconds": dt}


def run_ours(args) -> None:
    import torch
    rank, world, local = dist_env()
    if world != args.gpus:
        if world == 1 and args.gpus > 1:
            raise SystemExit("bench.py --gpus N>1 must be launched with torch.distributed.run (one rank per GPU)")
    assert torch.cuda.is_available(), "bench.py needs a CUDA device: there is no CPU fallback for the product path"
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    from paper_1005_5384_b200 import binding as B
    from paper_1005_5384_b200 import build as tc_build
    from paper_1005_5384_b200 import inputs
    if rank == 0:
        tc_build.build()
    if world > 1:
        dist.barrier()

    fn, kw, theta, eps, n_leaf = inputs.WORKLOADS[WORKLOAD]
    kw = dict(kw, seed=kw["seed"] + rank)            # rank r evaluates its own sphere (weak scaling)
    pos, mass = fn(**kw)
    n = len(mass)
    K, W = args.steps, args.warmup

    stream = torch.cuda.Stream(device=dev)
    tc = B.TreeCode(n_group=N_GROUP)
    tc.set_stream(stream.cuda_stream)
    with torch.cuda.stream(stream):
        d_pos, d_mass = torch.from_numpy(pos).to(dev), torch.from_numpy(mass).to(dev)
        d_acc = torch.empty((n, 3), dtype=torch.float32, device=dev)
        d_pot = torch.empty(n, dtype=torch.float32, device=dev)
        flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
        tc.set_particles(d_pos, d_mass)
        tc.build(n_leaf)

        def step():
            B.tc_forces(tc.ctx, theta, eps, d_acc, d_pot)

        for _ in range(W):
            flush.zero_()
            step()
        tc.sync()
        st = tc.stats()
        inter = st["n_pc_total"] + st["n_pp_total"]
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
        sampler = ClockSampler(local)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        sampler.start()
        t_wall0 = time.perf_counter()
        for i in range(K):
            flush.zero_()                              # L2 flush between timed iterations (outside the events)
            ev[i][0].record(stream)
            step()
            ev[i][1].record(stream)
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        t_wall = time.perf_counter() - t_wall0
        clocks = sampler.stop()
        tc.sync()
        per_step = [a.elapsed_time(b) for a, b in ev]
        t_dev_ms = float(sum(per_step))                # device time of exactly K steps
        st = tc.stats()

        # ---- the paper's second metric: data rate of the tree walk alone (A1-A3), lists dropped
        tc.set_option("walk_only", 1)
        walk_ms = []
        for i in range(5):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream); step(); b.record(stream)
            torch.cuda.synchronize()
            walk_ms.append(a.elapsed_time(b))
        tc.set_option("walk_only", 0)
        tc.sync()
        walk_ms = float(np.median(walk_ms[1:]))

        # ---- e2e: host buffers through the C ABI, every step: set_particles + build + forces
        h_pos = torch.from_numpy(pos).pin_memory().numpy()
        h_mass = torch.from_numpy(mass).pin_memory().numpy()
        h_acc = torch.empty((n, 3), dtype=torch.float32).pin_memory().numpy()
        h_pot = torch.empty(n, dtype=torch.float32).pin_memory().numpy()
        Ke = max(3, min(K, 10))
        t_e2e, t_host, t_copy = [], [], []
        for i in range(2 + Ke):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            tc.set_particles(h_pos, h_mass)
            tc.build(n_leaf)
            tc.forces(theta, eps, h_acc, h_pot)
            dt = time.perf_counter() - t0
            if i >= 2:
                t_e2e.append(dt)
                s2 = tc.stats()
                t_host.append(s2["t_host_ms"]); t_copy.append(s2["t_copy_ms"])
        e2e_s = float(np.mean(t_e2e))
        # the same call sequence with the device-side tree build (option "device_build")
        tc.set_option("device_build", 1)
        t_e2e_dev = []
        for i in range(2 + Ke):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            tc.set_particles(h_pos, h_mass)
            tc.build(n_leaf)
            tc.forces(theta, eps, h_acc, h_pot)
            if i >= 2:
                t_e2e_dev.append(time.perf_counter() - t0)
        e2e_dev_s = float(np.mean(t_e2e_dev))
        t_build_dev = tc.stats()["t_host_ms"]
        tc.set_option("device_build", 0)
        tree_bytes = st["tree_bytes"]
        measured_peak = B.tc_fp32_peak(tc.ctx)       # FFMA-only microbenchmark on this device, after the timed region
    tc.close()

    t_dev_ms = max_over_ranks(t_dev_ms, world, dev)
    e2e_s = max_over_ranks(e2e_s, world, dev)
    e2e_dev_s = max_over_ranks(e2e_dev_s, world, dev)
    inter_all = sum_over_ranks(float(inter), world, dev)
    n_all = sum_over_ranks(float(n), world, dev)
    flops = FLOPS_PC * st["n_pc_total"] + FLOPS_PP * st["n_pp_total"]
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    ms = t_dev_ms / K
    value = inter_all / (ms * 1e-3)
    kernel_ms = float(np.mean(per_step))
    ach = flops / (kernel_ms * 1e-3) / 1e12
    sm_max = clocks.get("sm_max_mhz") or 1965.0
    peak = fp32_peak_tflops(sm_max)
    out = {
        "metric": "interactions/s of one force evaluation (tree walk + list evaluation), N=2^20 Plummer, theta=0.5; "
                  "ms per force evaluation is ms_per_step",
        "value": value, "unit": "interactions/s", "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[2]: Plummer N={n} seed 3(+rank), eps={eps}, theta={theta}, "
                               f"N_leaf={n_leaf}, N_group={N_GROUP}, monopole+quadrupole",
                   "n": n, "theta": theta, "eps": eps, "n_leaf": n_leaf, "n_group": N_GROUP,
                   "l2": f"flushed between timed steps ({L2_FLUSH_BYTES >> 20} MiB memset outside the events)",
                   "sharding": "one independent force evaluation per rank, no collective"},
        "particles_per_s": n_all / (ms * 1e-3),
        "interactions_per_step": inter_all, "n_pc": st["n_pc_total"], "n_pp": st["n_pp_total"],
        "opening_tests": st["n_tests_total"], "n_groups": st["n_groups"], "n_cells": st["n_cells"],
        "gflops_paper_convention": (PAPER_FLOPS_PC * st["n_pc_total"] + PAPER_FLOPS_PP * st["n_pp_total"])
                                   / (kernel_ms * 1e-3) / 1e9,
        "ms_per_step_min": float(min(per_step)), "ms_per_step_median": float(np.median(per_step)),
        "wall_ms_per_step_incl_flush": t_wall * 1e3 / K,
        "walk": {"ms": walk_ms, "bytes_per_test": 64, "gb_per_s": 64.0 * st["n_tests_total"] / (walk_ms * 1e-3) / 1e9,
                 "what": "option walk_only: walk + list building without evaluation; 4 float4 loads per opening test "
                         "(L2-resident tree); the paper reports > 50 GB/s for its count pass on G80 (PAPER.md:177)"},
        "gpu_launches": K,
        "clocks": clocks,
        "e2e": {"value": inter_all / e2e_s, "unit": "interactions/s", "h2d_bytes_per_step": int(tree_bytes),
                "d2h_bytes_per_step": int(16 * n), "ms_per_step": e2e_s * 1e3,
                "t_host_build_ms": float(np.mean(t_host)), "t_copy_ms": float(np.mean(t_copy)),
                "what": "tc_set_particles(host)+tc_build(host octree, one bulk H2D)+tc_forces(host acc,pot); wall clock"},
        "e2e_device_build": {"value": inter_all / e2e_dev_s, "unit": "interactions/s", "h2d_bytes_per_step": int(16 * n),
                             "d2h_bytes_per_step": int(16 * n), "ms_per_step": e2e_dev_s * 1e3, "t_build_ms": float(t_build_dev),
                             "what": "same calls with tc_set_option('device_build', 1): particles H2D, tree built on the GPU"},
        "roofline": {"bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                     "traffic": DRAM_TRAFFIC_BYTES, "kernel": "tc::forces_kernel",
                     "peak_how": f"nominal: {N_SM} SMs x {LANES} FP32 lanes x 2 x {sm_max:.0f} MHz (DESIGN.md §6; "
                                 "MEASURED_PEAKS.json holds HBM and bf16 figures only, no FP32 entry)",
                     "peak_measured": measured_peak, "frac_of_measured": ach / measured_peak,
                     "peak_measured_how": "tc_fp32_peak: FFMA-only microbenchmark on this device in this run",
                     "flops_per_launch": flops, "algorithmic_bytes_per_launch": int(tree_bytes + 24 * n),
                     "traffic_how": "dram__bytes_read.sum + dram__bytes_write.sum of one ncu --set full capture "
                                    "(profiles/r01d_final.md); HBM is not the bound"},
    }
    out["cpu_baseline"] = cpu_baseline(*inputs.make(WORKLOAD)) if world == 1 else None
    print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_reference(args) -> None:
    """The oracle (fp64 CPU, as it stands) on a bounded sample of the same workload; rank 0 only."""
    rank, world, _ = dist_env()
    if rank != 0:
        return
    import oracle
    from paper_1005_5384_b200 import inputs
    pos, mass, theta, eps, n_leaf = inputs.make(WORKLOAD)
    n = len(mass)
    o = oracle.Oracle(pos, mass, n_leaf, N_GROUP)
    ng = o.n_groups
    K, W = args.steps, args.warmup
    # size the per-step sample so that the K + W steps take about two minutes in total
    probe = np.unique(np.linspace(0, ng - 1, 64).astype(np.int64))
    t0 = time.perf_counter()
    o.forces(theta, eps, shadow32=True, groups=probe)
    dt = time.perf_counter() - t0
    per_step_s = min(20.0, 120.0 / max(1, K + W))
    k = int(min(ng, max(64, 64 * per_step_s / max(dt, 1e-3))))
    sel = np.unique(np.linspace(0, ng - 1, k).astype(np.int64))
    for _ in range(W):
        o.forces(theta, eps, shadow32=True, groups=sel)
    t_all, inter = 0.0, 0
    for _ in range(K):
        t0 = time.perf_counter()
        r = o.forces(theta, eps, shadow32=True, groups=sel)
        t_all += time.perf_counter() - t0
        inter = r["interactions"]
    value = inter * K / t_all
    sample = f"{len(sel)} of {ng} groups per step (evenly spaced in Morton order), {inter} interactions per step"
    out = {
        "impl": "reference",
        "metric": "interactions/s of one force evaluation (tree walk + list evaluation), N=2^20 Plummer, theta=0.5; "
                  "ms per force evaluation is ms_per_step",
        "value": value, "unit": "interactions/s", "n_gpus": args.gpus, "steps": K, "warmup": W,
        "ms_per_step": t_all * 1e3 / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[2]: Plummer N={n} seed 3, eps={eps}, theta={theta}, "
                               f"N_leaf={n_leaf}, N_group={N_GROUP}, monopole+quadrupole",
                   "n": n, "theta": theta, "eps": eps, "n_leaf": n_leaf, "n_group": N_GROUP,
                   "sample": sample},
        "cpu_baseline": {"value": value, "unit": "interactions/s", "cores": oracle.num_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": "interactions/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out), flush=True)


def main() -> None:
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
