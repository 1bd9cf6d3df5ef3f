#!/usr/bin/env python
"""bench.py — the headline measurement of BASELINE.json.

Metric: interactions/s (and ms per force evaluation = `ms_per_step`) of ONE force
evaluation — the whole hot path A1-A6 of DESIGN.md section 1 (tree walk + interaction
list evaluation + write-back) — on config 3: Plummer sphere N = 2^20 (seed 3),
theta = 0.5, eps = 0.01, N_leaf = 16, N_group = 128 (tuned; option `n_group`), monopole+quadrupole, fp32.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A "step" is one `tc_forces` call through the C ABI on a tree that `tc_build`
(host, as in the paper — PAPER.md:17,41) built before the timed region.
  value : device-resident — particles, tree and outputs live in HBM; CUDA events
          on the launching stream around every step; L2 flushed between steps.
  e2e   : the call a user makes with HOST buffers every step —
          tc_set_particles(host) + tc_build (host tree, ONE bulk H2D) +
          tc_forces(host acc, pot) (D2H inside) — wall clock; pinned and pageable buffers.
Beside the headline the N = 1 line carries: `parity` (the timed launch against the oracle,
every group the oracle leg walked), `paper_literal` (N_group = N_leaf = 16), `config5`
(N = 2^24, the size at which the tree streams from HBM), `walk` (the paper's second metric).
N > 1 (torchrun): ONE force evaluation of the same config 3 sharded over the ranks (strong scaling):
every rank holds the particles and the tree, evaluates every N-th group of the schedule, one all-gather
of 16 bytes per particle, scatter to the caller's order (`paper_1005_5384_b200.parallel`); time = max over ranks.

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
N_GROUP = 128
# flops per interaction, SASS convention (FFMA = 2, FADD/FMUL = 1, MUFU.RSQ = 1) — DESIGN.md section 6
FLOPS_PC, FLOPS_PP = 54, 20
# paper convention (fn. 3)
PAPER_FLOPS_PC, PAPER_FLOPS_PP = 70, 38
# FP32 ALU peak: SMs x 128 lanes x 2 flops x clock
N_SM, LANES = 148, 128
L2_FLUSH_BYTES = 256 << 20        # > 126 MB L2
ACC_Q999, ACC_MAX, POT_MAX = 1e-4, 1e-3, 1e-4      # north_star tolerances
# SURVEY.md 8(d)'s own count (one flop fewer per interaction than the SASS convention above)
SURVEY_FLOPS_PC, SURVEY_FLOPS_PP = 53, 19
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "traffic.json")   # DRAM bytes per launch from committed ncu captures


def fp32_peak_tflops(mhz: float) -> float:
    return N_SM * LANES * 2 * mhz * 1e6 / 1e12


def measured_peaks() -> dict:
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except Exception:
        return {}


KERNEL_SOURCES = ["tc_kernels.cu", "tc_kernels_dense.cu", "tc_lanes.h", "tc_internal.h"]   # what tc::forces_kernel is compiled from


def kernel_source_sha16() -> str:
    """sha256 (first 16 hex digits) over the sources of the force kernel, in KERNEL_SOURCES order."""
    import hashlib
    h = hashlib.sha256()
    for name in KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_1005_5384_b200", "csrc", name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def traffic(key: str):
    """DRAM bytes of one launch (dram__bytes_read.sum + dram__bytes_write.sum) of a committed ncu capture, or None.
    The capture is a static file: `traffic_stale` says whether the kernel sources have changed since it was taken
    (profiles/traffic.json records their hash), so a figure from an older binary cannot pass as this run's."""
    try:
        with open(TRAFFIC_JSON) as f:
            doc = json.load(f)
        t = doc.get(key)
        if t is not None:
            t = dict(t)
            t["kernel_source_sha16_at_capture"] = doc.get("kernel_source_sha16")
            t["traffic_stale"] = bool(doc.get("kernel_source_sha16") != kernel_source_sha16())
        return t
    except Exception:
        return None


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


def cpu_baseline(pos, mass, theta, eps, n_leaf, target_s: float = 30.0):
    """The fp64 oracle as it stands, timed on this box's host cores on a bounded sample of groups (all of them when
    that fits the budget).  Returns (cpu_baseline object, oracle result, group sample) — the result also serves
    the `parity` object: nothing the oracle computes here is thrown away."""
    import oracle
    o = oracle.Oracle(pos, mass, n_leaf, N_GROUP)
    ng = o.n_groups
    probe = np.unique(np.linspace(0, ng - 1, min(ng, 256)).astype(np.int64))
    o.forces(theta, eps, shadow32=True, groups=probe[:16])       # spin the OpenMP threads up before the probe is timed
    t0 = time.perf_counter()
    r = o.forces(theta, eps, shadow32=True, groups=probe)
    dt = time.perf_counter() - t0
    k = int(min(ng, max(len(probe), len(probe) * target_s / max(dt, 1e-3))))   # all groups when that fits target_s (it does: ~5 s)
    sel = np.unique(np.linspace(0, ng - 1, k).astype(np.int64))
    t0 = time.perf_counter()
    r = o.forces(theta, eps, shadow32=True, groups=sel, stats=True)
    dt = time.perf_counter() - t0
    # R16 audit of the groups whose fp32 decision differs somewhere: bookkeeping, outside the timed part
    r["flip_audit"] = oracle.flip_audit(o, theta, r["flips"], sel)
    obj = {"value": r["interactions"] / dt, "unit": "interactions/s", "cores": oracle.num_threads(), "kind": "oracle",
           "sample": f"{len(sel)} of {ng} groups (evenly spaced in Morton order), {r['interactions']} interactions, "
                     f"{dt:.2f} s walk+evaluate in fp64 (tree build excluded)",
           "seconds": dt}
    return obj, r, sel, ng


def parity_object(ref, sel, ng, acc, pot, n_pc, n_pp) -> dict:
    """The timed launch's result against the oracle (fp32-shadow opening decisions, R16) on every particle
    of the groups the cpu_baseline leg walked; north_star tolerances."""
    m = ref["n_pc"] >= 0
    a64 = acc[m].astype(np.float64)
    rel = np.linalg.norm(a64 - ref["acc"][m], axis=1) / np.linalg.norm(ref["acc"][m], axis=1)
    prel = np.abs(pot[m] - ref["pot"][m]) / np.abs(ref["pot"][m])
    counts_equal = bool(np.array_equal(n_pc[m], ref["n_pc"][m]) and np.array_equal(n_pp[m], ref["n_pp"][m]))
    q999, amax, pmax = float(np.quantile(rel, 0.999)), float(rel.max()), float(prel.max())
    flips_ok = bool(all(len(cells) == f and all(s_ <= b for _, s_, b in cells) for _, f, cells in ref["flip_audit"]))
    return {"n_compared": int(m.sum()), "n_groups_compared": int(len(sel)), "n_groups": int(ng), "whole_population": bool(len(sel) == ng),
            "counts_equal": counts_equal, "acc_q50": float(np.median(rel)), "acc_q999": q999, "acc_max": amax, "pot_max": pmax,
            "flips": int(ref["flips"].sum()),
            # R16 audit: every group whose fp32 walk differs from the fp64 one, with the cells decided differently,
            # their fp64 slack |d theta - 2 h_c| and the bound 8 * 2^-23 * (max_k(|b_c,k| + |b_g,k|) + h_c + h_g) * max(theta, 1)
            "flip_groups": [{"group": g, "flips": f, "cells": [{"cell": x, "slack": s_, "bound": b} for x, s_, b in cells]}
                            for g, f, cells in ref["flip_audit"]],
            "flips_borderline": flips_ok,
            "tolerance": {"acc_q999": ACC_Q999, "acc_max": ACC_MAX, "pot_max": POT_MAX},
            "within_tolerance": bool(counts_equal and q999 <= ACC_Q999 and amax <= ACC_MAX and pmax <= POT_MAX and flips_ok),
            "what": "per-particle interaction counts (exact) and relative errors of acc / pot of the TIMED launch against the fp64 oracle "
                    "with fp32-shadow opening decisions; flips = opening tests the fp32 decision takes differently from fp64 (R16)"}


def timed_forces(tc, B, torch, stream, flush, theta, eps, d_acc, d_pot, reps):
    ms = []
    for _ in range(reps):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        B.tc_forces(tc.ctx, theta, eps, d_acc, d_pot)
        b.record(stream)
        torch.cuda.synchronize()
        ms.append(a.elapsed_time(b))
    return ms


def e2e_leg(tc, n_leaf, theta, eps, h_pos, h_mass, h_acc, h_pot, reps, torch):
    t_all, t_host, t_copy = [], [], []
    for i in range(2 + reps):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        tc.set_particles(h_pos, h_mass)
        tc.build(n_leaf)
        tc.forces(theta, eps, h_acc, h_pot)
        dt = time.perf_counter() - t0
        if i >= 2:
            t_all.append(dt)
            s2 = tc.stats()
            t_host.append(s2["t_host_ms"]); t_copy.append(s2["t_copy_ms"])
    return float(np.mean(t_all)), float(np.mean(t_host)), float(np.mean(t_copy))


def run_ours(args) -> None:
    import torch
    rank, world, local = dist_env()
    if world != args.gpus:
        if world == 1 and args.gpus > 1:
            raise SystemExit("bench.py --gpus N>1 must be launched with torch.distributed.run (one rank per GPU)")
    assert torch.cuda.is_available(), "bench.py needs a CUDA device: there is no CPU fallback for the product path"
    local = local % torch.cuda.device_count()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        # NCCL over NVLink / NVSwitch; TC_BENCH_BACKEND=gloo exists only to walk this code path on a one-GPU box
        backend = os.environ.get("TC_BENCH_BACKEND", "nccl")
        dist.init_process_group(backend, **({"device_id": dev} if backend == "nccl" else {}))
    from paper_1005_5384_b200 import binding as B
    from paper_1005_5384_b200 import build as tc_build
    from paper_1005_5384_b200 import inputs, parallel
    if rank == 0:
        tc_build.build()
    if world > 1:
        dist.barrier()

    pos, mass, theta, eps, n_leaf = inputs.make(WORKLOAD)       # every rank: the SAME particles (one evaluation)
    n = len(mass)
    K, W = args.steps, args.warmup

    stream = torch.cuda.Stream(device=dev)
    tc = B.TreeCode(n_group=N_GROUP)
    tc.set_stream(stream.cuda_stream)
    extra = {}
    with torch.cuda.stream(stream):
        d_pos, d_mass = torch.from_numpy(pos).to(dev), torch.from_numpy(mass).to(dev)
        d_acc = torch.empty((n, 3), dtype=torch.float32, device=dev)
        d_pot = torch.empty(n, dtype=torch.float32, device=dev)
        flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
        tc.set_particles(d_pos, d_mass)
        tc.build(n_leaf)
        # N > 1: the shard options, the shard size and the row buffers are fixed once per tree (parallel.ShardPlan)
        plan = parallel.ShardPlan(tc, dev) if world > 1 else None

        def step():
            if world == 1:
                B.tc_forces(tc.ctx, theta, eps, d_acc, d_pot)
            else:   # this rank's shard + ONE all-gather + scatter (paper_1005_5384_b200/parallel.py)
                plan.forces(theta, eps, d_acc, d_pot)

        for _ in range(W):
            flush.zero_()
            step()
        torch.cuda.synchronize()
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
        st = tc.stats()                                # N > 1: the totals of THIS rank's shard
        inter = st["n_pc_total"] + st["n_pp_total"]
        flops_rank = FLOPS_PC * st["n_pc_total"] + FLOPS_PP * st["n_pp_total"]
        kernel_ms_rank = st["t_gpu_ms"]
        tree_bytes = st["tree_bytes"]
        if plan is not None:
            plan.close()
        h_acc_res = h_pot_res = n_pc_res = n_pp_res = None
        if world == 1:
            h_acc_res, h_pot_res = d_acc.cpu().numpy(), d_pot.cpu().numpy()      # the timed launch's result, for `parity`
            n_pc_res, n_pp_res = tc.counts()

        # ---- e2e: host buffers through the public API, every step: set_particles + build + forces
        Ke = max(3, min(K, 10))
        h_pos = torch.from_numpy(pos).pin_memory().numpy()
        h_mass = torch.from_numpy(mass).pin_memory().numpy()
        h_acc = torch.empty((n, 3), dtype=torch.float32).pin_memory().numpy()
        h_pot = torch.empty(n, dtype=torch.float32).pin_memory().numpy()
        if world == 1:
            e2e_s, t_host, t_copy = e2e_leg(tc, n_leaf, theta, eps, h_pos, h_mass, h_acc, h_pot, Ke, torch)
            p_acc, p_pot = np.empty((n, 3), np.float32), np.empty(n, np.float32)                  # plain (pageable) numpy arrays
            e2e_pg_s, t_host_pg, _ = e2e_leg(tc, n_leaf, theta, eps, pos, mass, p_acc, p_pot, Ke, torch)
            tc.set_option("device_build", 1)
            e2e_dev_s, t_build_dev, _ = e2e_leg(tc, n_leaf, theta, eps, h_pos, h_mass, h_acc, h_pot, Ke, torch)
            e2e_dev_pg_s, _, _ = e2e_leg(tc, n_leaf, theta, eps, pos, mass, p_acc, p_pot, Ke, torch)
            tc.set_option("device_build", 0)
        else:
            # every rank: particles H2D + device tree build + its shard + all-gather + scatter + D2H of the full result
            tc.set_option("device_build", 1)
            t_all = []
            for i in range(2 + Ke):
                torch.cuda.synchronize(); dist.barrier()
                t0 = time.perf_counter()
                tc.set_particles(h_pos, h_mass)
                tc.build(n_leaf)
                with parallel.ShardPlan(tc, dev) as pl:           # a new tree: a new shard layout
                    pl.forces(theta, eps, d_acc, d_pot)
                torch.from_numpy(h_acc).copy_(d_acc, non_blocking=True); torch.from_numpy(h_pot).copy_(d_pot, non_blocking=True)
                torch.cuda.synchronize()
                if i >= 2:
                    t_all.append(time.perf_counter() - t0)
            e2e_s = float(np.mean(t_all))
            tc.set_option("device_build", 0)

        if world == 1:
            # ---- the paper's second metric: data rate of the tree walk alone (A1-A3), lists dropped
            tc.set_particles(d_pos, d_mass); tc.build(n_leaf)
            tc.set_option("walk_only", 1)
            walk_ms = float(np.median(timed_forces(tc, B, torch, stream, flush, theta, eps, d_acc, d_pot, 5)[1:]))
            sw = tc.stats()
            tc.set_option("walk_only", 0)
            # ---- the paper-literal group size N_group = N_leaf beside the tuned one
            tc.set_option("n_group", n_leaf); tc.set_option("device_build", 1)
            tc.build(n_leaf)
            lit_ms = timed_forces(tc, B, torch, stream, flush, theta, eps, d_acc, d_pot, 6)[1:]
            sl = tc.stats()
            lit_flops = FLOPS_PC * sl["n_pc_total"] + FLOPS_PP * sl["n_pp_total"]
            extra["paper_literal"] = {
                "n_group": n_leaf, "n_groups": sl["n_groups"], "ms": float(np.median(lit_ms)), "ms_min": float(min(lit_ms)),
                "interactions": sl["n_pc_total"] + sl["n_pp_total"], "n_pc": sl["n_pc_total"], "n_pp": sl["n_pp_total"],
                "opening_tests": sl["n_tests_total"],
                "interactions_per_s": (sl["n_pc_total"] + sl["n_pp_total"]) / (float(np.median(lit_ms)) * 1e-3),
                "tflops": lit_flops / (float(np.median(lit_ms)) * 1e-3) / 1e12,
                "what": "config 3 with N_group = N_leaf = 16 (groups = leaves, PAPER.md:145): fewer interactions, 5.8x the walks; "
                        "frac is against the same FP32 peak"}
            # ---- the paper's OWN setting N_leaf = N_group = 64, same particles, theta, eps
            tc.set_option("n_group", 64)
            tc.build(64)
            p64_ms = timed_forces(tc, B, torch, stream, flush, theta, eps, d_acc, d_pot, 6)[1:]
            s64 = tc.stats()
            p64_flops = FLOPS_PC * s64["n_pc_total"] + FLOPS_PP * s64["n_pp_total"]
            extra["paper_setting"] = {
                "n_leaf": 64, "n_group": 64, "n_groups": s64["n_groups"], "ms": float(np.median(p64_ms)), "ms_min": float(min(p64_ms)),
                "interactions": s64["n_pc_total"] + s64["n_pp_total"], "n_pc": s64["n_pc_total"], "n_pp": s64["n_pp_total"],
                "opening_tests": s64["n_tests_total"],
                "interactions_per_s": (s64["n_pc_total"] + s64["n_pp_total"]) / (float(np.median(p64_ms)) * 1e-3),
                "tflops": p64_flops / (float(np.median(p64_ms)) * 1e-3) / 1e12,
                "gflops_paper_convention": (PAPER_FLOPS_PC * s64["n_pc_total"] + PAPER_FLOPS_PP * s64["n_pp_total"]) / (float(np.median(p64_ms)) * 1e-3) / 1e9,
                "what": "config 3's particles at the paper's own N_leaf = N_group = 64 (PAPER.md:145); parity at this setting: "
                        "tests/test_gpu_configs.py"}
            tc.set_option("n_group", N_GROUP)
            # ---- config 5's size: N = 2^24, where the packed tree (0.6 GB) streams from HBM instead of sitting in L2
            p5, m5 = inputs.two_plummer(1 << 24)
            n5 = len(m5)
            d_pos5, d_mass5 = torch.from_numpy(p5).to(dev), torch.from_numpy(m5).to(dev)
            d_acc5 = torch.empty((n5, 3), dtype=torch.float32, device=dev); d_pot5 = torch.empty(n5, dtype=torch.float32, device=dev)
            tc.set_particles(d_pos5, d_mass5); tc.build(16)
            c5_ms = timed_forces(tc, B, torch, stream, flush, 0.5, 0.005, d_acc5, d_pot5, 4)[1:]
            s5 = tc.stats()
            c5_flops = FLOPS_PC * s5["n_pc_total"] + FLOPS_PP * s5["n_pp_total"]
            alg5 = int(s5["tree_bytes"] + 24 * n5)
            tr5 = traffic("config5")
            hbm_peak = measured_peaks().get("hbm_gbs")
            extra["config5"] = {
                "workload": "BASELINE.json configs[4] at step 0: two Plummer spheres, N = 2^24, eps = 0.005, theta = 0.5, N_leaf = 16, "
                            f"N_group = {N_GROUP}, device tree build",
                "n": n5, "n_groups": s5["n_groups"], "n_cells": s5["n_cells"], "ms": float(np.median(c5_ms)), "ms_min": float(min(c5_ms)),
                "t_build_ms": s5["t_host_ms"],
                "interactions": s5["n_pc_total"] + s5["n_pp_total"],
                "interactions_per_s": (s5["n_pc_total"] + s5["n_pp_total"]) / (float(np.median(c5_ms)) * 1e-3),
                "tflops": c5_flops / (float(np.median(c5_ms)) * 1e-3) / 1e12,
                "algorithmic_bytes_per_launch": alg5,
                "dram_traffic": tr5,
                "hbm_gb_per_s_algorithmic": alg5 / (float(np.median(c5_ms)) * 1e-3) / 1e9,
                "hbm_peak_gb_per_s": hbm_peak,
                "hbm_frac": (alg5 / (float(np.median(c5_ms)) * 1e-3) / 1e9 / hbm_peak) if hbm_peak else None,
                "what": "the tree (tree_bytes) is read and 24 B per particle of results are written once per launch: HBM is not the bound "
                        "at this size either; dram_traffic is the ncu capture named in profiles/traffic.json"}
            del d_pos5, d_mass5, d_acc5, d_pot5
            tc.set_option("device_build", 0)
            measured_peak = B.tc_fp32_peak(tc.ctx)       # FFMA-only microbenchmark on this device, after the timed region
        else:
            # ---- replicas (the weak-scaling mode of round 1, kept under its own key): every rank one whole evaluation
            tc.set_particles(d_pos, d_mass); tc.build(n_leaf)
            rep_ms = timed_forces(tc, B, torch, stream, flush, theta, eps, d_acc, d_pot, 4)[1:]
            srep = tc.stats()
            extra["_replica_ms"] = float(np.median(rep_ms)); extra["_replica_inter"] = srep["n_pc_total"] + srep["n_pp_total"]
            # ---- config 5 sharded over the ranks (the size at which T_gpu / N dominates the fixed costs)
            p5, m5 = inputs.two_plummer(1 << 24)
            n5 = len(m5)
            d_pos5, d_mass5 = torch.from_numpy(p5).to(dev), torch.from_numpy(m5).to(dev)
            d_acc5 = torch.empty((n5, 3), dtype=torch.float32, device=dev); d_pot5 = torch.empty(n5, dtype=torch.float32, device=dev)
            tc.set_option("device_build", 1)
            tc.set_particles(d_pos5, d_mass5); tc.build(16)
            ms5 = []
            with parallel.ShardPlan(tc, dev) as plan5:
                for i in range(4):
                    dist.barrier()
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record(stream)
                    plan5.forces(0.5, 0.005, d_acc5, d_pot5)
                    b.record(stream)
                    torch.cuda.synchronize()
                    ms5.append(a.elapsed_time(b))
                s5 = tc.stats()
            extra["_c5_ms"] = float(np.median(ms5[1:])); extra["_c5_inter"] = s5["n_pc_total"] + s5["n_pp_total"]
            tc.set_option("device_build", 0)
            measured_peak = None
    tc.close()

    t_dev_ms = max_over_ranks(t_dev_ms, world, dev)
    e2e_s = max_over_ranks(e2e_s, world, dev)
    inter_all = sum_over_ranks(float(inter), world, dev)
    if world > 1:
        rep_ms_max = max_over_ranks(extra.pop("_replica_ms"), world, dev)
        rep_inter = sum_over_ranks(float(extra.pop("_replica_inter")), world, dev)
        c5_ms_max = max_over_ranks(extra.pop("_c5_ms"), world, dev)
        c5_inter = sum_over_ranks(float(extra.pop("_c5_inter")), world, dev)
        kernel_ms_max = max_over_ranks(kernel_ms_rank, world, dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    ms = t_dev_ms / K
    value = inter_all / (ms * 1e-3)
    kernel_ms = float(np.mean(per_step)) if world == 1 else kernel_ms_rank
    ach = flops_rank / (kernel_ms * 1e-3) / 1e12        # the force kernel of ONE GPU against ONE GPU's peak
    sm_max = clocks.get("sm_max_mhz") or 1965.0
    peak = fp32_peak_tflops(sm_max)
    tr3 = traffic("config3")
    out = {
        "metric": "interactions/s of one force evaluation (tree walk + list evaluation), N=2^20 Plummer, theta=0.5; "
                  "ms per force evaluation is ms_per_step",
        "value": value, "unit": "interactions/s", "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms, "higher_is_better": True, "scaling": "weak" if world == 1 else "strong", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[2]: Plummer N={n} seed 3, eps={eps}, theta={theta}, "
                               f"N_leaf={n_leaf}, N_group={N_GROUP}, monopole+quadrupole",
                   "n": n, "theta": theta, "eps": eps, "n_leaf": n_leaf, "n_group": N_GROUP,
                   "l2": f"flushed between timed steps ({L2_FLUSH_BYTES >> 20} MiB memset outside the events)",
                   "sharding": "none (one GPU)" if world == 1 else
                               f"ONE evaluation over {world} GPUs: every rank evaluates every {world}-th group of the cost-ordered "
                               "schedule, one all-gather of 16 B per particle (NCCL), scatter to the caller's order"},
        "particles_per_s": n / (ms * 1e-3),
        "interactions_per_step": inter_all,
        "n_groups": st["n_groups"], "n_cells": st["n_cells"],
        "ms_per_step_min": float(min(per_step)), "ms_per_step_median": float(np.median(per_step)),
        "wall_ms_per_step_incl_flush": t_wall * 1e3 / K,
        "gpu_launches": K if world == 1 else 2 * K,     # rank 0's own kernels in the timed region: forces (+ scatter when sharded)
        "clocks": clocks,
        "roofline": {"bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                     "traffic": tr3["dram_bytes"] if tr3 else None, "traffic_stale": tr3["traffic_stale"] if tr3 else None,
                     "kernel": "tc::forces_kernel",
                     "peak_how": f"nominal: {N_SM} SMs x {LANES} FP32 lanes x 2 x {sm_max:.0f} MHz (DESIGN.md section 6; "
                                 "MEASURED_PEAKS.json holds HBM and bf16 figures only, no FP32 entry)",
                     "peak_measured": measured_peak, "frac_of_measured": (ach / measured_peak) if measured_peak else None,
                     "peak_measured_how": "tc_fp32_peak (include/tc_bench.h): FFMA-only microbenchmark on this device in this run",
                     "frac_survey_flops": ((SURVEY_FLOPS_PC * st["n_pc_total"] + SURVEY_FLOPS_PP * st["n_pp_total"]) / (kernel_ms * 1e-3) / 1e12 / peak),
                     "frac_survey_flops_how": f"the same launch counted with SURVEY.md 8(d)'s {SURVEY_FLOPS_PC} / {SURVEY_FLOPS_PP} flops per interaction",
                     "flops_per_launch": flops_rank, "flops_convention": f"{FLOPS_PC} per particle-cell, {FLOPS_PP} per particle-particle interaction "
                                                                         "(FFMA = 2, FADD/FMUL = 1, MUFU = 1); hardware counters in profiles/",
                     "algorithmic_bytes_per_launch": int(tree_bytes + 24 * n),
                     "traffic_how": (f"dram__bytes_read.sum + dram__bytes_write.sum of the ncu --set full capture {tr3['capture']} "
                                     f"(profiles/traffic.json); HBM is not the bound") if tr3 else None},
    }
    if world == 1:
        out.update({
            "n_pc": st["n_pc_total"], "n_pp": st["n_pp_total"], "opening_tests": st["n_tests_total"], "opened_cells": st["n_opened_total"],
            "gflops_paper_convention": (PAPER_FLOPS_PC * st["n_pc_total"] + PAPER_FLOPS_PP * st["n_pp_total"]) / (kernel_ms * 1e-3) / 1e9,
            "walk": {"ms": walk_ms,
                     "algorithmic_bytes": 16 * sw["n_tests_total"] + 16 * sw["n_opened_total"],
                     "gb_per_s": (16.0 * sw["n_tests_total"] + 16.0 * sw["n_opened_total"]) / (walk_ms * 1e-3) / 1e9,
                     "requested_bytes": 64 * sw["n_tests_total"],
                     "gb_per_s_requested": 64.0 * sw["n_tests_total"] / (walk_ms * 1e-3) / 1e9,
                     "what": "option walk_only (include/tc_bench.h): walk + list building without evaluation.  gb_per_s counts SURVEY 8(d)'s "
                             "algorithmic bytes (16 B per opening test + 16 B per opened cell); gb_per_s_requested counts what the kernel asks "
                             "L2 for (4 float4 per test: 84 % of the tested cells end on a cell list and need their 48 B of multipole); "
                             "lts__t_bytes of this launch is in profiles/; the paper reports > 50 GB/s for its count pass on G80 (PAPER.md:177)"},
            "e2e": {"value": inter_all / e2e_s, "unit": "interactions/s", "h2d_bytes_per_step": int(tree_bytes),
                    "d2h_bytes_per_step": int(16 * n), "ms_per_step": e2e_s * 1e3,
                    "t_host_build_ms": t_host, "t_copy_ms": t_copy,
                    "what": "tc_set_particles(host)+tc_build(host octree, one bulk H2D)+tc_forces(host acc,pot); wall clock; "
                            "PINNED (page-locked) host buffers",
                    "pageable": {"value": inter_all / e2e_pg_s, "ms_per_step": e2e_pg_s * 1e3, "t_host_build_ms": t_host_pg,
                                 "what": "the same calls with plain (pageable) numpy arrays for pos, mass, acc, pot"}},
            "e2e_device_build": {"value": inter_all / e2e_dev_s, "unit": "interactions/s", "h2d_bytes_per_step": int(16 * n),
                                 "d2h_bytes_per_step": int(16 * n), "ms_per_step": e2e_dev_s * 1e3, "t_build_ms": t_build_dev,
                                 "what": "same calls with tc_set_option('device_build', 1): particles H2D, tree built on the GPU; pinned host buffers",
                                 "pageable": {"value": inter_all / e2e_dev_pg_s, "ms_per_step": e2e_dev_pg_s * 1e3}},
        })
        extra["paper_literal"]["frac"] = extra["paper_literal"]["tflops"] / peak
        extra["paper_setting"]["frac"] = extra["paper_setting"]["tflops"] / peak
        extra["config5"]["frac"] = extra["config5"]["tflops"] / peak
        out.update(extra)
        cb, ref, sel, ng = cpu_baseline(pos, mass, theta, eps, n_leaf)
        out["cpu_baseline"] = cb
        out["parity"] = parity_object(ref, sel, ng, h_acc_res, h_pot_res, n_pc_res, n_pp_res)
    else:
        out["e2e"] = {"value": inter_all / e2e_s, "unit": "interactions/s", "h2d_bytes_per_step": int(16 * n) * world,
                      "d2h_bytes_per_step": int(16 * n) * world, "ms_per_step": e2e_s * 1e3,
                      "what": "per rank: tc_set_particles(pinned host) + tc_build(device build) + its shard + all-gather + scatter + "
                              "D2H of the full acc, pot; wall clock, max over ranks"}
        out["shard"] = {"kernel_ms_max_over_ranks": kernel_ms_max, "collective": "one NCCL all-gather of [n_slots,4] fp32 rows per rank",
                        "bytes_gathered_per_rank": int(16 * n), "interactions_rank0": inter}
        out["replicas"] = {"value": rep_inter / (rep_ms_max * 1e-3), "unit": "interactions/s", "ms_per_step": rep_ms_max, "scaling": "weak",
                           "what": "every rank one WHOLE evaluation of config 3, no collective (the mode round 1 reported)"}
        out["config5"] = {"n": 1 << 24, "ms": c5_ms_max, "interactions": c5_inter, "interactions_per_s": c5_inter / (c5_ms_max * 1e-3),
                          "what": "two Plummer spheres, N = 2^24, ONE evaluation sharded over the ranks (kernel + all-gather + scatter)"}
        out["cpu_baseline"] = None
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
        "ms_per_step": t_all * 1e3 / K, "higher_is_better": True, "scaling": "weak" if args.gpus == 1 else "strong", "vs_baseline": None,
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
