"""ONE force evaluation over several GPUs: one process per GPU, plumbing by
``torch.distributed``.

Groups are independent given the read-only tree (one walk per group, no communication between
groups), so the path shards with NO collective inside the walk or the evaluation: every rank holds the same
particles, builds the same tree (the device build takes ~1 ms at N = 2^20 — cheaper than broadcasting the
37 MB packed tree), evaluates the groups at schedule positions rank, rank + world, ... (library options
"shard_count" / "shard_rank": neighbours in the cost-ordered schedule cost the same, so the shards are
balanced) and leaves ZEROS for every particle outside its shard.  The only exchange is the one that hands
every rank the full result: one all-reduce (SUM) of acc and pot — over NCCL that is an NVSwitch in-switch
reduction of 16 bytes per particle.  Adding zeros is exact, so the combined result is bit-for-bit the
single-GPU result (tests/test_gpu_shard.py runs the shards one after the other on one GPU).

Marshalling only: all arithmetic is in the library's kernels or in the collective.
"""
from __future__ import annotations

import torch
import torch.distributed as dist

from . import binding as B


def shard_of(rank: int, world: int, n_groups: int) -> range:
    """Schedule positions rank `rank` evaluates (what the kernel does with shard_rank / shard_count)."""
    return range(rank, n_groups, world)


def combine(acc: "torch.Tensor", pot: "torch.Tensor | None" = None, counts=(), group=None) -> None:
    """Sum the zero-padded shard results of all ranks in place (every rank ends with the full arrays)."""
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return
    work = [dist.all_reduce(acc, op=dist.ReduceOp.SUM, group=group, async_op=True)]
    if pot is not None:
        work.append(dist.all_reduce(pot, op=dist.ReduceOp.SUM, group=group, async_op=True))
    for c in counts:
        work.append(dist.all_reduce(c, op=dist.ReduceOp.SUM, group=group, async_op=True))
    for w in work:
        w.wait()


def forces_sharded(tc: "B.TreeCode", theta: float, eps: float, acc: "torch.Tensor", pot: "torch.Tensor | None" = None,
                   group=None) -> None:
    """tc_forces of this rank's shard into the DEVICE tensors acc [n,3] / pot [n], then ``combine``.

    Every rank must have called set_particles / build with the same particles and options.
    """
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    tc.set_option("shard_count", world)
    tc.set_option("shard_rank", rank)
    try:
        B.tc_forces(tc.ctx, theta, eps, acc, pot)
        tc.sync()
    finally:
        tc.set_option("shard_count", 1)
        tc.set_option("shard_rank", 0)
    combine(acc, pot, group=group)


def main(argv=None) -> None:
    """Strong-scaling timing of ONE config-3 force evaluation over the ranks of a torchrun launch:

        python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \\
            -m paper_1005_5384_b200.parallel --steps 10

    Every rank holds the same particles and builds the same tree on its GPU; the timed region is the sharded
    ``tc_forces`` plus the all-reduce, CUDA events on the launching stream, max over ranks.  Rank 0 prints one
    JSON line.  (``bench.py`` keeps the weak-scaling contract: independent evaluations per rank, no collective.)
    """
    import argparse
    import json
    import os

    import numpy as np

    from . import build as tc_build
    from . import inputs

    ap = argparse.ArgumentParser()
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="plummer_1m")
    args = ap.parse_args(argv)
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    if rank == 0:
        tc_build.build()
    if world > 1:
        dist.barrier()
    pos, mass, theta, eps, n_leaf = inputs.make(args.workload)
    n = len(mass)
    stream = torch.cuda.Stream(device=dev)
    with B.TreeCode() as tc, torch.cuda.stream(stream):
        tc.set_stream(stream.cuda_stream)
        tc.set_option("device_build", 1)
        d_pos, d_mass = torch.from_numpy(pos).to(dev), torch.from_numpy(mass).to(dev)
        acc = torch.empty((n, 3), dtype=torch.float32, device=dev)
        pot = torch.empty(n, dtype=torch.float32, device=dev)
        tc.set_particles(d_pos, d_mass)
        tc.build(n_leaf)
        ms = []
        for i in range(args.warmup + args.steps):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            if world > 1:
                dist.barrier()
            a.record(stream)
            forces_sharded(tc, theta, eps, acc, pot)
            b.record(stream)
            torch.cuda.synchronize()
            t = torch.tensor([a.elapsed_time(b)], dtype=torch.float64, device=dev)
            if world > 1:
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
            if i >= args.warmup:
                ms.append(float(t))
        checksum = float(acc.double().abs().sum())
    if rank == 0:
        print(json.dumps({"what": "one force evaluation sharded over the ranks (groups strided over the cost-ordered schedule, "
                                  "one all-reduce of acc and pot)", "workload": args.workload, "n": n, "n_gpus": world,
                          "scaling": "strong", "ms_per_evaluation": float(np.mean(ms)), "ms_min": float(np.min(ms)),
                          "checksum_abs_acc": checksum}))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
