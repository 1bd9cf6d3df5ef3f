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
