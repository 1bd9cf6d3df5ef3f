"""ONE force evaluation over several GPUs: one process per GPU, plumbing by
``torch.distributed``.

Groups are independent given the read-only tree (one walk per group, no communication between
groups), so the path shards with NO collective inside the walk or the evaluation: every rank holds the same
particles and builds the same tree, rank r evaluates the groups at schedule positions r, r + world, ... (library
options "shard_count" / "shard_rank"; neighbours in the cost-ordered schedule cost the same, so strided shards are
balanced) and writes ONLY its own particles, as compact rows (ax, ay, az, phi).  The one exchange is the one that
hands every rank the rows of the others: ONE all-gather of 16 bytes per particle (NCCL over NVLink / NVSwitch),
then the library scatters the gathered rows to the caller's particle order (``tc_shard_scatter``).  Every particle
is computed by exactly one rank with the arithmetic of the single-GPU launch, so the result is bit for bit the
single-GPU result (tests/test_gpu_shard.py runs the shards one after the other on one GPU;
tests/test_multirank_cpu.py runs this module's protocol over gloo with two processes).

Marshalling only: all arithmetic is in the library's kernels.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard_of(rank: int, world: int, n_groups: int) -> range:
    """Schedule positions rank `rank` evaluates (what the kernel does with shard_rank / shard_count)."""
    return range(rank, n_groups, world)


def all_gather_rows(rows: "torch.Tensor", group=None) -> "torch.Tensor":
    """[n_slots, c] on every rank -> [world, n_slots, c], rank-major (the layout tc_shard_scatter reads)."""
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    out = torch.empty((world * rows.shape[0],) + tuple(rows.shape[1:]), dtype=rows.dtype, device=rows.device)
    if world == 1:
        out.copy_(rows)
    else:
        dist.all_gather_into_tensor(out, rows, group=group)      # concatenation along dim 0 = rank-major
    return out.view((world,) + tuple(rows.shape))


def forces_sharded(tc, theta: float, eps: float, acc: "torch.Tensor", pot: "torch.Tensor | None" = None, group=None,
                   n_pc: "torch.Tensor | None" = None, n_pp: "torch.Tensor | None" = None, scratch: dict | None = None) -> None:
    """This rank's shard, the all-gather, the scatter: acc [n,3] / pot [n] (and the counts, if asked for) end up
    complete and in the caller's order on EVERY rank.  Device tensors; stream-ordered on torch's current stream:
    the context is pointed at it here (``use_torch_stream``; the default stream, raw handle 0, goes in as
    cudaStreamLegacy), because the all-gather between the shard kernel and the scatter waits on that stream only.

    Every rank must have called set_particles / build with the same particles and options.  `tc` is a
    ``binding.TreeCode`` (anything with set_option / shard_size / forces_shard / shard_scatter works: the CPU test
    drives this function with a stand-in).  `scratch` keeps the row buffers between calls.
    """
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    if acc.is_cuda:
        tc.use_torch_stream(acc.device)
    tc.set_option("shard_count", world)
    tc.set_option("shard_rank", rank)
    try:
        n_slots = tc.shard_size()
        sc = scratch if scratch is not None else {}
        rows = sc.get("rows")
        if rows is None or rows.shape[0] != n_slots or rows.device != acc.device:
            rows = sc["rows"] = torch.empty((n_slots, 4), dtype=torch.float32, device=acc.device)
            sc["cnt"] = None
        cnt = None
        if n_pc is not None or n_pp is not None:
            cnt = sc.get("cnt")
            if cnt is None:
                cnt = sc["cnt"] = torch.empty((n_slots, 2), dtype=torch.int32, device=acc.device)
        tc.forces_shard(theta, eps, rows, cnt)
        gathered = all_gather_rows(rows, group)
        gathered_cnt = all_gather_rows(cnt, group) if cnt is not None else None
        tc.shard_scatter(gathered, gathered_cnt, acc, pot, n_pc, n_pp)
    finally:
        tc.set_option("shard_count", 1)
        tc.set_option("shard_rank", 0)
