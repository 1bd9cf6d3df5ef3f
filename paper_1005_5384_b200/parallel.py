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


class ShardPlan:
    """Everything about a sharded evaluation that depends on the TREE and the process group, not on the step: made once
    after ``tc.build`` and used for every force evaluation on that tree (a time step loop with a rebuilt tree makes
    one per build — the shard layout is a function of the tree).

    Creation points the context at torch's current stream, sets the library options "shard_count" / "shard_rank",
    asks for the shard size ONCE and allocates the row buffers; ``forces`` is then just shard kernel -> all-gather ->
    scatter, with no option traffic per step.  ``close`` (or the ``with`` statement) puts the options back so that the
    context can serve plain ``tc_forces`` calls again.  `tc` is a ``binding.TreeCode`` (or the CPU test's stand-in).
    """

    def __init__(self, tc, device, group=None, counts: bool = False, rows=None, cnt=None):
        self.tc, self.group, self.device = tc, group, torch.device(device)
        self.world = dist.get_world_size(group) if dist.is_initialized() else 1
        self.rank = dist.get_rank(group) if dist.is_initialized() else 0
        self._stream = None
        self._order_with_torch()
        tc.set_option("shard_count", self.world)
        tc.set_option("shard_rank", self.rank)
        self.open = True
        try:
            self.n_slots = tc.shard_size()
        except Exception:
            self.close()
            raise
        # (`rows` / `cnt`: buffers of an earlier plan, taken over when they still fit)
        fits = lambda t, c: t is not None and tuple(t.shape) == (self.n_slots, c) and t.device == self.device
        self.rows = rows if fits(rows, 4) else torch.empty((self.n_slots, 4), dtype=torch.float32, device=self.device)
        self.cnt = cnt if fits(cnt, 2) else (torch.empty((self.n_slots, 2), dtype=torch.int32, device=self.device) if counts else None)

    def _order_with_torch(self):
        # the all-gather between the shard kernel and the scatter waits on torch's current stream only: the library's work
        # must be on that stream (the default stream goes in as cudaStreamLegacy).  tc_set_stream synchronises the stream it
        # leaves, so it is only called when the stream has actually changed.
        if self.device.type != "cuda" or not hasattr(self.tc, "use_torch_stream"):
            return
        h = int(torch.cuda.current_stream(self.device).cuda_stream)
        if h != self._stream:
            self.tc.use_torch_stream(self.device)
            self._stream = h

    def forces(self, theta: float, eps: float, acc, pot=None, n_pc=None, n_pp=None) -> None:
        """acc [n,3] / pot [n] (and the counts, if asked for) complete and in the caller's order on EVERY rank."""
        assert self.open, "ShardPlan.forces after close()"
        self._order_with_torch()
        cnt = None
        if n_pc is not None or n_pp is not None:
            if self.cnt is None:
                self.cnt = torch.empty((self.n_slots, 2), dtype=torch.int32, device=self.device)
            cnt = self.cnt
        self.tc.forces_shard(theta, eps, self.rows, cnt)
        gathered = all_gather_rows(self.rows, self.group)
        gathered_cnt = all_gather_rows(cnt, self.group) if cnt is not None else None
        self.tc.shard_scatter(gathered, gathered_cnt, acc, pot, n_pc, n_pp)

    def close(self):
        if getattr(self, "open", False):
            self.open = False
            self.tc.set_option("shard_count", 1)
            self.tc.set_option("shard_rank", 0)

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()


def forces_sharded(tc, theta: float, eps: float, acc: "torch.Tensor", pot: "torch.Tensor | None" = None, group=None,
                   n_pc: "torch.Tensor | None" = None, n_pp: "torch.Tensor | None" = None, scratch: dict | None = None) -> None:
    """One-shot form of ``ShardPlan``: this rank's shard, the all-gather, the scatter: acc [n,3] / pot [n] (and the
    counts, if asked for) end up complete and in the caller's order on EVERY rank.  Device tensors; stream-ordered on
    torch's current stream (the context is pointed at it here).  A loop over many evaluations of ONE tree should make a
    ``ShardPlan`` once instead: this function sets and resets the shard options and queries the shard size every call.

    Every rank must have called set_particles / build with the same particles and options.  `tc` is a
    ``binding.TreeCode`` (anything with set_option / shard_size / forces_shard / shard_scatter works: the CPU test
    drives this function with a stand-in).  `scratch` keeps the row buffers between calls.
    """
    sc = scratch if scratch is not None else {}
    plan = ShardPlan(tc, acc.device, group, rows=sc.get("rows"), cnt=sc.get("cnt"))
    try:
        plan.forces(theta, eps, acc, pot, n_pc, n_pp)
    finally:
        plan.close()
    sc["rows"], sc["cnt"] = plan.rows, plan.cnt
