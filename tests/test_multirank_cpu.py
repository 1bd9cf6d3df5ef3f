"""N > 1 host logic on CPU: world_size-2 `gloo` processes (no GPU).

The walk and the evaluation have no collective (groups are independent); what N > 1 adds is
(a) the reductions `bench.py` reports with (max-over-ranks time, sum-over-ranks work), (b) the sharded evaluation's
one exchange — the all-gather of the compact rows in `parallel.forces_sharded` —, (c) the reference arm running on
rank 0 only.  All three are exercised here.
"""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    import bench
    from paper_1005_5384_b200 import inputs
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    # (a) rank r evaluates its own sphere: seeds differ, shapes agree
    fn, kw, *_ = inputs.WORKLOADS["plummer_1k"]
    pos, mass = fn(**dict(kw, seed=kw["seed"] + rank))
    gathered = [torch.zeros(3, dtype=torch.float64) for _ in range(world)]
    dist.all_gather(gathered, torch.from_numpy(pos[:1].astype(np.float64)).reshape(3))
    # (b) the two reductions of bench.py
    t_max = bench.max_over_ranks(10.0 + rank, world)
    w_sum = bench.sum_over_ranks(100.0 * (rank + 1), world)
    dist.barrier()
    with open(os.path.join(out_dir, f"r{rank}.json"), "w") as f:
        json.dump({"t_max": t_max, "w_sum": w_sum, "first": [g.tolist() for g in gathered], "n": len(mass)}, f)
    dist.destroy_process_group()


def test_two_ranks_gloo(tmp_path):
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    r = [json.load(open(tmp_path / f"r{k}.json")) for k in range(world)]
    for k in range(world):
        assert r[k]["t_max"] == 11.0 and r[k]["w_sum"] == 300.0 and r[k]["n"] == 1024
    assert r[0]["first"] == r[1]["first"]                 # the gather agrees on both ranks
    assert r[0]["first"][0] != r[0]["first"][1]           # different spheres per rank


class _OracleRank:
    """Stand-in for binding.TreeCode on a machine without a GPU: the same four calls `parallel.forces_sharded` makes
    (set_option / shard_size / forces_shard / shard_scatter), answered from the ORACLE's results.  Layout as the
    library's (include/tc.h): rank r owns the groups r, r + k, ... (here of the Morton order; the library strides its
    cost-ordered schedule), its rows are its groups in that order, particles in tree order inside a group."""

    def __init__(self, o, theta, eps):
        self.o, self.theta, self.eps = o, theta, eps
        self.opt = {"shard_count": 1, "shard_rank": 0}
        c = o.cells()
        g = o.groups()
        self.begin, self.count, self.perm = c["begin"][g], c["count"][g], o.perm()

    def set_option(self, k, v):
        self.opt[k] = int(v)

    def _rows_of(self, r):
        k = self.opt["shard_count"]
        gs = np.arange(r, self.o.n_groups, k)
        return gs, np.concatenate([[0], np.cumsum(self.count[gs])]).astype(np.int64)

    def shard_size(self):
        return int(max(self._rows_of(r)[1][-1] for r in range(self.opt["shard_count"])))

    def forces_shard(self, theta, eps, rows, cnt=None):
        gs, off = self._rows_of(self.opt["shard_rank"])
        res = self.o.forces(theta, eps, groups=gs)
        rows.fill_(float("nan"))
        for j, g in enumerate(gs):
            idx = self.perm[self.begin[g]: self.begin[g] + self.count[g]]
            rows[off[j]: off[j + 1], :3] = torch.from_numpy(res["acc"][idx]).to(rows.dtype)
            rows[off[j]: off[j + 1], 3] = torch.from_numpy(res["pot"][idx]).to(rows.dtype)
            if cnt is not None:
                cnt[off[j]: off[j + 1], 0] = torch.from_numpy(res["n_pc"][idx]).to(cnt.dtype)
                cnt[off[j]: off[j + 1], 1] = torch.from_numpy(res["n_pp"][idx]).to(cnt.dtype)

    def shard_scatter(self, gathered, gathered_cnt, acc, pot=None, n_pc=None, n_pp=None):
        for r in range(self.opt["shard_count"]):
            gs, off = self._rows_of(r)
            for j, g in enumerate(gs):
                idx = torch.from_numpy(self.perm[self.begin[g]: self.begin[g] + self.count[g]])
                acc[idx] = gathered[r, off[j]: off[j + 1], :3]
                if pot is not None:
                    pot[idx] = gathered[r, off[j]: off[j + 1], 3]
                if gathered_cnt is not None and n_pc is not None:
                    n_pc[idx] = gathered_cnt[r, off[j]: off[j + 1], 0]
                    n_pp[idx] = gathered_cnt[r, off[j]: off[j + 1], 1]


def _shard_worker(rank, world, port, out_dir):
    """`parallel.forces_sharded` end to end over gloo: every rank computes only its shard (here with the oracle —
    no GPU in this test), contributes its compact rows to ONE all-gather and must end with the full result."""
    sys.path.insert(0, ROOT)
    import oracle
    from paper_1005_5384_b200 import inputs, parallel
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    pos, mass, theta, eps, n_leaf = inputs.make("plummer_1k")
    n = len(mass)
    o = oracle.Oracle(pos, mass, n_leaf, 32)
    tc = _OracleRank(o, theta, eps)
    acc = torch.full((n, 3), float("nan"), dtype=torch.float64)
    pot = torch.full((n,), float("nan"), dtype=torch.float64)
    npc = torch.full((n,), -1, dtype=torch.int64); npp = torch.full((n,), -1, dtype=torch.int64)
    calls = []
    real_gather = dist.all_gather_into_tensor
    def counting_gather(out, inp, group=None):
        calls.append((tuple(out.shape), tuple(inp.shape)))
        return real_gather(out, inp, group=group)
    dist.all_gather_into_tensor = counting_gather
    # (rows in fp64 here so that the comparison with the oracle is exact; the library's rows are fp32)
    sc = {"rows": torch.empty((tc_rows := _rows(tc, world), 4), dtype=torch.float64), "cnt": torch.empty((tc_rows, 2), dtype=torch.int64)}
    parallel.forces_sharded(tc, theta, eps, acc, pot, n_pc=npc, n_pp=npp, scratch=sc)
    dist.all_gather_into_tensor = real_gather
    full = o.forces(theta, eps)
    ok = bool(np.array_equal(acc.numpy(), full["acc"]) and np.array_equal(pot.numpy(), full["pot"])
              and np.array_equal(npc.numpy(), full["n_pc"]) and np.array_equal(npp.numpy(), full["n_pp"]))
    mine = len(list(parallel.shard_of(rank, world, o.n_groups)))
    with open(os.path.join(out_dir, f"s{rank}.json"), "w") as f:
        json.dump({"ok": ok, "mine": mine, "groups": o.n_groups, "calls": calls, "n": n, "rows": tc_rows,
                   "options_reset": tc.opt == {"shard_count": 1, "shard_rank": 0}}, f)
    dist.destroy_process_group()


def _rows(tc, world):
    tc.set_option("shard_count", world)
    r = tc.shard_size()
    tc.set_option("shard_count", 1)
    return r


def test_sharded_force_evaluation_combines_to_the_whole(tmp_path):
    world, port = 2, _free_port()
    mp.spawn(_shard_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    r = [json.load(open(tmp_path / f"s{k}.json")) for k in range(world)]
    assert all(x["ok"] and x["options_reset"] for x in r)
    assert r[0]["mine"] + r[1]["mine"] == r[0]["groups"] and abs(r[0]["mine"] - r[1]["mine"]) <= 1
    # the exchange: ONE all-gather of the rows (+ one of the counts, asked for here), about n / world rows per rank
    for x in r:
        assert len(x["calls"]) == 2
        assert x["calls"][0] == [[world * x["rows"], 4], [x["rows"], 4]] and x["calls"][1] == [[world * x["rows"], 2], [x["rows"], 2]]
        assert x["n"] / world <= x["rows"] < 0.75 * x["n"]


def test_reference_arm_runs_on_rank0_only():
    """Under torchrun the oracle arm prints on rank 0; other ranks exit 0 without work."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert p.returncode == 0 and p.stdout.strip() == ""
