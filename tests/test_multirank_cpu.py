"""N > 1 host logic on CPU: world_size-2 `gloo` processes (no GPU).

The hot path has no data-path collective (groups / force evaluations are independent),
so what N > 1 adds is (a) per-rank workloads, (b) the max-over-ranks time and sum-over-ranks work that
`bench.py` reports, (c) the reference arm running on rank 0 only.  All three are exercised here.
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


def _shard_worker(rank, world, port, out_dir):
    """Rank r holds the results of its shard (here: the ORACLE restricted to the groups r, r + world, ... —
    no GPU in this test), zeros elsewhere; parallel.combine must hand every rank the full result."""
    sys.path.insert(0, ROOT)
    import oracle
    from paper_1005_5384_b200 import inputs, parallel
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    pos, mass, theta, eps, n_leaf = inputs.make("plummer_1k")
    o = oracle.Oracle(pos, mass, n_leaf, 32)
    mine = np.array(list(parallel.shard_of(rank, world, o.n_groups)), dtype=np.int64)
    r = o.forces(theta, eps, groups=mine)
    acc = torch.from_numpy(np.nan_to_num(r["acc"], nan=0.0))
    pot = torch.from_numpy(np.nan_to_num(r["pot"], nan=0.0))
    npc = torch.from_numpy(np.maximum(r["n_pc"], 0))
    parallel.combine(acc, pot, counts=(npc,))
    full = o.forces(theta, eps)
    ok = bool(np.array_equal(acc.numpy(), full["acc"]) and np.array_equal(pot.numpy(), full["pot"])
              and np.array_equal(npc.numpy(), full["n_pc"]))
    with open(os.path.join(out_dir, f"s{rank}.json"), "w") as f:
        json.dump({"ok": ok, "mine": len(mine), "groups": o.n_groups}, f)
    dist.destroy_process_group()


def test_sharded_force_evaluation_combines_to_the_whole(tmp_path):
    world, port = 2, _free_port()
    mp.spawn(_shard_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    r = [json.load(open(tmp_path / f"s{k}.json")) for k in range(world)]
    assert all(x["ok"] for x in r)
    assert r[0]["mine"] + r[1]["mine"] == r[0]["groups"] and abs(r[0]["mine"] - r[1]["mine"]) <= 1


def test_reference_arm_runs_on_rank0_only():
    """Under torchrun the oracle arm prints on rank 0; other ranks exit 0 without work."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert p.returncode == 0 and p.stdout.strip() == ""
