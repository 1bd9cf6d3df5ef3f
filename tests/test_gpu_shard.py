"""Multi-GPU sharding of ONE force evaluation (options "shard_count" / "shard_rank")
on one GPU — `-m gpu`: the k shards are run one after the other; every particle is evaluated by exactly one of
them, entries outside a shard are zero, so the SUM of the shards is bit-for-bit the unsharded result."""
import numpy as np
import pytest

from oracle import Oracle
from paper_1005_5384_b200 import binding as B
from paper_1005_5384_b200 import build as tc_build
from paper_1005_5384_b200 import inputs
from test_gpu_parity import check

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    tc_build.build()


@pytest.mark.parametrize("k", [2, 3, 8])
@pytest.mark.parametrize("device_ptrs", [False, True])
def test_shards_partition_the_particles_and_sum_to_the_whole(k, device_ptrs):
    import torch
    pos, mass, theta, eps, n_leaf = inputs.make("plummer_64k")
    n = len(mass)
    with B.TreeCode(n_group=64) as tc:
        tc.set_particles(pos, mass)
        tc.build(n_leaf)
        acc0, pot0 = tc.forces(theta, eps)
        c0, d0 = tc.counts()
        s0 = tc.stats()
        acc, pot = np.zeros_like(acc0), np.zeros_like(pot0)
        npc, npp = np.zeros_like(c0), np.zeros_like(d0)
        owner = np.zeros(n, np.int32)
        tot = np.zeros(3, np.int64)
        tc.set_option("shard_count", k)
        for r in range(k):
            tc.set_option("shard_rank", r)
            if device_ptrs:
                da = torch.full((n, 3), 7.0, dtype=torch.float32, device="cuda")      # stale contents must be zeroed
                dp = torch.full((n,), 7.0, dtype=torch.float32, device="cuda")
                B.tc_forces(tc.ctx, theta, eps, da, dp)
                tc.sync()
                a, p = da.cpu().numpy(), dp.cpu().numpy()
            else:
                a, p = tc.forces(theta, eps)
            c, d = tc.counts()
            s = tc.stats()
            mine = c + d > 0                                   # every evaluated particle has at least one interaction
            assert (a[~mine] == 0).all() and (p[~mine] == 0).all()
            assert abs(mine.sum() - n / k) < 0.25 * n / k      # balanced in particles ...
            assert abs((s["n_pc_total"] + s["n_pp_total"]) * k / (s0["n_pc_total"] + s0["n_pp_total"]) - 1) < 0.1   # ... and in work
            owner += mine
            acc += a; pot += p; npc += c; npp += d
            tot += (s["n_pc_total"], s["n_pp_total"], s["n_tests_total"])
        assert (owner == 1).all()
        assert np.array_equal(acc, acc0) and np.array_equal(pot, pot0)
        assert np.array_equal(npc, c0) and np.array_equal(npp, d0)
        assert tuple(tot) == (s0["n_pc_total"], s0["n_pp_total"], s0["n_tests_total"])
        # back to one shard: the whole again
        tc.set_option("shard_count", 1)
        a, p = tc.forces(theta, eps)
        assert np.array_equal(a, acc0)
    check(acc, pot, npc, npp, Oracle(pos, mass, n_leaf, 64).forces(theta, eps, shadow32=True))


def test_shard_argument_errors_and_more_shards_than_groups():
    pos, mass, theta, eps, n_leaf = inputs.make("plummer_1k")
    with B.TreeCode(n_group=64) as tc:
        tc.set_particles(pos, mass)
        tc.build(n_leaf)
        ng = tc.stats()["n_groups"]
        for bad in (0, 1.5, 1e6):
            with pytest.raises(B.TcError):
                tc.set_option("shard_count", bad)
        tc.set_option("shard_count", 2)
        tc.set_option("shard_rank", 2)
        with pytest.raises(B.TcError) as e:
            tc.forces(theta, eps)
        assert e.value.code == B.TC_EINVAL
        tc.set_option("shard_rank", 1)
        tc.set_option("two_pass", 1)
        with pytest.raises(B.TcError) as e:
            tc.forces(theta, eps)
        assert e.value.code == B.TC_EINVAL
        tc.set_option("two_pass", 0)
        # more shards than groups: the high ranks have nothing to do and return zeros
        k = ng + 3
        tc.set_option("shard_count", k)
        total = np.zeros((len(mass), 3), np.float32)
        for r in range(k):
            tc.set_option("shard_rank", r)
            a, _ = tc.forces(theta, eps)
            if r >= ng:
                assert (a == 0).all()
            total += a
        tc.set_option("shard_count", 1)
        a, _ = tc.forces(theta, eps)
        assert np.array_equal(total, a)


def test_forces_sharded_single_process_is_the_plain_call():
    import torch
    from paper_1005_5384_b200 import parallel
    pos, mass, theta, eps, n_leaf = inputs.make("plummer_1k")
    n = len(mass)
    with B.TreeCode() as tc:
        tc.set_particles(pos, mass)
        tc.build(n_leaf)
        a0, p0 = tc.forces(theta, eps)
        acc = torch.empty((n, 3), dtype=torch.float32, device="cuda")
        pot = torch.empty(n, dtype=torch.float32, device="cuda")
        parallel.forces_sharded(tc, theta, eps, acc, pot)
        assert np.array_equal(acc.cpu().numpy(), a0) and np.array_equal(pot.cpu().numpy(), p0)
