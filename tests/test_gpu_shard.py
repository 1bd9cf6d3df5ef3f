"""ONE force evaluation over k GPUs (tc_forces_shard / tc_shard_scatter, options "shard_count" / "shard_rank";
DESIGN.md section 8) on one GPU — `-m gpu`: the k shards are run one after the other into the
rows an all-gather would deliver; every particle is evaluated by exactly one of them and the scattered result is
bit for bit the unsharded one."""
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


def run_shards(tc, k, theta, eps, n, with_counts=True):
    """The k shards one after the other -> (gathered rows, gathered counts, per-shard stats)."""
    import torch
    tc.set_option("shard_count", k)
    tc.set_option("shard_rank", 0)
    n_slots = tc.shard_size()
    gathered = torch.full((k, n_slots, 4), float("nan"), dtype=torch.float32, device="cuda")
    gcnt = torch.full((k, n_slots, 2), -7, dtype=torch.int32, device="cuda") if with_counts else None
    stats = []
    for r in range(k):
        tc.set_option("shard_rank", r)
        assert tc.shard_size() == n_slots                      # the same on every rank
        tc.forces_shard(theta, eps, gathered[r], gcnt[r] if with_counts else None)
        tc.sync()
        stats.append(tc.stats())
    return gathered, gcnt, stats, n_slots


@pytest.mark.parametrize("k", [1, 2, 3, 8])
@pytest.mark.parametrize("device_build", [0, 1])
def test_shards_partition_the_particles_and_scatter_to_the_whole(k, device_build):
    import torch
    pos, mass, theta, eps, n_leaf = inputs.make("plummer_64k")
    n = len(mass)
    with B.TreeCode(n_group=64) as tc:
        tc.set_option("device_build", device_build)
        tc.set_particles(pos, mass)
        tc.build(n_leaf)
        acc0, pot0 = tc.forces(theta, eps)
        c0, d0 = tc.counts()
        s0 = tc.stats()
        gathered, gcnt, stats, n_slots = run_shards(tc, k, theta, eps, n)
        # every rank wrote only its own rows: exactly n rows are filled in total, balanced over the ranks
        filled = ~torch.isnan(gathered[:, :, 0])
        per_rank = filled.sum(1).cpu().numpy()
        assert per_rank.sum() == n and per_rank.max() == n_slots
        assert (filled.cpu().numpy() == (np.arange(n_slots)[None, :] < per_rank[:, None])).all()   # compact: a prefix of the rows
        assert np.abs(per_rank - n / k).max() < 0.25 * n / k                                      # balanced in particles ...
        work = np.array([s["n_pc_total"] + s["n_pp_total"] for s in stats], dtype=np.float64)
        assert np.abs(work * k / (s0["n_pc_total"] + s0["n_pp_total"]) - 1).max() < 0.1             # ... and in work
        for key in ("n_pc_total", "n_pp_total", "n_tests_total"):
            assert sum(s[key] for s in stats) == s0[key]
        with pytest.raises(B.TcError) as e:                       # the counts of a shard live in its rows
            tc.counts()
        assert e.value.code == B.TC_ESTATE
        acc = torch.full((n, 3), float("nan"), dtype=torch.float32, device="cuda")
        pot = torch.full((n,), float("nan"), dtype=torch.float32, device="cuda")
        npc = torch.full((n,), -1, dtype=torch.int32, device="cuda")
        npp = torch.full((n,), -1, dtype=torch.int32, device="cuda")
        tc.shard_scatter(gathered, gcnt, acc, pot, npc, npp)
        tc.sync()
        acc, pot, npc, npp = acc.cpu().numpy(), pot.cpu().numpy(), npc.cpu().numpy(), npp.cpu().numpy()
        assert np.array_equal(acc, acc0) and np.array_equal(pot, pot0)        # bit for bit the single-GPU result
        assert np.array_equal(npc, c0) and np.array_equal(npp, d0)
        # without counts and without pot
        acc2 = torch.full((n, 3), float("nan"), dtype=torch.float32, device="cuda")
        tc.shard_scatter(gathered, None, acc2)
        tc.sync()
        assert np.array_equal(acc2.cpu().numpy(), acc0)
        # back to one shard: the plain call again
        tc.set_option("shard_count", 1); tc.set_option("shard_rank", 0)
        a, p = tc.forces(theta, eps)
        assert np.array_equal(a, acc0)
    check(acc, pot, npc, npp, Oracle(pos, mass, n_leaf, 64).forces(theta, eps, shadow32=True))


def test_shard_argument_errors_and_more_shards_than_groups():
    import torch
    pos, mass, theta, eps, n_leaf = inputs.make("plummer_1k")
    n = len(mass)
    with B.TreeCode(n_group=64) as tc:
        tc.set_particles(pos, mass)
        tc.build(n_leaf)
        ng = tc.stats()["n_groups"]
        a0, p0 = tc.forces(theta, eps)
        for bad in (0, 1.5, 1e6):
            with pytest.raises(B.TcError):
                tc.set_option("shard_count", bad)
        rows = torch.empty((n, 4), dtype=torch.float32, device="cuda")
        tc.set_option("shard_count", 2)
        with pytest.raises(B.TcError) as e:                       # the plain call refuses to be a shard
            tc.forces(theta, eps)
        assert e.value.code == B.TC_ESTATE
        tc.set_option("shard_rank", 2)
        with pytest.raises(B.TcError) as e:
            tc.forces_shard(theta, eps, rows)
        assert e.value.code == B.TC_EINVAL
        tc.set_option("shard_rank", 1)
        tc.set_option("two_pass", 1)
        with pytest.raises(B.TcError) as e:
            tc.forces_shard(theta, eps, rows)
        assert e.value.code == B.TC_EINVAL
        tc.set_option("two_pass", 0)
        with pytest.raises(B.TcError) as e:                       # host rows: device buffers only
            B.tc_forces_shard(tc.ctx, theta, eps, np.zeros((n, 4), np.float32))
        assert e.value.code == B.TC_EINVAL
        with pytest.raises(TypeError):                            # the binding checks dtype and shape before the C call
            B.tc_forces_shard(tc.ctx, theta, eps, torch.empty((n, 3), dtype=torch.float32, device="cuda"))
        # more shards than groups: the high ranks have nothing to do and write no row
        k = ng + 3
        gathered, gcnt, stats, n_slots = run_shards(tc, k, theta, eps, n, with_counts=False)
        assert torch.isnan(gathered[ng:, :, :]).all()
        acc = torch.empty((n, 3), dtype=torch.float32, device="cuda"); pot = torch.empty(n, dtype=torch.float32, device="cuda")
        tc.shard_scatter(gathered, None, acc, pot)
        tc.sync()
        assert np.array_equal(acc.cpu().numpy(), a0) and np.array_equal(pot.cpu().numpy(), p0)
        # a rebuilt tree gets a new layout
        tc.set_option("shard_count", 1); tc.set_option("shard_rank", 0)
        tc.set_option("n_group", 16)
        tc.build(n_leaf)
        a1, p1 = tc.forces(theta, eps)
        gathered, _, _, _ = run_shards(tc, 3, theta, eps, n, with_counts=False)
        tc.shard_scatter(gathered, None, acc, pot)
        tc.sync()
        assert np.array_equal(acc.cpu().numpy(), a1) and np.array_equal(pot.cpu().numpy(), p1)


def test_forces_sharded_single_process_is_the_plain_call():
    import torch
    from paper_1005_5384_b200 import parallel
    pos, mass, theta, eps, n_leaf = inputs.make("plummer_1k")
    n = len(mass)
    with B.TreeCode() as tc:
        tc.use_torch_stream()
        tc.set_particles(pos, mass)
        tc.build(n_leaf)
        a0, p0 = tc.forces(theta, eps)
        c0, d0 = tc.counts()
        acc = torch.empty((n, 3), dtype=torch.float32, device="cuda")
        pot = torch.empty(n, dtype=torch.float32, device="cuda")
        npc = torch.empty(n, dtype=torch.int32, device="cuda"); npp = torch.empty(n, dtype=torch.int32, device="cuda")
        sc = {}
        for _ in range(2):
            parallel.forces_sharded(tc, theta, eps, acc, pot, n_pc=npc, n_pp=npp, scratch=sc)
        tc.sync()
        assert np.array_equal(acc.cpu().numpy(), a0) and np.array_equal(pot.cpu().numpy(), p0)
        assert np.array_equal(npc.cpu().numpy(), c0) and np.array_equal(npp.cpu().numpy(), d0)


def test_sharded_large_groups_and_eps0():
    """Groups above the pass size (N_group = 256 > 128: two passes per group) and eps = 0 through the shard path."""
    import torch
    pos, mass, theta, _, _ = inputs.make("plummer_64k")
    n = len(mass)
    with B.TreeCode(n_group=256) as tc:
        tc.set_particles(pos, mass)
        tc.build(4)
        a0, p0 = tc.forces(theta, 0.0)
        gathered, _, _, _ = run_shards(tc, 4, theta, 0.0, n, with_counts=False)
        acc = torch.empty((n, 3), dtype=torch.float32, device="cuda"); pot = torch.empty(n, dtype=torch.float32, device="cuda")
        tc.shard_scatter(gathered, None, acc, pot)
        tc.sync()
        assert np.array_equal(acc.cpu().numpy(), a0) and np.array_equal(pot.cpu().numpy(), p0)
